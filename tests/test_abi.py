"""The C-ABI library builds, loads and exports every symbol include/rmhd.h declares (no GPU:
no compute calls), and fails loudly (RMHD_ERR_CUDA) rather than falling back when there is no
CUDA device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_1808_09721_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "rmhd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rmhd_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(B):
    syms = _declared_symbols()
    assert len(syms) >= 18
    L = B.lib()
    for s in syms:
        assert hasattr(L, s), s
    assert set(syms) == set(B.EXPORTS)


def test_params_struct_matches_header_field_order(B):
    text = open(os.path.join(ROOT, "include", "rmhd.h")).read()
    body = text[text.index("typedef struct {"):text.index("} rmhd_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.replace("typedef struct {", "").strip()
        if not decl:
            continue
        m = re.match(r"(?:int|double|void\s*\*)\s*(.*)", decl)
        for n in m.group(1).split(","):
            names.append(re.sub(r"\[.*\]", "", n).replace("*", "").strip())
    assert names == [f[0] for f in B.rmhd_params._fields_]


def test_bad_parameters_are_rejected_without_touching_the_gpu(B):
    h = C.c_void_p()
    for kw in (dict(model=7), dict(gamma=1.0), dict(model=1, mu_e=2.0, mu_p=2.0), dict(nx=0), dict(ng=1), dict(cfl=0.0),
               dict(bc=(0, 3, 0))):
        p = B.make_params(**{**dict(nx=8, sigma=1.0), **kw})
        assert B.lib().rmhd_create(C.byref(p), C.byref(h)) == B.RMHD_ERR_BAD_PARAM
        assert B.lib().rmhd_last_error(None)


def test_no_cpu_fallback_without_a_device(B):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    p = B.make_params(nx=8, sigma=1.0)
    with pytest.raises(B.RmhdError) as e:
        B.rmhd_create(p)
    assert e.value.code == B.RMHD_ERR_CUDA
    q = np.zeros((14, 4)); w = np.zeros((11, 4))
    with pytest.raises(B.RmhdError) as e:
        B.rmhd_stage_batch(p, q, w, 1e-3, q.copy(), w.copy())
    assert e.value.code == B.RMHD_ERR_CUDA
    with pytest.raises(B.RmhdError):
        B.rmhd_probe_fp64()


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1808_09721_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), f
                assert "liboracle" not in src and "rmhd_oracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "rmhd_oracle.cpp")).read()
    assert "#include \"" not in osrc            # the oracle includes no project header
    for f in ("oracle.py", "build.py"):
        assert "paper_1808_09721_b200" not in open(os.path.join(ROOT, "oracle", f)).read()


def test_binding_rejects_buffers_of_the_wrong_size_before_the_call(B):
    """Marshalling checks (binding.py `_expect`): a buffer with the wrong row or cell count would be an out-of-bounds device
    access inside the library; the binding refuses it before any pointer crosses the ABI (no GPU needed)."""
    p = B.make_params(nx=8, sigma=1.0)
    q = np.zeros((14, 4)); w = np.zeros((11, 4))
    with pytest.raises(ValueError):
        B.rmhd_stage_batch(p, q, np.zeros((10, 4)), 1e-3, q.copy(), w.copy())          # prim_guess one row short
    with pytest.raises(ValueError):
        B.rmhd_stage_batch(p, q, w, 1e-3, np.zeros((14, 3)), w.copy())                 # q_out one cell short
    with pytest.raises(ValueError):
        B.rmhd_stage_batch(p, q, w, 1e-3, q.copy(), w.copy(), sigma_cell=np.zeros(5))
    with pytest.raises(ValueError):
        B.rmhd_prim2cons_batch(p, w, np.zeros((18, 4)))                                 # two-fluid sized output, resistive model
    with pytest.raises(ValueError):
        B.rmhd_con2prim_batch(p, q, w, fail=np.zeros(3, np.int32))
    with pytest.raises(ValueError):
        B.rmhd_con2prim_batch(p, q.astype(np.float32), w)                               # wrong dtype


def test_the_one_environment_switch_is_documented(B):
    """include/rmhd.h names every environment variable the library reads."""
    src = open(os.path.join(ROOT, "paper_1808_09721_b200", "csrc", "rmhd.cu")).read()
    envs = set(re.findall(r'getenv\("([A-Z_0-9]+)"\)', src))
    assert envs == {"RMHD_FLUX"}
    hdr = open(os.path.join(ROOT, "include", "rmhd.h")).read()
    assert "RMHD_FLUX=split" in hdr and "test_ssp3_332_parity[blast_3d_split]" in hdr


def test_release_staging_without_anything_to_release(B):
    """No host-buffer batch call has run: nothing is held, nothing is touched (works without a GPU)."""
    assert B.lib().rmhd_release_staging(-1) == B.RMHD_OK
    assert B.lib().rmhd_release_staging(0) == B.RMHD_OK

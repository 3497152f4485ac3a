#!/usr/bin/env python
"""bench.py -- throughput of one full IMEX SSP2(222) step (all SURVEY.md 8(a) rows) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload cfg5|cfg2|cfg3|cfg4|cfg1|bw17|khi|khi2f] [--integrator ssp2|ssp3]

Workload at N=1: BASELINE.json configs[4], the 3-D 256^3 resistive blast -- the configuration
the metric ("FP64 zone-updates/s per full IMEX step") and the north-star target are quoted on;
configs[1] is a single implicit stage, not a full step: `--workload cfg2` times it on its own (2^20 device-resident
cells through rmhd_stage_batch, value = cells per second through one stage), it is not the headline.
`--integrator ssp3` times the SSP3(332) step on the same workloads; the headline is SSP2(222).  Inputs are synthetic (paper_1808_09721_b200.synth).
Prints ONE JSON line (rank 0).  Multi-GPU: the path does not shard in this build ("replicas
only"): each rank steps its own copy; value = zone-updates of all ranks / max time.

`--impl reference` times the CPU oracle as it stands on the host cores, on a bounded sample of
the same workload (a 96^3 sub-box of the 256^3 initial data around the blast, one step per
"step").  The oracle is a deliberately slow checker: the ratio to it is context, not a target.
"""
import argparse
import glob
import hashlib
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64_zone_updates_per_s_full_imex_step"
UNIT = "zone-updates/s"
SM_COUNT = 148
FP64_LANES_PER_SM = 64          # FP64 FMA lanes per SM (B200_PROFILING.md has no FP64 figure; DESIGN.md derives it)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return d.get("hbm_gbs", 6650.0), d.get("sm_max_mhz", 1965.0), "measured"
    return 6650.0, 1965.0, "fallback"


def csrc_sha16():
    """Hash of the CUDA sources: committed ncu figures are only quoted for the code they were captured on."""
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_1808_09721_b200", "csrc", "*.cu*"))):
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def committed_ncu(workload, integrator):
    """profiles/ncu_traffic.txt: DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) and FP64 pipe
    utilisation from one committed `ncu --set full` capture, keyed by workload/integrator; None if the capture was taken
    on other kernel sources."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.txt")
    if not os.path.exists(path):
        return None
    with open(path) as f:
        d = json.load(f)
    if d.get("csrc_sha16") != csrc_sha16():
        return None
    return d.get("captures", {}).get(f"{workload}/{integrator}")


# ---- clocks during the timed region ----------------------------------------------------------
class ClockSampler:
    def __init__(self, index=0, period=0.02):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._t = None
        self.index, self.period = index, period
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _reason_names(self, mask):
        nv = self.nv
        table = {
            "hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80),
        }
        return {k for k, bit in table.items() if mask & bit}

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                self.reasons |= self._reason_names(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
            except Exception:
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self.nv:
            self._t = threading.Thread(target=self._run, daemon=True)
            self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._t:
            self._t.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ---- workloads ---------------------------------------------------------------------------------
def make_workload(name, synth):
    if name == "cfg5":
        return synth.config5()
    if name == "cfg2":
        return synth.config2()
    if name == "cfg3":
        return synth.config3()
    if name == "cfg1":
        return synth.config1()
    if name == "cfg4":
        return synth.config4()
    if name == "bw17":              # the paper's profile-table workload: 1-D Brio-Wu, nx = 2^17, sigma = 1e4
        return synth.brio_wu_single(nx=2 ** 17, sigma=1e4)
    if name == "khi":               # the paper's Fig 8 workload: 512 x 1024 KHI, single fluid
        return synth.khi_paper(model=0)
    if name == "khi2f":             # ... two-fluid
        return synth.khi_paper(model=1)
    raise SystemExit(f"unknown workload {name}")


def oracle_sample(cfg, synth):
    """A bounded sample of the workload for the CPU oracle: central 96^3 (or whole grid if smaller)."""
    p = dict(cfg["params"])
    w = cfg["prims"]
    nz, ny, nx = w.shape[1:]
    m = 96
    if nz > m and ny > m and nx > m:
        sl = [slice((n - m) // 2, (n - m) // 2 + m) for n in (nz, ny, nx)]
        dx = [(p["zlim"][1] - p["zlim"][0]) / nz, (p["ylim"][1] - p["ylim"][0]) / ny, (p["xlim"][1] - p["xlim"][0]) / nx]
        lim = lambda lo, s, d: (lo + s.start * d, lo + s.stop * d)
        p.update(nx=m, ny=m, nz=m, zlim=lim(p["zlim"][0], sl[0], dx[0]), ylim=lim(p["ylim"][0], sl[1], dx[1]),
                 xlim=lim(p["xlim"][0], sl[2], dx[2]))
        w = np.ascontiguousarray(w[:, sl[0], sl[1], sl[2]])
        what = f"central {m}^3 sub-box of the {nx}^3 initial data (same dx), 1 oracle step per sample step"
    else:
        what = "the whole grid, 1 oracle step per sample step"
    return p, w, what


def time_oracle_one_thread(cfg, integrator="ssp2", m=48, budget_s=12.0):
    """The oracle on ONE host thread (the paper's baseline is one Xeon core): >= 2 steps of a central m^3 (or
    m^2, m) sub-box of the workload."""
    from oracle import oracle as O
    p = dict(cfg["params"]); w = cfg["prims"]
    shp = w.shape[1:]
    sl = [slice((n - m) // 2, (n - m) // 2 + m) if n > m else slice(0, n) for n in shp]
    lims = [p.get("zlim", (0.0, 1.0)), p.get("ylim", (0.0, 1.0)), p.get("xlim", (0.0, 1.0))]
    new = [(lo + s_.start * (hi - lo) / n, lo + s_.stop * (hi - lo) / n) for (lo, hi), s_, n in zip(lims, sl, shp)]
    w = np.ascontiguousarray(w[:, sl[0], sl[1], sl[2]])
    p.update(nz=w.shape[1], ny=w.shape[2], nx=w.shape[3], zlim=new[0], ylim=new[1], xlim=new[2], integrator=integrator)
    rc = cfg.get("rho_charge")
    if rc is not None:
        rc = np.ascontiguousarray(rc[sl[0], sl[1], sl[2]])
    prev = O.set_threads(0)
    O.set_threads(1)
    try:
        S = O.OracleSim(O.make_params(**p)); S.set_initial(w, rc)
        t0 = time.perf_counter(); done = 0
        while done < 2 or (time.perf_counter() - t0 < min(1.0, budget_s / 3) and done < 4096):
            S.step(1); done += 1
        dt = time.perf_counter() - t0
        S.close()
    finally:
        O.set_threads(prev)
    ncell = w.shape[1] * w.shape[2] * w.shape[3]
    return ncell * done / dt, f"central {w.shape[3]}x{w.shape[2]}x{w.shape[1]} sub-box, {done} steps in {dt:.1f} s on 1 thread"


def time_oracle(cfg, synth, steps, warmup, budget_s=40.0, integrator="ssp2"):
    from oracle import oracle as O
    p, w, what = oracle_sample(cfg, synth)
    p["integrator"] = integrator
    cores = O.set_threads(0)
    S = O.OracleSim(O.make_params(**p))
    S.set_initial(w, cfg.get("rho_charge"))
    ncell = w.shape[1] * w.shape[2] * w.shape[3]
    t0 = time.perf_counter()
    for _ in range(max(warmup, 0)):
        S.step(1)
        if time.perf_counter() - t0 > budget_s / 2:
            break
    t0 = time.perf_counter()
    done = 0
    for _ in range(steps):
        S.step(1)
        done += 1
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    S.close()
    return {"value": ncell * done / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{what}; {done} steps in {dt:.1f} s"}, dt / done * 1e3, done


# ---- reference arm --------------------------------------------------------------------------
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1808_09721_b200 import synth
    cfg = make_workload(args.workload, synth)
    if args.workload == "cfg2":
        v, cores, sample = cfg2_oracle_rate(cfg, 0, 1 << 16, budget_s=30.0)
        base = {"value": v, "unit": CFG2_UNIT, "cores": cores, "kind": "oracle", "sample": sample}
        print(json.dumps({"impl": "reference", "metric": CFG2_METRIC, "value": v, "unit": CFG2_UNIT, "n_gpus": args.gpus, "steps": args.steps,
                          "warmup": 0, "ms_per_step": (1 << 16) / v * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                          "dtype": "f64", "data": "synthetic", "config": {"workload": cfg["name"] + " (oracle sample)", "sample": sample},
                          "cpu_baseline": base, "e2e": {"value": v, "unit": CFG2_UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                          "gpu_launches": 0}))
        return
    base, ms, done = time_oracle(cfg, synth, args.steps, min(args.warmup, 1), budget_s=120.0, integrator=args.integrator)
    line = {
        "impl": "reference", "metric": METRIC, "value": base["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": done,
        "warmup": min(args.warmup, 1), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"] + " (oracle sample)", "sample": base["sample"]},
        "cpu_baseline": base,
        "e2e": {"value": base["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ---- replicas-only aggregation --------------------------------------------
def whole_job_rate(ms_local, units_local, dist, device):
    """Whole-job throughput over all ranks: units of every rank summed, divided by the slowest rank's device time.
    No data-path collective exists (each rank steps its own replica); these two reductions are the only exchange.
    Returns (units per second, max ms).  `dist` is torch.distributed or None (one process)."""
    import torch
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    ms = float(t.item())
    return float(u.item()) / (ms * 1e-3), ms


# ---- our arm ----------------------------------------------------------------------------------
def stage_flops(hist):
    """Algorithmic flops of one resistive implicit-stage launch from the logged iteration histogram.
    Per Newton iteration of the 4x4 system (stage.cuh r_stage_iter; FMA = 2, div/rsqrt = 1):
    ~420 flop; init + finish ~150 flop."""
    its = (hist * np.arange(hist.size)).sum()
    n = hist.sum()
    return 420.0 * its + 150.0 * n


# ---- BASELINE.json configs[1]: one batched implicit stage ------------------------------------------
CFG2_METRIC, CFG2_UNIT = "fp64_cells_per_s_one_implicit_stage", "cells/s"
CFG2_DOUBLES = 14 + 5 + 1 + 14 + 11        # R q_ex, guess (rho, v, p: B, E come with q_ex), sigma; W q*, prims  (+ 2 int32: iterations, flag)


def cfg2_oracle_rate(cfg, threads, ncell, budget_s=10.0):
    from oracle import oracle as O
    prev = O.set_threads(0)
    used = O.set_threads(threads) if threads else prev
    try:
        P = O.make_params(**cfg["params"])
        w = np.ascontiguousarray(cfg["prims"][:, :ncell]); sg = np.ascontiguousarray(cfg["sigma_cell"][:ncell])
        q_ex = O.prim2cons(P, w)
        t0 = time.perf_counter(); done = 0
        while done < 1 or time.perf_counter() - t0 < budget_s / 2:
            O.stage_batch(P, q_ex, w, cfg["a_dt"], sg); done += 1
        dt = time.perf_counter() - t0
    finally:
        O.set_threads(prev)
    return ncell * done / dt, used, f"first {ncell} cells of the 2^20-cell batch, {done} stage solves in {dt:.1f} s"


def run_cfg2(args, B, synth, torch, dist, dev, rank, world, local, hbm_peak, sm_max_mhz, peak_src, fp64_meas):
    """2^20 independent resistive cells through rmhd_stage_batch (the implicit root-find is 55.3 % of the
    paper's run time).  A step = one implicit stage over the whole batch, inputs and outputs resident in HBM."""
    cfg = synth.config2()
    n = cfg["prims"].shape[1]
    P = B.make_params(**dict(cfg["params"], device=local))
    w_d = torch.from_numpy(cfg["prims"]).to(dev); sg_d = torch.from_numpy(cfg["sigma_cell"]).to(dev)
    qex_d = torch.empty((14, n), dtype=torch.float64, device=dev)
    B.rmhd_prim2cons_batch(P, w_d, qex_d)
    q_d = torch.empty_like(qex_d); wo_d = torch.empty_like(w_d)
    it_d = torch.zeros(n, dtype=torch.int32, device=dev); fl_d = torch.zeros(n, dtype=torch.int32, device=dev)

    def one():
        B.rmhd_stage_batch(P, qex_d, w_d, cfg["a_dt"], q_d, wo_d, sg_d, it_d, fl_d)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    flush = torch.empty(160 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)   # > 126 MB L2
    for _ in range(args.warmup):
        one()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    with ClockSampler(local) as clk:
        for a, b in ev:
            flush.fill_(1.0)                      # the batch (218 MB in + 210 MB out) exceeds L2, flushed all the same
            a.record(); one(); b.record()
        barrier()
    ms_total = sum(a.elapsed_time(b) for a, b in ev)
    value, ms_total = whole_job_rate(ms_total, n * args.steps, dist, dev)
    its = it_d.cpu().numpy(); fl = fl_d.cpu().numpy()
    hist = np.bincount(its, minlength=64).astype(np.float64)
    ms = ms_total / args.steps
    flops = stage_flops(hist)
    t_hbm = (CFG2_DOUBLES * 8 + 8) * n / (hbm_peak * 1e9); t_alu = flops / (fp64_meas * 1e12)
    bound = "hbm" if t_hbm >= t_alu else "alu"
    roof = {"bound": bound, "kernel": "k_stage_batch_resistive",
            "achieved": (flops / (ms * 1e-3) * 1e-12) if bound == "alu" else ((CFG2_DOUBLES * 8 + 8) * n / (ms * 1e-3) * 1e-9),
            "peak": fp64_meas if bound == "alu" else hbm_peak, "unit": "TFLOP/s" if bound == "alu" else "GB/s",
            "peak_source": "measured in this run: rmhd_probe_fp64 (DFMA chains on all SMs)" if bound == "alu" else peak_src + " (MEASURED_PEAKS.json hbm_gbs)",
            "hbm_frac": t_hbm / (ms * 1e-3), "alu_frac": t_alu / (ms * 1e-3), "fp64_peak_measured_tflops": fp64_meas,
            "fp64_peak_nominal_tflops": SM_COUNT * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 * 1e-12, "hbm_peak_gbs": hbm_peak,
            "alg_bytes_per_cell": CFG2_DOUBLES * 8 + 8, "alg_flops_per_cell": flops / n, "avg_launch_ms": ms, "traffic": None,
            "stage_iters_mean": float((hist * np.arange(hist.size)).sum() / n), "stage_iters_max": int(its.max()),
            "stage_iters_hist": [int(x) for x in hist[:int(its.max()) + 1]]}
    roof["frac"] = roof["achieved"] / roof["peak"]
    cap = committed_ncu("cfg2", "stage")
    if cap:
        roof["traffic"] = cap.get("dram_bytes_per_launch", {}).get("stage_batch")
        roof["fp64_pipe_busy_ncu"] = cap.get("fp64_pipe_busy", {}).get("stage_batch")
        roof["ncu_traffic_committed"] = {"file": "profiles/ncu_traffic.txt", "capture": cap.get("source"), "csrc_sha16": csrc_sha16()}
    # end to end: host buffers in, host buffers out through the same C-ABI call (the library stages them on the device)
    e2e = None
    if rank == 0 or world > 1:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        w_h, sg_h = pin(cfg["prims"]), pin(cfg["sigma_cell"])
        qex_h = pin(qex_d.cpu().numpy())
        q_h = torch.empty((14, n), dtype=torch.float64).pin_memory(); wo_h = torch.empty((11, n), dtype=torch.float64).pin_memory()
        it_h = torch.zeros(n, dtype=torch.int32).pin_memory(); fl_h = torch.zeros(n, dtype=torch.int32).pin_memory()
        e_steps = max(1, min(args.steps, 5))
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        B.rmhd_stage_batch(P, qex_h, w_h, cfg["a_dt"], q_h, wo_h, sg_h, it_h, fl_h)
        barrier(); a.record()
        for _ in range(e_steps):
            B.rmhd_stage_batch(P, qex_h, w_h, cfg["a_dt"], q_h, wo_h, sg_h, it_h, fl_h)
        b.record(); barrier()
        e_rate, _ = whole_job_rate(a.elapsed_time(b), n * e_steps, dist, dev)
        e2e = {"value": e_rate, "unit": CFG2_UNIT, "h2d_bytes_per_step": (14 + 11 + 1) * 8 * n, "d2h_bytes_per_step": (14 + 11 + 1) * 8 * n,
               "steps": e_steps, "call": "rmhd_stage_batch(on_device = 0), pinned host buffers"}
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    cpu_base = None
    if world == 1 and not args.no_cpu_baseline:
        vN, cores, sample = cfg2_oracle_rate(cfg, 0, 1 << 16)
        v1, _, s1 = cfg2_oracle_rate(cfg, 1, 1 << 13)
        cpu_base = {"value": vN, "unit": CFG2_UNIT, "cores": cores, "kind": "oracle", "sample": sample, "value_1thread": v1, "sample_1thread": s1}
    line = {"metric": CFG2_METRIC, "value": value, "unit": CFG2_UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg['name']}: {n} independent resistive cells, one implicit stage a = gamma x 1e-3, sigma log-uniform [1, 1e6]",
                       "parallelism": "replicas only" if world > 1 else "1 gpu", "l2": "L2 flushed (160 MB fill) before every timed launch",
                       "n_failed_cells": int((fl != 0).sum())},
            "clocks": clk.summary(), "e2e": e2e, "gpu_launches": args.steps, "roofline": roof, "cpu_baseline": cpu_base}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def run_ours(args):
    import torch
    from paper_1808_09721_b200 import binding as B, synth
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()
    hbm_peak, sm_max_mhz, peak_src = load_peaks()
    dev = torch.device("cuda", local)
    fp64_meas = B.rmhd_probe_fp64(local)                # TFLOP/s, DFMA chains on all SMs
    if args.workload == "cfg2":
        return run_cfg2(args, B, synth, torch, dist, dev, rank, world, local, hbm_peak, sm_max_mhz, peak_src, fp64_meas)

    cfg = make_workload(args.workload, synth)
    p = dict(cfg["params"]); p["device"] = local; p["integrator"] = args.integrator
    nstage = 3 if args.integrator == "ssp3" else 2
    nz, ny, nx = cfg["prims"].shape[1:]
    ncell = nx * ny * nz
    sim = B.Rmhd(**p)
    prims_d = torch.from_numpy(np.ascontiguousarray(cfg["prims"])).to(dev)
    sim.set_initial(prims_d)
    del prims_d

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing -------------------------------------------------------------
    # K steps through one rmhd_step(ctx, K) call (one statistics read and stream sync at its end), CUDA events on the
    # library's stream around it; a second, instrumented pass of K steps (an event pair around every launch) gives the
    # per-kernel times the roofline object uses, so that instrumentation does not sit inside the timed region.
    for _ in range(args.warmup):
        sim.step(1)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    with ClockSampler(local) as clk:
        ev0.record()
        sim.step(args.steps)
        ev1.record()
        barrier()
    ms_total = ev0.elapsed_time(ev1)
    B.rmhd_set_profiling(sim.ctx, True)
    B.rmhd_debug_hm_cycles(local, reset=True)           # None unless this is a measurement build (-DRMHD_HM_CYCLES)
    sim.step(args.steps)
    kt = B.rmhd_get_kernel_times(sim.ctx)
    hm_cycles = B.rmhd_debug_hm_cycles(local)
    stats = sim.stats()
    B.rmhd_set_profiling(sim.ctx, False)
    value, ms_total = whole_job_rate(ms_total, ncell * args.steps, dist, dev)

    # ---- roofline of the dominant kernel class -------------------------------------------------
    naxes = sum(1 for n in (nx, ny, nz) if n > 1)
    model = p["model"]
    dom = max(("stage1", "stage2", "flux", "combine_c2p"), key=lambda k: kt[k]["ms"])
    avg_ms = kt[dom]["ms"] / max(kt[dom]["launches"], 1)
    shares = {k: round(v["ms"] / max(sum(x["ms"] for x in kt.values()), 1e-30), 4) for k, v in kt.items()}
    fused = nx > 1 and ny > 1 and os.environ.get("RMHD_FLUX") != "split"
    nfl = max(kt["flux"]["launches"], 1) / (float(nstage) * args.steps)   # launches per L(q): 1 fused, naxes split
    # Algorithmic doubles per cell per launch: every array touched once by its producer and once by
    # each consumer, halo re-reads excluded.  NC conserved rows, NH hydro primitives, NS rows with a source.
    NC, NH, NS = (14, 5, 5) if model == 0 else (18, 10, 9)
    NQ = NC - NS                                       # rows without a source
    d_s1 = NC + NH + NS + NH + NS                      # R qn, w; W the NS rows of q1, w, Psi1
    d_s_full = NC + NC + NS + NH + NC + NH + NS        # R qn, L1, Psi1, w; W q2, w, Psi2 (per-axis path, and SSP3 stage 2)
    d_s_fused = NQ + NS + NS + NS + NH + NS + NH + NS  # fused SSP2 stage 2: R q_ex (NQ rows, left by F1), qn, L1, Psi1 (NS rows each), w; W q2 (NS), w, A (NS)
    d_f = NC + NH + NC                                 # R q, w; W L
    d_f_last = NC + NH + NQ + NS + NC                  # last fused flux launch: + R qn (NQ rows), A (NS rows); W q^{n+1}
    d_p = (NC - 3 if model == 0 else NC - 2) + NH + NH # con2prim: R D, S, tau, (Dbar, Sbar, taubar,) B, E + guess; W w
    d_final = 3 * NC + 2 * NS + NH + NC + NH           # k_final (per-axis path): R qn, L1, L2, Psi1, Psi2, guess; W q, w
    per_launch = {
        "stage1": d_s1,
        "stage2": (d_s_fused if nstage == 2 else d_s_full) if fused else d_s_full,
        "flux": (d_f * (nstage - 1) + d_f_last) / float(nstage) if fused else d_f / nfl,
        "combine_c2p": d_p if fused else d_final,
    }
    alg_bytes = {k: v * 8.0 * ncell for k, v in per_launch.items()}
    # Algorithmic flops per launch (FMA = 2, div / sqrt / rsqrt = 1; DESIGN.md section 5 "flop model")
    its_stage = float((stats["hist_stage"] * np.arange(stats["hist_stage"].size)).sum() / max(stats["hist_stage"].sum(), 1))
    its_c2p = float((stats["hist_c2p"] * np.arange(stats["hist_c2p"].size)).sum() / max(stats["hist_c2p"].sum(), 1))
    it_fl, fix_fl = (420.0, 150.0) if model == 0 else (1800.0, 300.0)
    per_axis, per_cell = (430.0, 30.0) if model == 0 else (628.0, 45.0)
    alg_flops = {
        "stage1": (it_fl * its_stage + fix_fl) * ncell,
        "stage2": (it_fl * its_stage + fix_fl) * ncell,
        "flux": (per_axis * naxes + per_cell) * ncell / nfl,
        "combine_c2p": (30.0 * its_c2p + 40.0) * (1 if model == 0 else 2) * ncell,
    }
    t_hbm = alg_bytes[dom] / (hbm_peak * 1e9)           # roofline times of the dominant kernel, seconds
    t_alu = alg_flops[dom] / (fp64_meas * 1e12)
    bound = "hbm" if t_hbm >= t_alu else "alu"
    hbm_frac = t_hbm / (avg_ms * 1e-3)
    alu_frac = t_alu / (avg_ms * 1e-3)
    if bound == "hbm":
        roof = {"bound": "hbm", "kernel": dom, "achieved": alg_bytes[dom] / (avg_ms * 1e-3) * 1e-9, "peak": hbm_peak, "unit": "GB/s",
                "peak_source": peak_src + " (MEASURED_PEAKS.json hbm_gbs)"}
    else:
        roof = {"bound": "alu", "kernel": dom, "achieved": alg_flops[dom] / (avg_ms * 1e-3) * 1e-12, "peak": fp64_meas, "unit": "TFLOP/s",
                "peak_source": "measured in this run: rmhd_probe_fp64 (DFMA chains on all SMs)"}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["hbm_frac"] = hbm_frac                         # algorithmic bytes / (launch time x measured HBM peak)
    roof["alu_frac"] = alu_frac                         # algorithmic flops / (launch time x measured FP64 peak)
    roof["fp64_peak_measured_tflops"] = fp64_meas
    roof["fp64_peak_nominal_tflops"] = SM_COUNT * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 * 1e-12
    roof["hbm_peak_gbs"] = hbm_peak
    roof["alg_doubles_per_cell_per_launch"] = per_launch[dom]
    roof["alg_flops_per_cell_per_launch"] = alg_flops[dom] / ncell
    roof["avg_launch_ms"] = avg_ms
    roof["kernel_time_shares"] = shares
    roof["kernel_ms_per_step"] = {k: v["ms"] / args.steps for k, v in kt.items()}
    if hm_cycles is not None:   # measurement build: clock() ticks per warp and plane, by role and phase (csrc/flux_hm.cuh); never a bench number
        roof["hm_cycles_per_warp_plane"] = {r: [float(hm_cycles[i][ph]) / max(float(hm_cycles[i][7]), 1.0) for ph in range(7)]
                                            for i, r in enumerate(("H", "M"))}
        roof["hm_warp_planes"] = [int(hm_cycles[0][7]), int(hm_cycles[1][7])]
        roof["measurement_build"] = "-DRMHD_HM_CYCLES: the times of this line are perturbed by the instrumentation"
    # DRAM bytes per launch from the committed ncu capture of exactly these kernel sources, else null
    cap = committed_ncu(args.workload, args.integrator)
    roof["traffic"] = None
    if cap and dom in cap.get("dram_bytes_per_launch", {}):
        roof["traffic"] = cap["dram_bytes_per_launch"][dom]
        roof["ncu_traffic_committed"] = {"file": "profiles/ncu_traffic.txt", "capture": cap.get("source"), "csrc_sha16": csrc_sha16()}
        if dom in cap.get("fp64_pipe_busy", {}):
            roof["fp64_pipe_busy_ncu"] = cap["fp64_pipe_busy"][dom]
    # Whole step: the bytes THIS build's launches move (sum over the launches of a step of the per-launch figures above),
    # and, separately, the survey's minimum-traffic model (195 doubles resistive SSP2; not what the kernels move)
    lps = {k: kt[k]["launches"] / float(args.steps) for k in per_launch}
    step_doubles_build = sum(per_launch[k] * lps[k] for k in per_launch)
    step_ms = ms_total / args.steps
    roof["whole_step_doubles_per_zone_update"] = step_doubles_build
    roof["whole_step_hbm_frac"] = step_doubles_build * 8 * ncell / (step_ms * 1e-3) * 1e-9 / hbm_peak
    survey_doubles = (323 if nstage == 3 else 195) if model == 0 else (469 if nstage == 3 else 286)
    roof["whole_step_hbm_frac_vs_survey_model"] = survey_doubles * 8 * ncell / (step_ms * 1e-3) * 1e-9 / hbm_peak

    # ---- end to end through the C-ABI with host buffers ---------------------------------------
    e2e = None
    if rank == 0 or world > 1:
        # the call a user makes to advance a host-resident state by one step: conserved state in, conserved state out
        # (primitives are recovered on the device; no guess is sent, none is read back)
        nc = B.NCONS[p["model"]]
        cons_h = torch.empty((nc, nz, ny, nx), dtype=torch.float64, pin_memory=True)
        B.rmhd_get_state(sim.ctx, cons_h, None)
        e_steps = max(1, min(args.steps, 3))
        barrier()
        ev0.record()
        for _ in range(e_steps):
            B.rmhd_set_cons(sim.ctx, cons_h, None)         # H2D of this step's input state
            sim.step(1)
            B.rmhd_get_state(sim.ctx, cons_h, None)        # D2H of the step's result
        ev1.record()
        barrier()
        e_rate, _ = whole_job_rate(ev0.elapsed_time(ev1), ncell * e_steps, dist, dev)
        e2e = {"value": e_rate, "unit": UNIT,
               "h2d_bytes_per_step": nc * ncell * 8, "d2h_bytes_per_step": nc * ncell * 8,
               "steps": e_steps, "call": "rmhd_set_cons(host cons) + rmhd_step(1) + rmhd_get_state(host cons), pinned host buffers"}
        del cons_h
    n_failed = stats["n_failed"]
    sim.close()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    cpu_base = None
    if world == 1 and not args.no_cpu_baseline:
        cpu_base, _, _ = time_oracle(cfg, synth, steps=12, warmup=0, budget_s=20.0, integrator=args.integrator)
        v1, s1 = time_oracle_one_thread(cfg, integrator=args.integrator)
        cpu_base["value_1thread"] = v1
        cpu_base["sample_1thread"] = s1
    launches = sum(v["launches"] for v in kt.values())
    state_bytes = ((5 if nstage == 3 else 4) * NC + NH + 2 * NS) * ncell * 8
    # Three cases, not two: a working set between 1x and 4x the L2 is neither resident nor streamed from HBM every launch (each launch
    # touches 1/3 to 1/2 of the state arrays, and the previous launch's output is still partly in L2 when the next one reads it)
    L2_BYTES = 126e6
    if state_bytes <= L2_BYTES:
        l2_res = "fits"
        l2_note = ("state arrays (%.1f MB) fit in the 126 MB L2: this workload is timed L2-resident (launch-bound), as it runs in "
                   "production; no flush; the HBM fractions are L2-assisted" % (state_bytes / 1e6))
    elif state_bytes <= 4 * L2_BYTES:
        l2_res = "partly resident"
        l2_note = ("state arrays (%.1f MB) are 1-4x the 126 MB L2: partly L2-resident from launch to launch, as it runs in production; "
                   "no flush; the HBM fractions are L2-assisted" % (state_bytes / 1e6))
    else:
        l2_res = "exceeds"
        l2_note = "state arrays (%.2f GB) exceed the 126 MB L2 several times; no flush needed" % (state_bytes / 1e9)
    roof["l2_residency"] = l2_res
    roof["l2_assisted"] = l2_res != "exceeds"      # true: hbm_frac / whole_step_hbm_frac count bytes that partly never left the L2
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{cfg['name']}: {nx}x{ny}x{nz} cells, {'resistive' if p['model'] == 0 else 'two_fluid'}, "
                               f"{'SSP3(332)' if nstage == 3 else 'SSP2(222)'}, cfl {p['cfl']}, sigma {p.get('sigma')}",
                   "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": l2_note,
                   "n_failed_cells": int(n_failed),
                   "stage_iters_mean": float((stats["hist_stage"] * np.arange(stats["hist_stage"].size)).sum() / max(stats["hist_stage"].sum(), 1))},
        "clocks": clk.summary(), "e2e": e2e, "gpu_launches": int(launches),
        "roofline": roof, "cpu_baseline": cpu_base,
    }
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5")
    ap.add_argument("--integrator", default="ssp2", choices=["ssp2", "ssp3"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        # started plainly (`python bench.py --gpus N`): become the launcher the driver would have used, one rank per GPU,
        # replicas only.  The ranks' output (rank 0's JSON line, NCCL's log) passes through.
        import socket
        import subprocess
        with socket.socket() as so:
            so.bind(("127.0.0.1", 0))
            port = so.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus != world:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}: the launcher's --nproc-per-node and --gpus must agree")
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

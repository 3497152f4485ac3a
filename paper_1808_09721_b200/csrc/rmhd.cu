// rmhd.cu -- C-ABI of librmhd.so (include/rmhd.h): context, launches, copies.  No CPU fallback.
#include "rmhd.h"

#include <climits>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "kernels.cuh"
#include "flux_fused.cuh"
#include "flux_hm.cuh"

using namespace rmhd;

namespace {

enum { KC_STAGE1 = 0, KC_STAGE2 = 1, KC_FLUX = 2, KC_FINAL = 3, KC_OTHER = 4, KC_N = 5 };

thread_local std::string g_create_error;

struct EvRec { int cls; cudaEvent_t a, b; };

}  // namespace

struct rmhd_ctx {
  rmhd_params p;
  DevPar P;
  int model, nc, nh, ns, np;
  int n[3];
  size_t N;
  double dx[3], dt;
  long long nsteps;
  int device;
  cudaStream_t stream;
  double *q, *w, *qs, *L1, *L2, *Ps1, *Ps2, *A;   // A: eq-(11) partial sum, SSP3(332) only (SSP2 keeps it in L2)
  Stats* d_stats;
  Stats* h_stats;  // pinned
  bool profiling;
  bool fused_flux;   // one-pass L(q) over all axes (flux_hm.cuh) when nx, ny > 1; RMHD_FLUX=split (see rmhd.h) forces the per-axis kernels
  int hm_ty;         // tile rows of the two-role flux kernel: 8 (one 16-warp CTA per SM) when ny >= 8, else 4 (two CTAs)
  int sm_count;
  // small grids are launch-bound: one step's launch sequence is captured once into a CUDA graph and replayed (rmhd_step)
  cudaGraphExec_t step_graph;
  cudaStream_t cap_stream;
  bool graph_failed;
  bool capturing;                    // build_step_graph is recording: launches are counted into graph_launches, not launches
  long long graph_launches[5];       // launches of one captured step per kernel class, added to `launches` at every replay
  std::vector<EvRec> pending;
  std::vector<cudaEvent_t> ev_pool;
  double ms[KC_N];
  long long launches[KC_N];
  std::string err;
};

namespace {

struct DeviceGuard {
  int prev;
  bool ok;
  explicit DeviceGuard(int dev) : prev(-1), ok(true) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; prev = -1; }
    if (cudaSetDevice(dev) != cudaSuccess) ok = false;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

int fail_cuda(rmhd_ctx* c, cudaError_t e, const char* what) {
  char buf[256];
  snprintf(buf, sizeof buf, "CUDA error in %s: %s", what, cudaGetErrorString(e));
  if (c) c->err = buf; else g_create_error = buf;
  return RMHD_ERR_CUDA;
}
#define CK(c, call)                                              \
  do {                                                           \
    cudaError_t e__ = (call);                                    \
    if (e__ != cudaSuccess) return fail_cuda((c), e__, #call);   \
  } while (0)

int make_devpar(const rmhd_params* p, DevPar& P, std::string& err) {
  if (p->model != RMHD_RESISTIVE && p->model != RMHD_TWO_FLUID) { err = "model must be RMHD_RESISTIVE or RMHD_TWO_FLUID"; return RMHD_ERR_BAD_PARAM; }
  if (!(p->gamma > 1.0)) { err = "gamma must be > 1"; return RMHD_ERR_BAD_PARAM; }
  if (p->model == RMHD_TWO_FLUID && p->mu_e == p->mu_p) { err = "mu_e must differ from mu_p"; return RMHD_ERR_BAD_PARAM; }
  if (p->model == RMHD_RESISTIVE && !(p->sigma >= 0.0)) { err = "sigma must be >= 0"; return RMHD_ERR_BAD_PARAM; }
  P.gam = p->gamma; P.g = (p->gamma - 1.0) / p->gamma; P.gi = p->gamma / (p->gamma - 1.0);
  P.sigma = p->sigma; P.eta = p->eta; P.mu_e = p->mu_e; P.mu_p = p->mu_p; P.kappa = p->kappa;
  P.tol_c2p = p->tol_c2p > 0 ? p->tol_c2p : 1e-13;
  P.tol_stage = p->tol_stage > 0 ? p->tol_stage : 1e-12;
  P.maxit_c2p = p->max_iter_c2p > 0 ? p->max_iter_c2p : 100;
  P.maxit_stage = p->max_iter_stage > 0 ? p->max_iter_stage : 50;
  return RMHD_OK;
}

inline unsigned blocks_for(size_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

// ---- profiling helpers -------------------------------------------------------------------
cudaEvent_t get_event(rmhd_ctx* c) {
  if (!c->ev_pool.empty()) { cudaEvent_t e = c->ev_pool.back(); c->ev_pool.pop_back(); return e; }
  cudaEvent_t e; cudaEventCreate(&e); return e;
}
struct Timed {
  rmhd_ctx* c; int cls; cudaEvent_t a, b;
  Timed(rmhd_ctx* c_, int cls_) : c(c_), cls(cls_), a(nullptr), b(nullptr) {
    if (c->capturing) c->graph_launches[cls]++; else c->launches[cls]++;
    if (c->profiling) { a = get_event(c); b = get_event(c); cudaEventRecord(a, c->stream); }
  }
  ~Timed() { if (c->profiling) { cudaEventRecord(b, c->stream); c->pending.push_back({cls, a, b}); } }
};
void resolve_events(rmhd_ctx* c) {  // stream must be synchronised
  for (auto& r : c->pending) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess) c->ms[r.cls] += ms;
    c->ev_pool.push_back(r.a); c->ev_pool.push_back(r.b);
  }
  c->pending.clear();
}

// ---- launches ----------------------------------------------------------------------------
template <int MODEL, int AXIS>
int launch_flux_axis(rmhd_ctx* c, const ConsRows<MODEL>& qr, const HydRows<MODEL>& wr, double* L, int accumulate) {
  const int nx = c->n[0], ny = c->n[1], nz = c->n[2];
  const int ns = c->n[AXIS];
  if constexpr (AXIS == 0) {
    constexpr int TS = Tile<AXIS>::TS, TO = Tile<AXIS>::TO;
    const size_t smem = flux_smem_bytes<MODEL, AXIS>();
    CK(c, cudaFuncSetAttribute(k_flux<MODEL, AXIS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    dim3 grid((ny * nz + TO - 1) / TO, (ns + TS - 1) / TS, 1);
    if (ny * nz == 1) grid = dim3(1, (ns + TS * TO - 1) / (TS * TO), 1);   // 1-D: the tile rows are laid along x
    Timed t(c, KC_FLUX);
    k_flux<MODEL, AXIS><<<grid, FLUX_THREADS, smem, c->stream>>>(qr, wr, L, c->N, nx, ny, nz, c->p.bc[AXIS], 1.0 / c->dx[AXIS], accumulate, c->P);
    CK(c, cudaGetLastError());
  } else {
    const size_t smem = march_smem_bytes<MODEL>();
    CK(c, cudaFuncSetAttribute(k_flux_march<MODEL, AXIS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    // segments along the sweep axis: enough threads for ~8 resident waves-worth of columns, segments >= 8 cells
    const long long columns = (long long)((nx + MARCH_THREADS - 1) / MARCH_THREADS) * MARCH_THREADS * (AXIS == 1 ? nz : ny);
    const long long want_threads = 148LL * 384 * 4;
    int nseg = (int)((want_threads + columns - 1) / columns);
    if (nseg < 1) nseg = 1;
    if (nseg > (ns + 7) / 8) nseg = (ns + 7) / 8;
    if (nseg > 65535) nseg = 65535;
    const int seg_len = (ns + nseg - 1) / nseg;
    nseg = (ns + seg_len - 1) / seg_len;
    dim3 grid((nx + MARCH_THREADS - 1) / MARCH_THREADS, AXIS == 1 ? nz : ny, nseg);
    Timed t(c, KC_FLUX);
    k_flux_march<MODEL, AXIS><<<grid, MARCH_THREADS, smem, c->stream>>>(qr, wr, L, c->N, nx, ny, nz, c->p.bc[AXIS], 1.0 / c->dx[AXIS], accumulate, seg_len, c->P);
    CK(c, cudaGetLastError());
  }
  return RMHD_OK;
}

// all present axes in one pass (flux_hm.cuh); needs nx > 1 and ny > 1.  TYP: tile rows of the two-role kernel
template <int MODEL, bool HAS_Z, bool COMB, int TYP>
int launch_flux_fused(rmhd_ctx* c, const ConsRows<MODEL>& qr, const HydRows<MODEL>& wr, double* L, const FluxComb& cb) {
  const int nx = c->n[0], ny = c->n[1], nz = c->n[2];
  const size_t smem = HMGeom<TYP, MODEL>::bytes(HAS_Z);
  CK(c, cudaFuncSetAttribute(k_flux_hm<HAS_Z, COMB, TYP, true, 2, MODEL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int gx = (nx + FF_TX - 1) / FF_TX, gy = (ny + TYP - 1) / TYP;
  int nseg = 1, seg_len = 1;
  if (HAS_Z) {
    // z segments: pick the count (segments of >= 16 planes) that wastes least, counting the partially filled
    // last wave of resident CTAs and the 4 feed-only prologue planes of every segment
    const bool one_cta = TYP == 8 || MODEL == 1;
    const long long tiles = (long long)gx * gy, slots = (one_cta ? 1LL : 2LL) * c->sm_count;
    double best = 1e300;
    for (int s = 1; s <= (nz + 15) / 16 && s <= 64; ++s) {
      const int len = (nz + s - 1) / s, cnt = (nz + len - 1) / len;
      const long long ctas = tiles * cnt, waves = (ctas + slots - 1) / slots;
      const double cost = (double)waves * slots / (double)ctas * (1.0 + 3.0 / len);
      if (cost < best - 1e-9) { best = cost; nseg = cnt; seg_len = len; }
    }
  }
  dim3 grid(gx, gy, nseg);
  Timed t(c, KC_FLUX);
  k_flux_hm<HAS_Z, COMB, TYP, true, 2, MODEL><<<grid, HMGeom<TYP, MODEL>::THREADS, smem, c->stream>>>(
      qr, wr, L, c->N, nx, ny, nz, c->p.bc[0], c->p.bc[1], c->p.bc[2], 0.5 / c->dx[0], 0.5 / c->dx[1], 0.5 / c->dx[2], seg_len, c->P, cb);
  CK(c, cudaGetLastError());
  return RMHD_OK;
}
template <int MODEL, bool HAS_Z, bool COMB>
int launch_flux_fused(rmhd_ctx* c, const ConsRows<MODEL>& qr, const HydRows<MODEL>& wr, double* L, const FluxComb& cb) {
  if constexpr (MODEL == 0 || !HAS_Z) {     // 32 x 8 tiles: resistive always, two-fluid in 2-D (its 3-D ring does not fit)
    if (c->hm_ty == 8) return launch_flux_fused<MODEL, HAS_Z, COMB, 8>(c, qr, wr, L, cb);
  }
  return launch_flux_fused<MODEL, HAS_Z, COMB, 4>(c, qr, wr, L, cb);
}

// resistive 2-D grids: the two-role kernel with the tile rows laid along x and the grid's y axis as the marching axis
// (flux_hm.cuh, HAS_Y = false, ZDIR = 1)
template <bool COMB>
int launch_flux_march2d(rmhd_ctx* c, const ConsRows<0>& qr, const HydRows<0>& wr, double* L, const FluxComb& cb) {
  constexpr int TYP = 8;
  const int nx = c->n[0], ny = c->n[1];
  const size_t smem = HMGeom<TYP>::bytes(true);
  CK(c, cudaFuncSetAttribute(k_flux_hm<true, COMB, TYP, false, 1, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int gx = (nx + FF_TX * TYP - 1) / (FF_TX * TYP);
  // segments along y: fill the SMs (one CTA each), at least 4 planes per segment, then the same waste measure as in 3-D
  int nseg = 1, seg_len = ny;
  {
    const long long slots = c->sm_count;
    double best = 1e300;
    for (int s = 1; s <= (ny + 3) / 4 && s <= 4096; ++s) {
      const int len = (ny + s - 1) / s, cnt = (ny + len - 1) / len;
      const long long ctas = (long long)gx * cnt, waves = (ctas + slots - 1) / slots;
      const double cost = (double)waves * slots / (double)ctas * (1.0 + 1.5 / len);   // 4 feed-only planes ~ 1.5 full ones
      if (cost < best - 1e-9) { best = cost; nseg = cnt; seg_len = len; }
    }
  }
  dim3 grid(gx, 1, nseg);
  Timed t(c, KC_FLUX);
  k_flux_hm<true, COMB, TYP, false, 1, 0><<<grid, HMGeom<TYP>::THREADS, smem, c->stream>>>(
      qr, wr, L, c->N, nx, 1, ny, c->p.bc[0], 0, c->p.bc[1], 0.5 / c->dx[0], 0.0, 0.5 / c->dx[1], seg_len, c->P, cb);
  CK(c, cudaGetLastError());
  return RMHD_OK;
}

inline bool uses_fused_flux(const rmhd_ctx* c) { return c->fused_flux && c->n[0] > 1 && c->n[1] > 1; }

// `cb` (fused path only): store the eq-(11) update of q instead of L (a5 fused into F2)
template <int MODEL>
int launch_flux(rmhd_ctx* c, const double* qa, const double* qb, bool mix, const double* w, double* L, const FluxComb* cb = nullptr) {
  constexpr int NC = Dim<MODEL>::NC, NH = Dim<MODEL>::NH, NS = Dim<MODEL>::NS;
  ConsRows<MODEL> qr; HydRows<MODEL> wr;
  for (int v = 0; v < NC; ++v) qr.r[v] = qa + (size_t)v * c->N;
  if (mix) for (int k = 0; k < NS; ++k) { int v = MODEL == 0 ? (k < 3 ? 8 + k : 9 + k) : (k < 4 ? 6 + k : 9 + k); qr.r[v] = qb + (size_t)v * c->N; }
  for (int v = 0; v < NH; ++v) wr.r[v] = w + (size_t)v * c->N;
  if (uses_fused_flux(c)) {
    const FluxComb none = {nullptr, nullptr, 0.0, nullptr, 0.0, 0};
    if constexpr (MODEL == 0) {
      if (c->n[2] == 1) return cb ? launch_flux_march2d<true>(c, qr, wr, L, *cb) : launch_flux_march2d<false>(c, qr, wr, L, none);
    }
    if (cb) return c->n[2] > 1 ? launch_flux_fused<MODEL, true, true>(c, qr, wr, L, *cb) : launch_flux_fused<MODEL, false, true>(c, qr, wr, L, *cb);
    return c->n[2] > 1 ? launch_flux_fused<MODEL, true, false>(c, qr, wr, L, none) : launch_flux_fused<MODEL, false, false>(c, qr, wr, L, none);
  }
  if (cb) { c->err = "internal: combine epilogue needs the fused flux kernel"; return RMHD_ERR_BAD_PARAM; }
  int acc = 0, rc;
  if (c->n[0] > 1) { if ((rc = launch_flux_axis<MODEL, 0>(c, qr, wr, L, acc))) return rc; acc = 1; }
  if (c->n[1] > 1) { if ((rc = launch_flux_axis<MODEL, 1>(c, qr, wr, L, acc))) return rc; acc = 1; }
  if (c->n[2] > 1) { if ((rc = launch_flux_axis<MODEL, 2>(c, qr, wr, L, acc))) return rc; acc = 1; }
  if (!acc) CK(c, cudaMemsetAsync(L, 0, sizeof(double) * NC * c->N, c->stream));
  return RMHD_OK;
}

template <int MODEL, int NL, bool MKA>
int launch_stage(rmhd_ctx* c, int cls, const StageCoef& k, double* Ps_out, double* A) {
  const unsigned nb = blocks_for(c->N, 128);
  Timed t(c, cls);
  if (MODEL == 0) k_stage_resistive<NL, MKA><<<nb, 128, 0, c->stream>>>(c->q, c->L1, c->L2, c->Ps1, c->Ps2, c->w, c->qs, Ps_out, A, c->N, k, c->P, c->d_stats);
  else k_stage_two_fluid<NL, MKA><<<nb, 128, 0, c->stream>>>(c->q, c->L1, c->L2, c->Ps1, c->Ps2, c->w, c->qs, Ps_out, A, c->N, k, c->P, c->d_stats);
  CK(c, cudaGetLastError());
  return RMHD_OK;
}

template <int MODEL>
int launch_con2prim(rmhd_ctx* c) {   // P: w^{n+1} = con2prim(q^{n+1}), guess = the last stage's primitives
  Timed t(c, KC_FINAL);
  k_con2prim<MODEL><<<blocks_for(c->N, 256), 256, 0, c->stream>>>(c->q, c->w, c->N, c->w, c->N, nullptr, nullptr, nullptr, c->N, c->P, c->d_stats);
  CK(c, cudaGetLastError());
  return RMHD_OK;
}

// one SSP2(222) step, Table 2
template <int MODEL>
int step_once(rmhd_ctx* c) {
  const double g = 1.0 - 1.0 / sqrt(2.0);
  const double dt = c->dt;
  int rc;
  StageCoef k1 = {};
  k1.a = g * dt;
  if ((rc = launch_stage<MODEL, 0, false>(c, KC_STAGE1, k1, c->Ps1, nullptr))) return rc;
  const bool fuse_c = uses_fused_flux(c);
  // F1 on the fused path also leaves q_ex of stage 2 for the rows without a source (qn + dt L1) in the stage-state buffer
  const bool pre = fuse_c;
  if (pre) {
    const FluxComb cb1 = {c->qs, nullptr, dt, c->q, 0.0, 1};
    if ((rc = launch_flux<MODEL>(c, c->q, c->qs, true, c->w, c->L1, &cb1))) return rc;
  } else if ((rc = launch_flux<MODEL>(c, c->q, c->qs, true, c->w, c->L1))) return rc;
  StageCoef k2 = {};
  k2.pre = pre;
  k2.a = g * dt; k2.cL[0] = dt; k2.cP[0] = (1.0 - 2.0 * g) * dt;
  k2.hL[0] = 0.5 * dt; k2.hP[0] = 0.5 * dt; k2.hP[2] = 0.5 * dt;
  if (fuse_c) {
    // stage 2 leaves A = qn + dt/2 L1 + dt/2 (Psi1 + Psi2) in the L2 buffer; F2 + C in one launch
    // (q^{n+1} = A + dt/2 L2 row by row in the flux kernel's epilogue), then P
    k2.a_src_only = true;
    if ((rc = launch_stage<MODEL, 1, true>(c, KC_STAGE2, k2, nullptr, c->L2))) return rc;
    const FluxComb cb = {c->q, c->L2, 0.5 * dt, c->qs, 0.5, 0};
    if ((rc = launch_flux<MODEL>(c, c->qs, nullptr, false, c->w, c->L2, &cb))) return rc;
    return launch_con2prim<MODEL>(c);
  }
  if ((rc = launch_stage<MODEL, 1, false>(c, KC_STAGE2, k2, c->Ps2, nullptr))) return rc;
  if ((rc = launch_flux<MODEL>(c, c->qs, nullptr, false, c->w, c->L2))) return rc;
  {
    Timed t(c, KC_FINAL);
    k_final<MODEL><<<blocks_for(c->N, 256), 256, 0, c->stream>>>(c->q, c->L1, c->L2, c->Ps1, c->Ps2, c->w, c->N, 0.5 * dt, c->P, c->d_stats);
    CK(c, cudaGetLastError());
  }
  return RMHD_OK;
}

// one SSP3(332) step, Table 3 P:L174-180 (reading G13):
//   S1 q1 = qn + g dt Psi1;  F1;  S2 q2 = qn + dt L1 + (1-2g) dt Psi1 + g dt Psi2;  F2;
//   S3 q3 = qn + dt/4 (L1 + L2) + (1/2-g) dt Psi1 + g dt Psi3, which also leaves
//      A = qn + dt/6 (L1 + L2) + dt/6 (Psi1 + Psi2) + 2dt/3 Psi3;   F3 + C: q^{n+1} = A + 2dt/3 L3;   P
template <int MODEL>
int step_once_ssp3(rmhd_ctx* c) {
  const double g = 1.0 - 1.0 / sqrt(2.0);
  const double dt = c->dt;
  int rc;
  StageCoef k1 = {};
  k1.a = g * dt;
  if ((rc = launch_stage<MODEL, 0, false>(c, KC_STAGE1, k1, c->Ps1, nullptr))) return rc;
  if ((rc = launch_flux<MODEL>(c, c->q, c->qs, true, c->w, c->L1))) return rc;
  StageCoef k2 = {};
  k2.a = g * dt; k2.cL[0] = dt; k2.cP[0] = (1.0 - 2.0 * g) * dt;
  if ((rc = launch_stage<MODEL, 1, false>(c, KC_STAGE2, k2, c->Ps2, nullptr))) return rc;
  if ((rc = launch_flux<MODEL>(c, c->qs, nullptr, false, c->w, c->L2))) return rc;
  StageCoef k3 = {};
  k3.a = g * dt; k3.cL[0] = 0.25 * dt; k3.cL[1] = 0.25 * dt; k3.cP[0] = (0.5 - g) * dt; k3.cP[1] = 0.0;
  k3.hL[0] = dt / 6.0; k3.hL[1] = dt / 6.0; k3.hP[0] = dt / 6.0; k3.hP[1] = dt / 6.0; k3.hP[2] = 2.0 * dt / 3.0;
  const bool fuse3 = uses_fused_flux(c);
  k3.a_src_only = fuse3;
  if ((rc = launch_stage<MODEL, 2, true>(c, KC_STAGE2, k3, nullptr, c->A))) return rc;
  const double wl = 2.0 * dt / 3.0;
  if (fuse3) {
    const FluxComb cb = {c->q, c->A, wl, c->qs, 2.0 / 3.0, 0};
    if ((rc = launch_flux<MODEL>(c, c->qs, nullptr, false, c->w, c->L1, &cb))) return rc;
    return launch_con2prim<MODEL>(c);
  }
  if ((rc = launch_flux<MODEL>(c, c->qs, nullptr, false, c->w, c->L1))) return rc;   // L3 into the L1 buffer (L1 is folded into A)
  {
    Timed t(c, KC_FINAL);
    k_final_A<MODEL><<<blocks_for(c->N, 256), 256, 0, c->stream>>>(c->q, c->A, c->L1, c->w, c->N, wl, c->P, c->d_stats);
    CK(c, cudaGetLastError());
  }
  return RMHD_OK;
}

int step_any(rmhd_ctx* c) {
  if (c->p.integrator == RMHD_SSP3_332) return c->model == 0 ? step_once_ssp3<0>(c) : step_once_ssp3<1>(c);
  return c->model == 0 ? step_once<0>(c) : step_once<1>(c);
}

constexpr size_t GRAPH_MAX_CELLS = (size_t)1 << 21;

// Capture one step on a private stream (the caller's may be the legacy default stream, which cannot be captured) and
// instantiate it; the graph is launched into the caller's stream.  Any failure leaves the plain launch path in force.
void build_step_graph(rmhd_ctx* c) {
  c->graph_failed = true;
  if (!c->cap_stream && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return; }
  cudaStream_t user = c->stream;
  cudaGraph_t g = nullptr;
  if (cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) { cudaGetLastError(); return; }
  c->stream = c->cap_stream;
  c->capturing = true;
  for (int i = 0; i < KC_N; ++i) c->graph_launches[i] = 0;
  const int rc = step_any(c);
  c->capturing = false;
  c->stream = user;
  const cudaError_t e = cudaStreamEndCapture(c->cap_stream, &g);
  if (rc != RMHD_OK || e != cudaSuccess || !g) { if (g) cudaGraphDestroy(g); cudaGetLastError(); c->err.clear(); return; }
  if (cudaGraphInstantiate(&c->step_graph, g, 0) != cudaSuccess) { c->step_graph = nullptr; cudaGetLastError(); }
  else c->graph_failed = false;
  cudaGraphDestroy(g);
}

int read_stats(rmhd_ctx* c) {
  CK(c, cudaMemcpyAsync(c->h_stats, c->d_stats, sizeof(Stats), cudaMemcpyDeviceToHost, c->stream));
  CK(c, cudaStreamSynchronize(c->stream));
  resolve_events(c);
  return RMHD_OK;
}

int reset_stats(rmhd_ctx* c) {
  memset(c->h_stats, 0, sizeof(Stats));
  c->h_stats->first_failed = LLONG_MAX;
  CK(c, cudaMemcpyAsync(c->d_stats, c->h_stats, sizeof(Stats), cudaMemcpyHostToDevice, c->stream));
  return RMHD_OK;
}

}  // namespace

// =========================================================================================
extern "C" {

int rmhd_create(const rmhd_params* p, rmhd_ctx** out) {
  if (!p || !out) { g_create_error = "null argument"; return RMHD_ERR_BAD_PARAM; }
  *out = nullptr;
  DevPar P;
  int rc = make_devpar(p, P, g_create_error);
  if (rc) return rc;
  if (p->integrator != RMHD_SSP2_222 && p->integrator != RMHD_SSP3_332) { g_create_error = "integrator must be RMHD_SSP2_222 or RMHD_SSP3_332"; return RMHD_ERR_BAD_PARAM; }
  if (p->nx < 1 || p->ny < 1 || p->nz < 1 || p->ng < 2 || !(p->cfl > 0.0)) { g_create_error = "bad grid size, ng < 2 or cfl <= 0"; return RMHD_ERR_BAD_PARAM; }
  for (int d = 0; d < 3; ++d) if (p->bc[d] != RMHD_BC_OUTFLOW && p->bc[d] != RMHD_BC_PERIODIC) { g_create_error = "bad boundary condition"; return RMHD_ERR_BAD_PARAM; }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0 || p->device < 0 || p->device >= ndev) {
    cudaGetLastError();
    g_create_error = "no CUDA device (this library has no CPU fallback)";
    return RMHD_ERR_CUDA;
  }
  rmhd_ctx* c = new rmhd_ctx();
  c->p = *p; c->P = P; c->model = p->model;
  c->nc = p->model == 0 ? R_NC : T_NC; c->nh = p->model == 0 ? R_NH : T_NH;
  c->ns = p->model == 0 ? R_NS : T_NS; c->np = p->model == 0 ? 11 : 16;
  c->n[0] = p->nx; c->n[1] = p->ny; c->n[2] = p->nz;
  c->N = (size_t)p->nx * p->ny * p->nz;
  if (c->N >= (size_t)1 << 31) { g_create_error = "grid too large: the kernels index a row with 32-bit offsets (N < 2^31)"; delete c; return RMHD_ERR_BAD_PARAM; }
  const double lo[3] = {p->xmin, p->ymin, p->zmin}, hi[3] = {p->xmax, p->ymax, p->zmax};
  double inv = 0.0;
  for (int d = 0; d < 3; ++d) {
    c->dx[d] = (hi[d] - lo[d]) / c->n[d];
    if (c->n[d] > 1) {
      if (!(c->dx[d] > 0.0)) { g_create_error = "empty domain"; delete c; return RMHD_ERR_BAD_PARAM; }
      inv += 1.0 / c->dx[d];
    }
  }
  c->dt = inv > 0.0 ? p->cfl / inv : p->cfl;   // G9
  c->nsteps = 0; c->device = p->device; c->stream = (cudaStream_t)p->stream;
  c->profiling = false;
  { const char* e = getenv("RMHD_FLUX"); c->fused_flux = !(e && strcmp(e, "split") == 0); }   // documented in rmhd.h
  c->hm_ty = p->ny >= 8 ? 8 : 4;
  c->sm_count = 148;
  for (int i = 0; i < KC_N; ++i) { c->ms[i] = 0.0; c->launches[i] = 0; }
  c->q = c->w = c->qs = c->L1 = c->L2 = c->Ps1 = c->Ps2 = c->A = nullptr; c->d_stats = nullptr; c->h_stats = nullptr;
  c->step_graph = nullptr; c->cap_stream = nullptr; c->graph_failed = false; c->capturing = false;
  for (int i = 0; i < KC_N; ++i) c->graph_launches[i] = 0;
  DeviceGuard dg(c->device);
  { int n = 0; if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, c->device) == cudaSuccess && n > 0) c->sm_count = n; }
  const size_t rows = (size_t)((p->integrator == RMHD_SSP3_332 ? 5 : 4) * c->nc + c->nh + 2 * c->ns);
  cudaError_t e = cudaMalloc(&c->q, sizeof(double) * rows * c->N);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_stats, sizeof(Stats));
  if (e == cudaSuccess) e = cudaMallocHost(&c->h_stats, sizeof(Stats));
  if (e != cudaSuccess) { fail_cuda(nullptr, e, "allocating device state"); rmhd_destroy(c); return RMHD_ERR_CUDA; }
  double* b = c->q;
  b += (size_t)c->nc * c->N; c->qs = b;
  b += (size_t)c->nc * c->N; c->L1 = b;
  b += (size_t)c->nc * c->N; c->L2 = b;
  b += (size_t)c->nc * c->N; c->w = b;
  b += (size_t)c->nh * c->N; c->Ps1 = b;
  b += (size_t)c->ns * c->N; c->Ps2 = b;
  if (p->integrator == RMHD_SSP3_332) { b += (size_t)c->ns * c->N; c->A = b; }
  e = cudaMemsetAsync(c->q, 0, sizeof(double) * rows * c->N, c->stream);
  if (e != cudaSuccess) { fail_cuda(nullptr, e, "clearing device state"); rmhd_destroy(c); return RMHD_ERR_CUDA; }
  if (reset_stats(c)) { g_create_error = c->err; rmhd_destroy(c); return RMHD_ERR_CUDA; }
  *out = c;
  return RMHD_OK;
}

void rmhd_destroy(rmhd_ctx* c) {
  if (!c) return;
  {
    DeviceGuard dg(c->device);
    if (c->stream || c->q) cudaStreamSynchronize(c->stream);
    for (auto& r : c->pending) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (auto& e : c->ev_pool) cudaEventDestroy(e);
    if (c->step_graph) cudaGraphExecDestroy(c->step_graph);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    if (c->q) cudaFree(c->q);
    if (c->d_stats) cudaFree(c->d_stats);
    if (c->h_stats) cudaFreeHost(c->h_stats);
  }
  delete c;
}

double rmhd_dt(const rmhd_ctx* c) { return c ? c->dt : 0.0; }
double rmhd_time(const rmhd_ctx* c) { return c ? (double)c->nsteps * c->dt : 0.0; }
const char* rmhd_last_error(const rmhd_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

int rmhd_set_initial(rmhd_ctx* c, const double* prims, const double* rho_charge, int on_device) {
  if (!c || !prims) return RMHD_ERR_BAD_PARAM;
  DeviceGuard dg(c->device);
  const size_t N = c->N;
  const double* d_prims = prims;
  const double* d_rc = rho_charge;
  if (!on_device) {  // stage through qs (nc >= np rows) and L2 (one row)
    CK(c, cudaMemcpyAsync(c->qs, prims, sizeof(double) * c->np * N, cudaMemcpyHostToDevice, c->stream));
    d_prims = c->qs;
    if (rho_charge) { CK(c, cudaMemcpyAsync(c->L2, rho_charge, sizeof(double) * N, cudaMemcpyHostToDevice, c->stream)); d_rc = c->L2; }
  }
  int rc = reset_stats(c);
  if (rc) return rc;
  const double i2[3] = {0.5 / c->dx[0], 0.5 / c->dx[1], 0.5 / c->dx[2]};
  {
    Timed t(c, KC_OTHER);
    if (c->model == 0)
      k_set_initial<0><<<blocks_for(N, 256), 256, 0, c->stream>>>(d_prims, d_rc, c->q, c->w, N, c->n[0], c->n[1], c->n[2], c->p.bc[0], c->p.bc[1], c->p.bc[2], i2[0], i2[1], i2[2], c->P, c->d_stats);
    else
      k_set_initial<1><<<blocks_for(N, 256), 256, 0, c->stream>>>(d_prims, nullptr, c->q, c->w, N, c->n[0], c->n[1], c->n[2], c->p.bc[0], c->p.bc[1], c->p.bc[2], i2[0], i2[1], i2[2], c->P, c->d_stats);
    CK(c, cudaGetLastError());
  }
  c->nsteps = 0;
  if ((rc = read_stats(c))) return rc;
  if (c->h_stats->n_bad_input) { c->err = "set_initial: cells with rho <= 0, p <= 0 or |v| >= 1"; return RMHD_ERR_UNPHYSICAL_INPUT; }
  return RMHD_OK;
}

int rmhd_set_cons(rmhd_ctx* c, const double* cons, const double* prim_guess, int on_device) {
  if (!c || !cons) return RMHD_ERR_BAD_PARAM;
  DeviceGuard dg(c->device);
  const size_t N = c->N;
  CK(c, cudaMemcpyAsync(c->q, cons, sizeof(double) * c->nc * N, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
  { int rc0 = reset_stats(c); if (rc0) return rc0; }
  const double* d_guess = prim_guess;
  if (prim_guess && !on_device) {
    CK(c, cudaMemcpyAsync(c->qs, prim_guess, sizeof(double) * c->nh * N, cudaMemcpyHostToDevice, c->stream));
    d_guess = c->qs;
  }
  {
    Timed t(c, KC_OTHER);
    if (c->model == 0) k_con2prim<0><<<blocks_for(N, 256), 256, 0, c->stream>>>(c->q, d_guess, N, c->w, N, nullptr, nullptr, nullptr, N, c->P, c->d_stats);
    else k_con2prim<1><<<blocks_for(N, 256), 256, 0, c->stream>>>(c->q, d_guess, N, c->w, N, nullptr, nullptr, nullptr, N, c->P, c->d_stats);
    CK(c, cudaGetLastError());
  }
  int rc = read_stats(c);
  if (rc) return rc;
  return c->h_stats->n_failed ? RMHD_ERR_NONCONVERGED : RMHD_OK;
}

int rmhd_step(rmhd_ctx* c, int nsteps) {
  if (!c || nsteps < 0) return RMHD_ERR_BAD_PARAM;
  DeviceGuard dg(c->device);
  // Grids below GRAPH_MAX_CELLS are bound by launch latency (cfg1: 128 cells, 5 launches of a few microseconds each): the
  // launch sequence of one step is the same every step (constant dt, fixed buffers), so it is captured once and replayed.
  if (!c->profiling && nsteps >= 1 && c->N <= GRAPH_MAX_CELLS && !c->step_graph && !c->graph_failed) build_step_graph(c);
  for (int s = 0; s < nsteps; ++s) {
    int rc;
    if (c->step_graph && !c->profiling) {
      CK(c, cudaGraphLaunch(c->step_graph, c->stream));
      for (int i = 0; i < KC_N; ++i) c->launches[i] += c->graph_launches[i];
      rc = RMHD_OK;
    } else rc = step_any(c);
    if (rc) return rc;
    c->nsteps++;
  }
  int rc = read_stats(c);
  if (rc) return rc;
  if (c->h_stats->n_failed) { c->err = "root-find failed in some cells (see rmhd_get_stats)"; return RMHD_ERR_NONCONVERGED; }
  return RMHD_OK;
}

int rmhd_get_state(rmhd_ctx* c, double* cons, double* prims, int on_device) {
  if (!c) return RMHD_ERR_BAD_PARAM;
  DeviceGuard dg(c->device);
  const size_t N = c->N;
  const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  if (cons) CK(c, cudaMemcpyAsync(cons, c->q, sizeof(double) * c->nc * N, kind, c->stream));
  if (prims) {
    const int ib = c->model == 0 ? 5 : 10;   // B, E rows are contiguous in the conserved state
    CK(c, cudaMemcpyAsync(prims, c->w, sizeof(double) * c->nh * N, kind, c->stream));
    CK(c, cudaMemcpyAsync(prims + (size_t)c->nh * N, c->q + (size_t)ib * N, sizeof(double) * 6 * N, kind, c->stream));
  }
  CK(c, cudaStreamSynchronize(c->stream));
  return RMHD_OK;
}

int rmhd_flux_divergence(rmhd_ctx* c, double* Lout, int on_device) {
  if (!c || !Lout) return RMHD_ERR_BAD_PARAM;
  DeviceGuard dg(c->device);
  int rc = c->model == 0 ? launch_flux<0>(c, c->q, nullptr, false, c->w, c->L1) : launch_flux<1>(c, c->q, nullptr, false, c->w, c->L1);
  if (rc) return rc;
  CK(c, cudaMemcpyAsync(Lout, c->L1, sizeof(double) * c->nc * c->N, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
  CK(c, cudaStreamSynchronize(c->stream));
  resolve_events(c);
  return RMHD_OK;
}

int rmhd_get_stats(rmhd_ctx* c, long long* hist_stage, long long* hist_c2p, int nbins, long long* n_failed, long long* first_failed_cell) {
  if (!c || nbins < 0) return RMHD_ERR_BAD_PARAM;
  DeviceGuard dg(c->device);
  int rc = read_stats(c);
  if (rc) return rc;
  for (int b = 0; b < nbins; ++b) {
    if (hist_stage) hist_stage[b] = 0;
    if (hist_c2p) hist_c2p[b] = 0;
  }
  for (int b = 0; b < NBINS; ++b) {   // fold the library's bins into the caller's (overflow -> last bin)
    const int t = b < nbins ? b : nbins - 1;
    if (t < 0) break;
    if (hist_stage) hist_stage[t] += (long long)c->h_stats->hist_stage[b];
    if (hist_c2p) hist_c2p[t] += (long long)c->h_stats->hist_c2p[b];
  }
  if (n_failed) *n_failed = (long long)c->h_stats->n_failed;
  if (first_failed_cell) *first_failed_cell = c->h_stats->first_failed == LLONG_MAX ? -1 : c->h_stats->first_failed;
  return RMHD_OK;
}

int rmhd_set_profiling(rmhd_ctx* c, int enabled) {
  if (!c) return RMHD_ERR_BAD_PARAM;
  DeviceGuard dg(c->device);
  CK(c, cudaStreamSynchronize(c->stream));
  resolve_events(c);
  c->profiling = enabled != 0;
  for (int i = 0; i < KC_N; ++i) { c->ms[i] = 0.0; c->launches[i] = 0; }
  return RMHD_OK;
}

int rmhd_get_kernel_times(rmhd_ctx* c, double* ms, long long* launches, int n) {
  if (!c) return RMHD_ERR_BAD_PARAM;
  DeviceGuard dg(c->device);
  CK(c, cudaStreamSynchronize(c->stream));
  resolve_events(c);
  for (int i = 0; i < n; ++i) {
    if (ms) ms[i] = i < KC_N ? c->ms[i] : 0.0;
    if (launches) launches[i] = i < KC_N ? c->launches[i] : 0;
  }
  return RMHD_OK;
}

}  // extern "C"

// ---- batched per-cell operations -----------------------------------------------------------
namespace {
// Device copies of host buffers for the on_device == 0 path.  They are carved out of ONE grow-only allocation per device that
// outlives the call (rmhd_release_staging frees it): a caller who feeds host batches in a loop pays cudaMalloc once, not
// up to seven cudaMalloc + cudaFree per call (each cudaFree synchronises the device).  The arena's mutex is held for the whole
// call: host-buffer batch calls on one process serialise, which they did in effect before (every one ends in a stream synchronise).
constexpr int STAGING_MAX_DEVICES = 64;
struct StagingArena { void* base; size_t cap; };
StagingArena g_staging[STAGING_MAX_DEVICES];
std::mutex g_staging_mu;
inline size_t staging_align(size_t b) { return (b + 255) & ~(size_t)255; }
struct Staging {
  cudaStream_t s;
  int dev;
  size_t used;
  std::unique_lock<std::mutex> lk;
  Staging(cudaStream_t s_, int dev_) : s(s_), dev(dev_), used(0), lk(g_staging_mu) {}
  // make room for `bytes` (the sum of staging_align(size) over the buffers of this call); the device must be current
  cudaError_t reserve(size_t bytes) {
    if (dev < 0 || dev >= STAGING_MAX_DEVICES) return cudaErrorInvalidDevice;
    StagingArena& a = g_staging[dev];
    if (a.cap >= bytes) return cudaSuccess;
    if (a.base) { cudaFree(a.base); a.base = nullptr; a.cap = 0; }
    const size_t want = (bytes + ((size_t)1 << 20) - 1) & ~(((size_t)1 << 20) - 1);
    const cudaError_t e = cudaMalloc(&a.base, want);
    if (e == cudaSuccess) a.cap = want; else a.base = nullptr;
    return e;
  }
  void* take(size_t bytes) { void* d = (char*)g_staging[dev].base + used; used += staging_align(bytes); return d; }
  template <class T> cudaError_t in(const T* host, size_t n, const T** dev_ptr) {
    if (!host) { *dev_ptr = nullptr; return cudaSuccess; }
    void* d = take(sizeof(T) * n); *dev_ptr = (const T*)d;
    return cudaMemcpyAsync(d, host, sizeof(T) * n, cudaMemcpyHostToDevice, s);
  }
  template <class T> cudaError_t out(T* host, size_t n, T** dev_ptr) {
    if (!host) { *dev_ptr = nullptr; return cudaSuccess; }
    *dev_ptr = (T*)take(sizeof(T) * n);
    return cudaSuccess;
  }
};
int batch_prologue(const rmhd_params* p, long long n, DevPar& P) {
  if (!p || n < 0) { g_create_error = "bad argument"; return RMHD_ERR_BAD_PARAM; }
  int rc = make_devpar(p, P, g_create_error);
  if (rc) return rc;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0 || p->device < 0 || p->device >= ndev) {
    cudaGetLastError(); g_create_error = "no CUDA device (this library has no CPU fallback)"; return RMHD_ERR_CUDA;
  }
  return RMHD_OK;
}
}  // namespace

extern "C" {

int rmhd_stage_batch(const rmhd_params* p, long long ncells, const double* q_ex, const double* prim_guess,
                     const double* sigma_cell, double a_dt, double* q_out, double* prims_out, int* iters, int* fail,
                     int on_device) {
  DevPar P;
  int rc = batch_prologue(p, ncells, P);
  if (rc) return rc;
  if (!q_ex || !prim_guess || !q_out || !prims_out) { g_create_error = "null buffer"; return RMHD_ERR_BAD_PARAM; }
  if (p->model == RMHD_TWO_FLUID && sigma_cell) { g_create_error = "sigma_cell is a resistive-model argument"; return RMHD_ERR_BAD_PARAM; }
  if (ncells == 0) return RMHD_OK;
  DeviceGuard dg(p->device);
  cudaStream_t s = (cudaStream_t)p->stream;
  const size_t N = (size_t)ncells;
  const int nc = p->model == 0 ? 14 : 18, np = p->model == 0 ? 11 : 16;
  const double *d_qex = q_ex, *d_pg = prim_guess, *d_sig = sigma_cell;
  double *d_qo = q_out, *d_po = prims_out; int *d_it = iters, *d_fl = fail;
  if (on_device) {
    if (p->model == 0) k_stage_batch_resistive<<<blocks_for(N, 128), 128, 0, s>>>(d_qex, d_pg, d_sig, a_dt, d_qo, d_po, d_it, d_fl, N, P);
    else k_stage_batch_two_fluid<<<blocks_for(N, 128), 128, 0, s>>>(d_qex, d_pg, a_dt, d_qo, d_po, d_it, d_fl, N, P);
    CK(nullptr, cudaGetLastError());
    return RMHD_OK;
  }
  Staging st(s, p->device);
  {
    const size_t D = sizeof(double), I = sizeof(int);
    CK(nullptr, st.reserve(2 * staging_align(D * nc * N) + 2 * staging_align(D * np * N) + (sigma_cell ? staging_align(D * N) : 0) +
                           (iters ? staging_align(I * N) : 0) + (fail ? staging_align(I * N) : 0)));
    CK(nullptr, st.in(q_ex, nc * N, &d_qex)); CK(nullptr, st.in(prim_guess, np * N, &d_pg)); CK(nullptr, st.in(sigma_cell, N, &d_sig));
    CK(nullptr, st.out(q_out, nc * N, &d_qo)); CK(nullptr, st.out(prims_out, np * N, &d_po));
    CK(nullptr, st.out(iters, N, &d_it)); CK(nullptr, st.out(fail, N, &d_fl));
  }
  if (p->model == 0) k_stage_batch_resistive<<<blocks_for(N, 128), 128, 0, s>>>(d_qex, d_pg, d_sig, a_dt, d_qo, d_po, d_it, d_fl, N, P);
  else k_stage_batch_two_fluid<<<blocks_for(N, 128), 128, 0, s>>>(d_qex, d_pg, a_dt, d_qo, d_po, d_it, d_fl, N, P);
  CK(nullptr, cudaGetLastError());
  if (!on_device) {
    CK(nullptr, cudaMemcpyAsync(q_out, d_qo, sizeof(double) * nc * N, cudaMemcpyDeviceToHost, s));
    CK(nullptr, cudaMemcpyAsync(prims_out, d_po, sizeof(double) * np * N, cudaMemcpyDeviceToHost, s));
    if (iters) CK(nullptr, cudaMemcpyAsync(iters, d_it, sizeof(int) * N, cudaMemcpyDeviceToHost, s));
    if (fail) CK(nullptr, cudaMemcpyAsync(fail, d_fl, sizeof(int) * N, cudaMemcpyDeviceToHost, s));
    CK(nullptr, cudaStreamSynchronize(s));
  }
  return RMHD_OK;
}

int rmhd_prim2cons_batch(const rmhd_params* p, long long ncells, const double* prims, const double* rho_charge, double* cons,
                         int on_device) {
  DevPar P;
  int rc = batch_prologue(p, ncells, P);
  if (rc) return rc;
  if (!prims || !cons) { g_create_error = "null buffer"; return RMHD_ERR_BAD_PARAM; }
  if (ncells == 0) return RMHD_OK;
  DeviceGuard dg(p->device);
  cudaStream_t s = (cudaStream_t)p->stream;
  const size_t N = (size_t)ncells;
  const int nc = p->model == 0 ? 14 : 18, np = p->model == 0 ? 11 : 16;
  const double *d_pr = prims, *d_rc = rho_charge; double* d_co = cons;
  if (on_device) {
    if (p->model == 0) k_prim2cons_batch<0><<<blocks_for(N, 256), 256, 0, s>>>(d_pr, d_rc, d_co, N, P);
    else k_prim2cons_batch<1><<<blocks_for(N, 256), 256, 0, s>>>(d_pr, nullptr, d_co, N, P);
    CK(nullptr, cudaGetLastError());
    return RMHD_OK;
  }
  Staging st(s, p->device);
  CK(nullptr, st.reserve(staging_align(sizeof(double) * np * N) + (rho_charge ? staging_align(sizeof(double) * N) : 0) + staging_align(sizeof(double) * nc * N)));
  if (!on_device) { CK(nullptr, st.in(prims, np * N, &d_pr)); CK(nullptr, st.in(rho_charge, N, &d_rc)); CK(nullptr, st.out(cons, nc * N, &d_co)); }
  if (p->model == 0) k_prim2cons_batch<0><<<blocks_for(N, 256), 256, 0, s>>>(d_pr, d_rc, d_co, N, P);
  else k_prim2cons_batch<1><<<blocks_for(N, 256), 256, 0, s>>>(d_pr, nullptr, d_co, N, P);
  CK(nullptr, cudaGetLastError());
  if (!on_device) { CK(nullptr, cudaMemcpyAsync(cons, d_co, sizeof(double) * nc * N, cudaMemcpyDeviceToHost, s)); CK(nullptr, cudaStreamSynchronize(s)); }
  return RMHD_OK;
}

int rmhd_con2prim_batch(const rmhd_params* p, long long ncells, const double* cons, const double* prim_guess, double* prims,
                        int* iters, int* fail, int on_device) {
  DevPar P;
  int rc = batch_prologue(p, ncells, P);
  if (rc) return rc;
  if (!cons || !prims) { g_create_error = "null buffer"; return RMHD_ERR_BAD_PARAM; }
  if (ncells == 0) return RMHD_OK;
  DeviceGuard dg(p->device);
  cudaStream_t s = (cudaStream_t)p->stream;
  const size_t N = (size_t)ncells;
  const int nc = p->model == 0 ? 14 : 18, np = p->model == 0 ? 11 : 16, nh = p->model == 0 ? 5 : 10;
  const double *d_co = cons, *d_pg = prim_guess; double* d_pr = prims; int *d_it = iters, *d_fl = fail;
  if (on_device) {
    if (p->model == 0) k_con2prim<0><<<blocks_for(N, 256), 256, 0, s>>>(d_co, d_pg, N, d_pr, N, d_pr + (size_t)nh * N, d_it, d_fl, N, P, nullptr);
    else k_con2prim<1><<<blocks_for(N, 256), 256, 0, s>>>(d_co, d_pg, N, d_pr, N, d_pr + (size_t)nh * N, d_it, d_fl, N, P, nullptr);
    CK(nullptr, cudaGetLastError());
    return RMHD_OK;
  }
  Staging st(s, p->device);
  {
    const size_t D = sizeof(double), I = sizeof(int);
    CK(nullptr, st.reserve(staging_align(D * nc * N) + (prim_guess ? staging_align(D * np * N) : 0) + staging_align(D * np * N) +
                           (iters ? staging_align(I * N) : 0) + (fail ? staging_align(I * N) : 0)));
    CK(nullptr, st.in(cons, nc * N, &d_co)); CK(nullptr, st.in(prim_guess, np * N, &d_pg)); CK(nullptr, st.out(prims, np * N, &d_pr));
    CK(nullptr, st.out(iters, N, &d_it)); CK(nullptr, st.out(fail, N, &d_fl));
  }
  if (p->model == 0) k_con2prim<0><<<blocks_for(N, 256), 256, 0, s>>>(d_co, d_pg, N, d_pr, N, d_pr + (size_t)nh * N, d_it, d_fl, N, P, nullptr);
  else k_con2prim<1><<<blocks_for(N, 256), 256, 0, s>>>(d_co, d_pg, N, d_pr, N, d_pr + (size_t)nh * N, d_it, d_fl, N, P, nullptr);
  CK(nullptr, cudaGetLastError());
  if (!on_device) {
    CK(nullptr, cudaMemcpyAsync(prims, d_pr, sizeof(double) * np * N, cudaMemcpyDeviceToHost, s));
    if (iters) CK(nullptr, cudaMemcpyAsync(iters, d_it, sizeof(int) * N, cudaMemcpyDeviceToHost, s));
    if (fail) CK(nullptr, cudaMemcpyAsync(fail, d_fl, sizeof(int) * N, cudaMemcpyDeviceToHost, s));
    CK(nullptr, cudaStreamSynchronize(s));
  }
  return RMHD_OK;
}

int rmhd_release_staging(int device) {
  std::lock_guard<std::mutex> lk(g_staging_mu);
  int rc = RMHD_OK;
  for (int d = 0; d < STAGING_MAX_DEVICES; ++d) {
    if ((device >= 0 && d != device) || !g_staging[d].base) continue;
    DeviceGuard dg(d);
    if (cudaFree(g_staging[d].base) != cudaSuccess) { cudaGetLastError(); rc = RMHD_ERR_CUDA; }
    g_staging[d].base = nullptr; g_staging[d].cap = 0;
  }
  return rc;
}

// ---- probes ----------------------------------------------------------------------------------
int rmhd_probe_fp64(int device, void* stream, double* tflops) {
  if (!tflops) return RMHD_ERR_BAD_PARAM;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { cudaGetLastError(); g_create_error = "no CUDA device"; return RMHD_ERR_CUDA; }
  DeviceGuard dg(device);
  cudaStream_t s = (cudaStream_t)stream;
  cudaDeviceProp prop; CK(nullptr, cudaGetDeviceProperties(&prop, device));
  const int blocks = prop.multiProcessorCount * 8, threads = 256, iters = 1 << 15;
  double* d = nullptr; CK(nullptr, cudaMalloc(&d, sizeof(double) * blocks * threads));
  cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
  double best = 0.0;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(a, s);
    k_probe_fp64<<<blocks, threads, 0, s>>>(d, iters, 1.0 + rep);
    cudaEventRecord(b, s);
    cudaError_t e = cudaEventSynchronize(b);
    if (e != cudaSuccess) { cudaFree(d); return fail_cuda(nullptr, e, "fp64 probe"); }
    float ms; cudaEventElapsedTime(&ms, a, b);
    const double fl = 2.0 * 8.0 * (double)iters * blocks * threads;
    if (rep > 0) best = fmax(best, fl / (ms * 1e-3) * 1e-12);
  }
  cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(d);
  *tflops = best;
  return RMHD_OK;
}

int rmhd_probe_hbm(int device, void* stream, long long bytes, double* gbs) {
  if (!gbs || bytes < 1024) return RMHD_ERR_BAD_PARAM;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { cudaGetLastError(); g_create_error = "no CUDA device"; return RMHD_ERR_CUDA; }
  DeviceGuard dg(device);
  cudaStream_t s = (cudaStream_t)stream;
  cudaDeviceProp prop; CK(nullptr, cudaGetDeviceProperties(&prop, device));
  const size_t n2 = (size_t)bytes / sizeof(double2);
  double2 *src = nullptr, *dst = nullptr;
  CK(nullptr, cudaMalloc(&src, n2 * sizeof(double2)));
  cudaError_t e = cudaMalloc(&dst, n2 * sizeof(double2));
  if (e != cudaSuccess) { cudaFree(src); return fail_cuda(nullptr, e, "hbm probe alloc"); }
  cudaMemsetAsync(src, 1, n2 * sizeof(double2), s);
  cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
  double best = 0.0;
  for (int rep = 0; rep < 6; ++rep) {
    cudaEventRecord(a, s);
    k_probe_copy<<<prop.multiProcessorCount * 16, 256, 0, s>>>(src, dst, n2);
    cudaEventRecord(b, s);
    e = cudaEventSynchronize(b);
    if (e != cudaSuccess) break;
    float ms; cudaEventElapsedTime(&ms, a, b);
    if (rep > 0) best = fmax(best, 2.0 * n2 * sizeof(double2) / (ms * 1e-3) * 1e-9);
  }
  cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(src); cudaFree(dst);
  if (e != cudaSuccess) return fail_cuda(nullptr, e, "hbm probe");
  *gbs = best;
  return RMHD_OK;
}

}  // extern "C"

// ---- L(q) of a caller-supplied conserved state with no allocation (rmhd_flux_divergence_static, rmhd.h) -------------
// The flux kernels read the hydro primitives next to the conserved rows, and the recovery kernel that produces them counts
// its failures in a statistics block: two pieces of device memory that are neither input nor output of "cons in, L out".
// Everywhere else in this file they come from cudaMalloc (rmhd_create).  Here they live in one fixed array that is part of
// the library image, for the programs that must not let a library allocate: a host application that has given the card's
// memory to a pool of its own (an allocation made behind the pool's back can fail while the pool still has room, and the
// pool's accounting never sees it), or a time loop that cannot afford the device-wide synchronisation cudaFree performs and
// cudaMalloc may perform (it serialises every other stream on the card).
namespace {

constexpr size_t STATIC_MAX_CELLS = RMHD_STATIC_MAX_CELLS;
constexpr size_t STATIC_STATS_BYTES = 4096;   // the Stats block, padded so that the primitive rows behind it start on a 256-byte boundary
constexpr size_t STATIC_BYTES = STATIC_STATS_BYTES + sizeof(double) * T_NH * STATIC_MAX_CELLS;   // 20 MiB + 4 KiB: 10 rows (two-fluid) of 2^18 cells
static_assert(sizeof(Stats) <= STATIC_STATS_BYTES, "statistics block outgrew its slot");

// Resident on every GPU that loads librmhd.so, from module load to process exit.  Device code may name it; in host code the
// name is only a handle for cudaGetSymbolAddress, never an address a kernel can use.
static __device__ __align__(256) unsigned char g_static_scratch[STATIC_BYTES];

constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mu;
unsigned char* g_static_addr[STATIC_MAX_DEVICES];   // the array's address on each device, looked up on that device's first call

// p->device must be the current device
int static_scratch_address(int device, unsigned char** out) {
  if (device < 0 || device >= STATIC_MAX_DEVICES) { g_create_error = "rmhd_flux_divergence_static: device ordinal beyond 63"; return RMHD_ERR_BAD_PARAM; }
  std::lock_guard<std::mutex> lk(g_static_mu);
  if (!g_static_addr[device]) {
    void* a = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&a, g_static_scratch);
    if (e != cudaSuccess || !a) return fail_cuda(nullptr, e, "cudaGetSymbolAddress(g_static_scratch)");
    g_static_addr[device] = (unsigned char*)a;
  }
  *out = g_static_addr[device];
  return RMHD_OK;
}

// the counters are accumulated with atomics and the array keeps whatever the previous call left: every call starts here
__global__ void k_static_reset(Stats* st) {
  for (int b = threadIdx.x; b < NBINS; b += blockDim.x) { st->hist_stage[b] = 0ULL; st->hist_c2p[b] = 0ULL; }
  if (threadIdx.x == 0) { st->n_failed = 0ULL; st->first_failed = LLONG_MAX; st->n_bad_input = 0ULL; }
}

template <int MODEL>
int flux_divergence_static(rmhd_ctx* c, const double* cons, double* w, Stats* st, double* Lout) {
  k_static_reset<<<1, NBINS, 0, c->stream>>>(st);
  CK(c, cudaGetLastError());
  k_con2prim<MODEL><<<blocks_for(c->N, 256), 256, 0, c->stream>>>(cons, nullptr, c->N, w, c->N, nullptr, nullptr, nullptr, c->N, c->P, st);
  CK(c, cudaGetLastError());
  return launch_flux<MODEL>(c, cons, nullptr, false, w, Lout);
}

}  // namespace

extern "C" int rmhd_flux_divergence_static(const rmhd_params* p, const double* cons, double* Lout, long long* n_failed) {
  if (n_failed) *n_failed = 0;
  if (!p || !cons || !Lout) { g_create_error = "rmhd_flux_divergence_static: null argument"; return RMHD_ERR_BAD_PARAM; }
  if (p->nx < 1 || p->ny < 1 || p->nz < 1) { g_create_error = "rmhd_flux_divergence_static: bad grid size"; return RMHD_ERR_BAD_PARAM; }
  const unsigned long long cells = (unsigned long long)p->nx * (unsigned long long)p->ny * (unsigned long long)p->nz;
  if (cells > STATIC_MAX_CELLS) {
    char buf[400];
    snprintf(buf, sizeof buf, "rmhd_flux_divergence_static: %d x %d x %d = %llu cells exceed RMHD_STATIC_MAX_CELLS = %llu, the capacity of the "
             "library's fixed scratch array; larger grids go through rmhd_create + rmhd_set_cons + rmhd_flux_divergence",
             p->nx, p->ny, p->nz, cells, (unsigned long long)STATIC_MAX_CELLS);
    g_create_error = buf;
    return RMHD_ERR_BAD_PARAM;
  }
  for (int d = 0; d < 3; ++d) if (p->bc[d] != RMHD_BC_OUTFLOW && p->bc[d] != RMHD_BC_PERIODIC) { g_create_error = "rmhd_flux_divergence_static: bad boundary condition"; return RMHD_ERR_BAD_PARAM; }
  rmhd_ctx c{};   // lives on this stack frame only: the launch helpers read the grid, the parameters and the stream from it
  int rc = batch_prologue(p, (long long)cells, c.P);   // parameter checks; RMHD_ERR_CUDA without a device (no CPU fallback)
  if (rc) return rc;
  c.p = *p; c.model = p->model;
  c.nc = p->model == 0 ? R_NC : T_NC; c.nh = p->model == 0 ? R_NH : T_NH; c.ns = p->model == 0 ? R_NS : T_NS; c.np = p->model == 0 ? 11 : 16;
  c.n[0] = p->nx; c.n[1] = p->ny; c.n[2] = p->nz; c.N = (size_t)cells;
  const double lo[3] = {p->xmin, p->ymin, p->zmin}, hi[3] = {p->xmax, p->ymax, p->zmax};
  for (int d = 0; d < 3; ++d) {
    c.dx[d] = (hi[d] - lo[d]) / c.n[d];
    if (c.n[d] > 1 && !(c.dx[d] > 0.0)) { g_create_error = "rmhd_flux_divergence_static: empty domain"; return RMHD_ERR_BAD_PARAM; }
  }
  c.device = p->device; c.stream = (cudaStream_t)p->stream;
  { const char* e = getenv("RMHD_FLUX"); c.fused_flux = !(e && strcmp(e, "split") == 0); }   // the same switch rmhd_create reads (rmhd.h)
  c.hm_ty = p->ny >= 8 ? 8 : 4;
  c.sm_count = 148;
  DeviceGuard dg(c.device);
  { int n = 0; if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, c.device) == cudaSuccess && n > 0) c.sm_count = n; }
  unsigned char* scratch = nullptr;
  if ((rc = static_scratch_address(c.device, &scratch))) return rc;
  Stats* st = (Stats*)scratch;
  double* w = (double*)(scratch + STATIC_STATS_BYTES);
  rc = c.model == 0 ? flux_divergence_static<0>(&c, cons, w, st, Lout) : flux_divergence_static<1>(&c, cons, w, st, Lout);
  if (rc) { g_create_error = c.err; return rc; }
  Stats h;   // the call returns when L is complete, like rmhd_flux_divergence: one 1 KB read-back and a stream synchronisation
  cudaError_t e = cudaMemcpyAsync(&h, st, sizeof(Stats), cudaMemcpyDeviceToHost, c.stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c.stream);
  if (e != cudaSuccess) return fail_cuda(nullptr, e, "rmhd_flux_divergence_static");
  if (n_failed) *n_failed = (long long)h.n_failed;
  if (h.n_failed) { g_create_error = "rmhd_flux_divergence_static: primitive recovery failed in some cells (count in *n_failed); L is not valid near them"; return RMHD_ERR_NONCONVERGED; }
  return RMHD_OK;
}

// ---- measurement build only (-DRMHD_HM_CYCLES, flux_hm.cuh): read / clear the cycle account of k_flux_hm ---------------
#ifdef RMHD_HM_CYCLES
extern "C" int rmhd_debug_hm_cycles(int device, unsigned long long* out16, int reset) {
  DeviceGuard dg(device);
  if (cudaDeviceSynchronize() != cudaSuccess) return RMHD_ERR_CUDA;
  if (out16 && cudaMemcpyFromSymbol(out16, g_hm_cycles, sizeof(unsigned long long) * 16) != cudaSuccess) return RMHD_ERR_CUDA;
  if (reset) {
    unsigned long long z[16] = {};
    if (cudaMemcpyToSymbol(g_hm_cycles, z, sizeof z) != cudaSuccess) return RMHD_ERR_CUDA;
  }
  return RMHD_OK;
}
#endif

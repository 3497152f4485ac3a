// kernels.cuh -- sm_100a kernels of the IMEX SSP2(222) step.  State is SoA FP64, one plane per
// variable, x fastest, INTERIOR CELLS ONLY: ghost zones are virtual (the stencil loads apply
// the outflow / periodic index map), so no ghost-fill pass and no ghost storage exist.
#pragma once
#include "stage.cuh"

namespace rmhd {

constexpr int NBINS = 64;

struct Stats {
  unsigned long long hist_stage[NBINS];
  unsigned long long hist_c2p[NBINS];
  unsigned long long n_failed;
  long long first_failed;       // smallest failing cell index, LLONG_MAX if none
  unsigned long long n_bad_input;
};

// coefficients of one implicit stage (times dt), from the Butcher tables (Table 2, Table 3)
struct StageCoef {
  double a;                // a_ii dt
  double cL[2], cP[2];     // q_ex = qn + cL0 L1 + cL1 L2 + cP0 Psi1 + cP1 Psi2            (a~_ij dt, a_ij dt)
  double hL[2], hP[3];     // A    = qn + hL0 L1 + hL1 L2 + hP0 Psi1 + hP1 Psi2 + hP2 Psi  (w~_j dt, w_j dt)
  int a_src_only;          // MKA: store A only for the rows with a source (the flux epilogue rebuilds the others, FluxComb.theta)
  int pre;                 // NL = 1: the rows without a source already hold q_ex = qn + cL0 L1 in qs (written by the F1 epilogue,
                           // FluxComb.pre); they are read from there and neither qn, L1 of those rows is read nor qs rewritten
};

template <int MODEL> struct ConsRows { const double* r[Dim<MODEL>::NC]; };
template <int MODEL> struct HydRows { const double* r[Dim<MODEL>::NH]; };

__device__ __forceinline__ int bc_map(int c, int n, int bc) {
  if (bc == 1) { c %= n; return c < 0 ? c + n : c; }
  return c < 0 ? 0 : (c >= n ? n - 1 : c);
}

// L2 prefetch of the line holding *p (no register, no scoreboard: hides DRAM latency for loads that
// ptxas sinks next to their first use when registers are short)
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

__device__ __forceinline__ void record_fail(Stats* st, long long cell) {
  atomicAdd(&st->n_failed, 1ULL);
  atomicMin(&st->first_failed, cell);
}

// block-level iteration histogram: shared counters, then one global atomic per non-empty bin
struct BlockHist {
  int* sh;
  __device__ __forceinline__ void init(int* s) { sh = s; for (int b = threadIdx.x; b < NBINS; b += blockDim.x) sh[b] = 0; __syncthreads(); }
  __device__ __forceinline__ void add(int it) { atomicAdd(&sh[it < NBINS - 1 ? it : NBINS - 1], 1); }
  __device__ __forceinline__ void flush(unsigned long long* g) {
    __syncthreads();
    for (int b = threadIdx.x; b < NBINS; b += blockDim.x) if (sh[b]) atomicAdd(&g[b], (unsigned long long)sh[b]);
  }
};

// =======================================================================================
// initial data: primitives -> conserved (+ Gauss's law for rho_charge, G10)
// prims_in: boundary layout (NP rows: hydro prims then B, E)
// =======================================================================================
template <int MODEL>
__global__ void __launch_bounds__(256) k_set_initial(const double* __restrict__ prims_in, const double* __restrict__ rho_charge,
                                                     double* __restrict__ q, double* __restrict__ w, size_t N, int nx, int ny, int nz,
                                                     int bcx, int bcy, int bcz, double i2dx, double i2dy, double i2dz,
                                                     DevPar P, Stats* st) {
  constexpr int NC = Dim<MODEL>::NC, NH = Dim<MODEL>::NH;
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= N) return;
  double wl[NH], B[3], E[3], ql[NC];
#pragma unroll
  for (int v = 0; v < NH; ++v) wl[v] = prims_in[(size_t)v * N + c];
#pragma unroll
  for (int d = 0; d < 3; ++d) { B[d] = prims_in[(size_t)(NH + d) * N + c]; E[d] = prims_in[(size_t)(NH + 3 + d) * N + c]; }
  bool bad = false;
#pragma unroll
  for (int s = 0; s < NH / 5; ++s) {
    const double v2 = wl[5 * s + 1] * wl[5 * s + 1] + wl[5 * s + 2] * wl[5 * s + 2] + wl[5 * s + 3] * wl[5 * s + 3];
    bad |= !(wl[5 * s] > 0.0) || !(wl[5 * s + 4] > 0.0) || !(v2 < 1.0);
  }
  if (bad) atomicAdd(&st->n_bad_input, 1ULL);
  if (MODEL == 0) {
    double rc = 0.0;
    if (rho_charge) rc = rho_charge[c];
    else {
      const int i = (int)(c % nx), j = (int)((c / nx) % ny), k = (int)(c / ((size_t)nx * ny));
      const double* Ex = prims_in + (size_t)(NH + 3) * N;
      const double* Ey = prims_in + (size_t)(NH + 4) * N;
      const double* Ez = prims_in + (size_t)(NH + 5) * N;
      if (nx > 1) rc += (Ex[((size_t)k * ny + j) * nx + bc_map(i + 1, nx, bcx)] - Ex[((size_t)k * ny + j) * nx + bc_map(i - 1, nx, bcx)]) * i2dx;
      if (ny > 1) rc += (Ey[((size_t)k * ny + bc_map(j + 1, ny, bcy)) * nx + i] - Ey[((size_t)k * ny + bc_map(j - 1, ny, bcy)) * nx + i]) * i2dy;
      if (nz > 1) rc += (Ez[((size_t)bc_map(k + 1, nz, bcz) * ny + j) * nx + i] - Ez[((size_t)bc_map(k - 1, nz, bcz) * ny + j) * nx + i]) * i2dz;
    }
    r_prim2cons(wl, B, E, rc, P, ql);
  } else {
    t_prim2cons(wl, B, E, P, ql);
  }
#pragma unroll
  for (int v = 0; v < NC; ++v) q[(size_t)v * N + c] = ql[v];
#pragma unroll
  for (int v = 0; v < NH; ++v) w[(size_t)v * N + c] = wl[v];
}

// batched prim -> cons (boundary layouts on both sides)
template <int MODEL>
__global__ void __launch_bounds__(256) k_prim2cons_batch(const double* __restrict__ prims, const double* __restrict__ rho_charge,
                                                         double* __restrict__ cons, size_t N, DevPar P) {
  constexpr int NC = Dim<MODEL>::NC, NH = Dim<MODEL>::NH;
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= N) return;
  double wl[NH], B[3], E[3], ql[NC];
#pragma unroll
  for (int v = 0; v < NH; ++v) wl[v] = prims[(size_t)v * N + c];
#pragma unroll
  for (int d = 0; d < 3; ++d) { B[d] = prims[(size_t)(NH + d) * N + c]; E[d] = prims[(size_t)(NH + 3 + d) * N + c]; }
  if (MODEL == 0) r_prim2cons(wl, B, E, rho_charge ? rho_charge[c] : 0.0, P, ql); else t_prim2cons(wl, B, E, P, ql);
#pragma unroll
  for (int v = 0; v < NC; ++v) cons[(size_t)v * N + c] = ql[v];
}

// =======================================================================================
// con2prim of a full conserved state (step P; rmhd_set_cons; rmhd_con2prim_batch)
// guess: NH hydro rows (stride N) or null.  prims_out NH rows; if full_out != null also B, E rows
// =======================================================================================
template <int MODEL>
__device__ __forceinline__ int cell_con2prim(const double* ql, const double* wg, bool have_guess, const DevPar& P, double* wl, int& iters) {
  constexpr int NH = Dim<MODEL>::NH;
  if (MODEL == 0) {
    Hyd h;
    const double Zg = have_guess ? Z_of_prims(wg[0], wg[1], wg[2], wg[3], wg[4], P) : -1.0;
    const int rc = r_con2prim(ql, Zg, P, h, iters);
    wl[0] = h.rho; wl[1] = h.vx; wl[2] = h.vy; wl[3] = h.vz; wl[4] = h.p;
    return rc;
  } else {
    Hyd h[2];
    double Zg[2] = {-1.0, -1.0};
    if (have_guess) { Zg[0] = Z_of_prims(wg[0], wg[1], wg[2], wg[3], wg[4], P); Zg[1] = Z_of_prims(wg[5], wg[6], wg[7], wg[8], wg[9], P); }
    const int rc = t_con2prim(ql, Zg, P, h, iters);
#pragma unroll
    for (int s = 0; s < 2; ++s) { wl[5 * s] = h[s].rho; wl[5 * s + 1] = h[s].vx; wl[5 * s + 2] = h[s].vy; wl[5 * s + 3] = h[s].vz; wl[5 * s + 4] = h[s].p; }
    (void)NH;
    return rc;
  }
}

template <int MODEL>
__global__ void __launch_bounds__(256) k_con2prim(const double* __restrict__ cons, const double* __restrict__ guess, size_t gstride,
                                                  double* __restrict__ w, size_t wstride, double* __restrict__ BE_out /*6 rows or null*/,
                                                  int* __restrict__ iters_out, int* __restrict__ fail_out, size_t N, DevPar P, Stats* st) {
  constexpr int NC = Dim<MODEL>::NC, NH = Dim<MODEL>::NH, IB = Dim<MODEL>::IB;
  __shared__ int shist[NBINS];
  BlockHist bh; bh.init(shist);
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c < N) {
    double ql[NC], wg[NH], wl[NH];
#pragma unroll
    for (int v = 0; v < NC; ++v) ql[v] = cons[(size_t)v * N + c];
    if (guess) {
#pragma unroll
      for (int v = 0; v < NH; ++v) wg[v] = guess[(size_t)v * gstride + c];
    }
    int it;
    const int rc = cell_con2prim<MODEL>(ql, wg, guess != nullptr, P, wl, it);
#pragma unroll
    for (int v = 0; v < NH; ++v) w[(size_t)v * wstride + c] = wl[v];
    if (BE_out) {
#pragma unroll
      for (int d = 0; d < 6; ++d) BE_out[(size_t)d * wstride + c] = ql[IB + d];
    }
    if (iters_out) iters_out[c] = it;
    if (fail_out) fail_out[c] = rc;
    if (st) { bh.add(it); if (rc) record_fail(st, (long long)c); }
  }
  if (st) bh.flush(st->hist_c2p);
}

// =======================================================================================
// a1: implicit stage, resistive.  One thread per cell, everything in registers; the Newton
// loop is warp-voted so a warp leaves as soon as all its 32 cells have converged.
// Stage i of eq (10) with NL = i - 1 earlier stages (SSP2(222): NL = 0, 1; SSP3(332): NL = 0, 1, 2):
//   NL = 0: q_ex = qn.                        writes E*, psi*, phi* rows of qs, prims, Psi
//   NL > 0: q_ex = qn + cL0 L1 + cL1 L2 + cP0 Psi1 + cP1 Psi2 (fused a5).  writes all rows of qs, prims, Psi
// Psi rows stored: -J (3), rhoc - kappa psi*, -kappa phi*.
// MKA (last stage): instead of Psi the kernel writes the part of eq (11) that is known once the last stage is
// solved,  A_v = qn_v + hL0 L1_v + hL1 L2_v + hP0 Psi1_v + hP1 Psi2_v + hP2 Psi_v(this stage)  (all NC rows), so
// that the last flux launch finishes the step with q^{n+1}_v = A_v + w~_last dt L_last,v (flux_fused.cuh, FluxComb).
// =======================================================================================
template <int NL, bool MKA = false>
__global__ void __launch_bounds__(128, 5) k_stage_resistive(const double* __restrict__ qn, const double* __restrict__ L1,
                                                         const double* __restrict__ L2, const double* __restrict__ Ps1,
                                                         const double* __restrict__ Ps2, double* __restrict__ w,
                                                         double* __restrict__ qs, double* __restrict__ Ps, double* __restrict__ A,
                                                         size_t N, StageCoef k, DevPar P, Stats* st) {
  __shared__ int shist[NBINS];
  BlockHist bh; bh.init(shist);
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = c < N;
  RStage s;
  s.status = 1; s.iters = 0;
  double qpsi = 0.0, qphi = 0.0;
  if (valid) {
    double qe[R_NC];
#pragma unroll
    for (int v = 0; v < R_NC; ++v) qe[v] = (NL == 1 && k.pre && (v < 8 || v == 11)) ? qs[(size_t)v * N + c] : qn[(size_t)v * N + c];
    if (NL >= 1) {
#pragma unroll
      for (int v = 0; v < R_NC; ++v) {
        if (NL == 1 && k.pre && (v < 8 || v == 11)) continue;
        double av = qe[v];
        const double l1 = L1[(size_t)v * N + c];
        if (MKA) av = fma(k.hL[0], l1, av);
        qe[v] = fma(k.cL[0], l1, qe[v]);
        if (NL >= 2) {
          const double l2 = L2[(size_t)v * N + c];
          if (MKA) av = fma(k.hL[1], l2, av);
          qe[v] = fma(k.cL[1], l2, qe[v]);
        }
        if (MKA && !k.a_src_only && (v < 8 || v == 11)) A[(size_t)v * N + c] = av;
      }
#pragma unroll
      for (int j = 0; j < R_NS; ++j) {
        const int v = j < 3 ? 8 + j : 9 + j;
        qe[v] = fma(k.cP[0], Ps1[(size_t)j * N + c], qe[v]);
        if (NL >= 2 && k.cP[1] != 0.0) qe[v] = fma(k.cP[1], Ps2[(size_t)j * N + c], qe[v]);
      }
      if (!(NL == 1 && k.pre)) {
#pragma unroll
        for (int v = 0; v < R_NC; ++v) if (v < 8 || v == 11) qs[(size_t)v * N + c] = qe[v];
      }
    }
    qpsi = qe[12]; qphi = qe[13];
    r_stage_init(s, qe, w[c], w[N + c], w[2 * N + c], w[3 * N + c], w[4 * N + c], k.a, P.sigma, P);
  }
  while (true) {
    const bool active = s.status == 0 && s.iters < P.maxit_stage;
    if (!__any_sync(0xffffffffu, active)) break;
    if (active) r_stage_iter(s, P);
  }
  if (valid) {
    Hyd h; double J[3], psi, phi;
    double Ap[R_NS];
    if (MKA) {       // qn, L, Psi of the source rows again (L2 hits) rather than 10 registers held across the Newton loop
#pragma unroll
      for (int j = 0; j < R_NS; ++j) {
        const size_t v = j < 3 ? 8 + j : 9 + j;
        double av = fma(k.hL[0], L1[v * N + c], fma(k.hP[0], Ps1[(size_t)j * N + c], qn[v * N + c]));
        if (NL >= 2) av = fma(k.hL[1], L2[v * N + c], fma(k.hP[1], Ps2[(size_t)j * N + c], av));
        Ap[j] = av;
      }
    }
    r_stage_finish(s, P, h, J, psi, phi, qpsi, qphi);
    qs[8 * N + c] = s.Ex; qs[9 * N + c] = s.Ey; qs[10 * N + c] = s.Ez; qs[12 * N + c] = psi; qs[13 * N + c] = phi;
    w[c] = h.rho; w[N + c] = h.vx; w[2 * N + c] = h.vy; w[3 * N + c] = h.vz; w[4 * N + c] = h.p;
    const double ps[R_NS] = {-J[0], -J[1], -J[2], s.rhoc - P.kappa * psi, -P.kappa * phi};
#pragma unroll
    for (int j = 0; j < R_NS; ++j) {
      if (MKA) A[(size_t)(j < 3 ? 8 + j : 9 + j) * N + c] = fma(k.hP[2], ps[j], Ap[j]);
      else Ps[(size_t)j * N + c] = ps[j];
    }
    bh.add(s.iters);
    if (s.status != 1 || !(h.p > 0.0) || !(h.rho > 0.0)) record_fail(st, (long long)c);
  }
  bh.flush(st->hist_stage);
}

// batched implicit stage on independent cells (config 2): boundary layouts, per-cell sigma
__global__ void __launch_bounds__(128) k_stage_batch_resistive(const double* __restrict__ q_ex, const double* __restrict__ prim_guess,
                                                               const double* __restrict__ sigma_cell, double a, double* __restrict__ q_out,
                                                               double* __restrict__ prims_out, int* __restrict__ iters,
                                                               int* __restrict__ fail, size_t N, DevPar P) {
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = c < N;
  RStage s;
  s.status = 1; s.iters = 0;
  double qpsi = 0.0, qphi = 0.0;
  if (valid) {
    double qe[R_NC];
#pragma unroll
    for (int v = 0; v < R_NC; ++v) qe[v] = q_ex[(size_t)v * N + c];
#pragma unroll
    for (int v = 0; v < R_NC; ++v) if (v < 8 || v == 11) q_out[(size_t)v * N + c] = qe[v];
    qpsi = qe[12]; qphi = qe[13];
    r_stage_init(s, qe, prim_guess[c], prim_guess[N + c], prim_guess[2 * N + c], prim_guess[3 * N + c], prim_guess[4 * N + c], a,
                 sigma_cell ? sigma_cell[c] : P.sigma, P);
  }
  while (true) {
    const bool active = s.status == 0 && s.iters < P.maxit_stage;
    if (!__any_sync(0xffffffffu, active)) break;
    if (active) r_stage_iter(s, P);
  }
  if (valid) {
    Hyd h; double J[3], psi, phi;
    r_stage_finish(s, P, h, J, psi, phi, qpsi, qphi);
    q_out[8 * N + c] = s.Ex; q_out[9 * N + c] = s.Ey; q_out[10 * N + c] = s.Ez; q_out[12 * N + c] = psi; q_out[13 * N + c] = phi;
    prims_out[c] = h.rho; prims_out[N + c] = h.vx; prims_out[2 * N + c] = h.vy; prims_out[3 * N + c] = h.vz; prims_out[4 * N + c] = h.p;
    prims_out[5 * N + c] = s.Bx; prims_out[6 * N + c] = s.By; prims_out[7 * N + c] = s.Bz;
    prims_out[8 * N + c] = s.Ex; prims_out[9 * N + c] = s.Ey; prims_out[10 * N + c] = s.Ez;
    if (iters) iters[c] = s.iters;
    if (fail) fail[c] = (s.status == 1 && h.p > 0.0 && h.rho > 0.0) ? 0 : (s.status == 1 ? 3 : (s.status == 0 ? 2 : 10 - s.status));
  }
}

// =======================================================================================
// a1: implicit stage, two-fluid (same launch shape and warp-voted loop as the resistive one).
// Source rows (Psi storage order): Sbar(3), taubar, E(3), psi, phi  = cons rows 6..9, 13..17.
// =======================================================================================
template <int NL, bool MKA = false>
__global__ void __launch_bounds__(128) k_stage_two_fluid(const double* __restrict__ qn, const double* __restrict__ L1,
                                                         const double* __restrict__ L2, const double* __restrict__ Ps1,
                                                         const double* __restrict__ Ps2, double* __restrict__ w,
                                                         double* __restrict__ qs, double* __restrict__ Ps, double* __restrict__ A,
                                                         size_t N, StageCoef k, DevPar P, Stats* st) {
  __shared__ int shist[NBINS];
  BlockHist bh; bh.init(shist);
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = c < N;
  TStage s;
  s.status = 1; s.iters = 0;
  double qpsi = 0.0, qphi = 0.0;
  if (valid) {
    double qe[T_NC], wg[T_NH];
#pragma unroll
    for (int v = 0; v < T_NC; ++v) qe[v] = (NL == 1 && k.pre && (v < 6 || (v >= 10 && v < 13))) ? qs[(size_t)v * N + c] : qn[(size_t)v * N + c];
    if (NL >= 1) {
#pragma unroll
      for (int v = 0; v < T_NC; ++v) {
        if (NL == 1 && k.pre && (v < 6 || (v >= 10 && v < 13))) continue;
        double av = qe[v];
        const double l1 = L1[(size_t)v * N + c];
        if (MKA) av = fma(k.hL[0], l1, av);
        qe[v] = fma(k.cL[0], l1, qe[v]);
        if (NL >= 2) {
          const double l2 = L2[(size_t)v * N + c];
          if (MKA) av = fma(k.hL[1], l2, av);
          qe[v] = fma(k.cL[1], l2, qe[v]);
        }
        if (MKA && !k.a_src_only && (v < 6 || (v >= 10 && v < 13))) A[(size_t)v * N + c] = av;
      }
#pragma unroll
      for (int j = 0; j < T_NS; ++j) {
        const int v = j < 4 ? 6 + j : 9 + j;
        qe[v] = fma(k.cP[0], Ps1[(size_t)j * N + c], qe[v]);
        if (NL >= 2 && k.cP[1] != 0.0) qe[v] = fma(k.cP[1], Ps2[(size_t)j * N + c], qe[v]);
      }
      if (!(NL == 1 && k.pre)) {
#pragma unroll
        for (int v = 0; v < T_NC; ++v) if (v < 6 || (v >= 10 && v < 13)) qs[(size_t)v * N + c] = qe[v];
      }
    }
    qpsi = qe[16]; qphi = qe[17];
#pragma unroll
    for (int v = 0; v < T_NH; ++v) wg[v] = w[(size_t)v * N + c];
    t_stage_init(s, qe, wg, k.a, P);
  }
  while (true) {
    const bool active = s.status == 0 && s.iters < P.maxit_stage;
    if (!__any_sync(0xffffffffu, active)) break;
    if (active) t_stage_iter(s, P);
  }
  if (valid) {
    double wl[T_NH], src[T_NS], psi, phi;
    t_stage_finish(s, P, wl, src, psi, phi, qpsi, qphi);
#pragma unroll
    for (int i = 0; i < 3; ++i) { qs[(size_t)(6 + i) * N + c] = s.Sb[i]; qs[(size_t)(13 + i) * N + c] = s.E[i]; }
    qs[9 * N + c] = s.tb; qs[16 * N + c] = psi; qs[17 * N + c] = phi;
#pragma unroll
    for (int v = 0; v < T_NH; ++v) w[(size_t)v * N + c] = wl[v];
#pragma unroll
    for (int j = 0; j < T_NS; ++j) {
      if (MKA) {
        const size_t v = j < 4 ? 6 + j : 9 + j;
        double av = fma(k.hL[0], L1[v * N + c], fma(k.hP[0], Ps1[(size_t)j * N + c], qn[v * N + c]));
        if (NL >= 2) av = fma(k.hL[1], L2[v * N + c], fma(k.hP[1], Ps2[(size_t)j * N + c], av));
        A[v * N + c] = fma(k.hP[2], src[j], av);
      } else Ps[(size_t)j * N + c] = src[j];
    }
    bh.add(s.iters);
    if (s.status != 1 || !(wl[0] > 0.0) || !(wl[4] > 0.0) || !(wl[5] > 0.0) || !(wl[9] > 0.0)) record_fail(st, (long long)c);
  }
  bh.flush(st->hist_stage);
}

// batched two-fluid implicit stage on independent cells: boundary layouts
__global__ void __launch_bounds__(128) k_stage_batch_two_fluid(const double* __restrict__ q_ex, const double* __restrict__ prim_guess,
                                                               double a, double* __restrict__ q_out, double* __restrict__ prims_out,
                                                               int* __restrict__ iters, int* __restrict__ fail, size_t N, DevPar P) {
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = c < N;
  TStage s;
  s.status = 1; s.iters = 0;
  double qpsi = 0.0, qphi = 0.0;
  if (valid) {
    double qe[T_NC], wg[T_NH];
#pragma unroll
    for (int v = 0; v < T_NC; ++v) qe[v] = q_ex[(size_t)v * N + c];
#pragma unroll
    for (int v = 0; v < T_NC; ++v) if (v < 6 || (v >= 10 && v < 13)) q_out[(size_t)v * N + c] = qe[v];
    qpsi = qe[16]; qphi = qe[17];
#pragma unroll
    for (int v = 0; v < T_NH; ++v) wg[v] = prim_guess[(size_t)v * N + c];
    t_stage_init(s, qe, wg, a, P);
  }
  while (true) {
    const bool active = s.status == 0 && s.iters < P.maxit_stage;
    if (!__any_sync(0xffffffffu, active)) break;
    if (active) t_stage_iter(s, P);
  }
  if (valid) {
    double wl[T_NH], src[T_NS], psi, phi;
    t_stage_finish(s, P, wl, src, psi, phi, qpsi, qphi);
#pragma unroll
    for (int i = 0; i < 3; ++i) { q_out[(size_t)(6 + i) * N + c] = s.Sb[i]; q_out[(size_t)(13 + i) * N + c] = s.E[i]; }
    q_out[9 * N + c] = s.tb; q_out[16 * N + c] = psi; q_out[17 * N + c] = phi;
#pragma unroll
    for (int v = 0; v < T_NH; ++v) prims_out[(size_t)v * N + c] = wl[v];
    prims_out[10 * N + c] = s.Bx; prims_out[11 * N + c] = s.By; prims_out[12 * N + c] = s.Bz;
#pragma unroll
    for (int i = 0; i < 3; ++i) prims_out[(size_t)(13 + i) * N + c] = s.E[i];
    if (iters) iters[c] = s.iters;
    const bool phys = wl[0] > 0.0 && wl[4] > 0.0 && wl[5] > 0.0 && wl[9] > 0.0;
    if (fail) fail[c] = (s.status == 1 && phys) ? 0 : (s.status == 1 ? 3 : (s.status == 0 ? 2 : 10 - s.status));
  }
}

// =======================================================================================
// a4, axes 1 and 2 (sweep axis strided in memory): MARCHING kernel.  Lanes run along x, so the
// stencil never crosses lanes: each thread owns one (x, other) column and marches along the
// sweep axis over a segment, keeping the 3-cell f+ / 2-cell f- window of its column in shared
// memory (used as per-thread scratch: no barrier anywhere in the kernel) and the previous
// face flux in registers.  Per new cell c: load q, w (boundary index map), flux vector,
// f+- = (f +- q)/2, face between c-2 and c-1 by WENO3, then L of cell c-2.  The next cell's
// inputs are loaded before the current cell's arithmetic (software prefetch).
// =======================================================================================
#ifndef RMHD_MARCH_MINB
#define RMHD_MARCH_MINB 3
#endif
constexpr int MARCH_THREADS = 128;
template <int MODEL> constexpr size_t march_smem_bytes() { return sizeof(double) * 5 * Dim<MODEL>::NC * MARCH_THREADS; }

template <int MODEL, int AXIS>
__global__ void __launch_bounds__(MARCH_THREADS, MODEL == 0 ? RMHD_MARCH_MINB : 2)
k_flux_march(ConsRows<MODEL> qin, HydRows<MODEL> win, double* __restrict__ L, size_t N, int nx, int ny, int nz, int bc,
             double inv_dx, int accumulate, int seg_len, DevPar P) {
  static_assert(AXIS == 1 || AXIS == 2, "marching kernel is for the strided axes");
  constexpr int NC = Dim<MODEL>::NC, NH = Dim<MODEL>::NH, T = MARCH_THREADS;
  extern __shared__ double sm[];   // f+ ring [3][NC][T], f- ring [2][NC][T]
  const int i = blockIdx.x * T + threadIdx.x;
  if (i >= nx) return;
  const int other = blockIdx.y;
  const int ns = AXIS == 1 ? ny : nz;
  const int s_begin = blockIdx.z * seg_len;
  const int s_end = min(ns, s_begin + seg_len);
  const size_t stride = AXIS == 1 ? (size_t)nx : (size_t)nx * ny;
  const size_t base = AXIS == 1 ? (size_t)other * ny * nx + i : (size_t)other * nx + i;
  double* ring = sm + threadIdx.x;
  int a0 = 0, a1 = NC * T, a2 = 2 * NC * T;            // f+ slots of cells c-3, c-2, c-1
  int b0 = 3 * NC * T, b1 = 4 * NC * T;                // f- slots of cells c-2, c-1

  double qc[NC], wc[NH], qn_[NC], wn_[NH];
  auto load = [&](int c, double* q_, double* w_) {
    const size_t idx = base + (size_t)bc_map(c, ns, bc) * stride;
#pragma unroll
    for (int v = 0; v < NC; ++v) q_[v] = __ldg(qin.r[v] + idx);
#pragma unroll
    for (int v = 0; v < NH; ++v) w_[v] = __ldg(win.r[v] + idx);
  };
  // prologue: cells s_begin-2, s_begin-1, s_begin
  load(s_begin - 2, qn_, wn_);
#pragma unroll 1
  for (int c = s_begin - 2; c <= s_begin; ++c) {
#pragma unroll
    for (int v = 0; v < NC; ++v) qc[v] = qn_[v];
#pragma unroll
    for (int v = 0; v < NH; ++v) wc[v] = wn_[v];
    load(c + 1, qn_, wn_);
    double f[NC];
    if (MODEL == 0) r_flux<AXIS>(qc, wc, P.sigma, P, f); else t_flux<AXIS>(qc, wc, P, f);
#pragma unroll
    for (int v = 0; v < NC; ++v) {
      ring[a0 + v * T] = 0.5 * (f[v] + qc[v]);
      ring[b0 + v * T] = 0.5 * (f[v] - qc[v]);   // for c = s_begin-2 this slot is overwritten next
    }
    { const int t = a0; a0 = a1; a1 = a2; a2 = t; }
    { const int t = b0; b0 = b1; b1 = t; }
  }
  double Fp[NC], La[NC];
  // main loop: new cell c, face between c-2 and c-1, L of cell c-2
#pragma unroll 1
  for (int c = s_begin + 1; c <= s_end + 1; ++c) {
#pragma unroll
    for (int v = 0; v < NC; ++v) qc[v] = qn_[v];
#pragma unroll
    for (int v = 0; v < NH; ++v) wc[v] = wn_[v];
    const bool emit = c >= s_begin + 2;
    const size_t oidx = base + (size_t)(emit ? c - 2 : 0) * stride;
    if (c + 2 <= s_end + 1) {   // L2 prefetch of the inputs of step c + 1 (cell c + 2) and of the partial L it adds to
      const size_t pidx = base + (size_t)bc_map(c + 2, ns, bc) * stride;
#pragma unroll
      for (int v = 0; v < NC; ++v) prefetch_l2(qin.r[v] + pidx);
#pragma unroll
      for (int v = 0; v < NH; ++v) prefetch_l2(win.r[v] + pidx);
      if (accumulate && c < s_end) {
        const size_t lidx = base + (size_t)(c - 1) * stride;
#pragma unroll
        for (int v = 0; v < NC; ++v) prefetch_l2(L + (size_t)v * N + lidx);
      }
    }
    // issue every global load of this step up front: next cell's inputs and the partial L to add to
    if (c <= s_end) load(c + 1, qn_, wn_);
    if (accumulate && emit) {
#pragma unroll
      for (int v = 0; v < NC; ++v) La[v] = L[(size_t)v * N + oidx];
    } else {
#pragma unroll
      for (int v = 0; v < NC; ++v) La[v] = 0.0;
    }
    double f[NC];
    if (MODEL == 0) r_flux<AXIS>(qc, wc, P.sigma, P, f); else t_flux<AXIS>(qc, wc, P, f);
#pragma unroll
    for (int v0 = 0; v0 < NC; v0 += 4) {      // 4 variables = 8 reconstructions in flight (weno3_batch)
      constexpr int G = 4;
      double a[2 * G], b[2 * G], cc[2 * G], o[2 * G], fpc[G], fmc[G];
#pragma unroll
      for (int g = 0; g < G; ++g) {
        const int v = v0 + g < NC ? v0 + g : NC - 1;
        fpc[g] = 0.5 * (f[v] + qc[v]);
        fmc[g] = 0.5 * (f[v] - qc[v]);
        a[2 * g] = ring[a0 + v * T]; b[2 * g] = ring[a1 + v * T]; cc[2 * g] = ring[a2 + v * T];
        a[2 * g + 1] = fmc[g]; b[2 * g + 1] = ring[b1 + v * T]; cc[2 * g + 1] = ring[b0 + v * T];
      }
      weno3_batch<2 * G>(a, b, cc, o);
#pragma unroll
      for (int g = 0; g < G; ++g) {
        const int v = v0 + g;
        if (v < NC) {
          const double F = o[2 * g] + o[2 * g + 1];
          if (emit) L[(size_t)v * N + oidx] = La[v] - (F - Fp[v]) * inv_dx;
          Fp[v] = F;
          ring[a0 + v * T] = fpc[g];
          ring[b0 + v * T] = fmc[g];
        }
      }
    }
    { const int t = a0; a0 = a1; a1 = a2; a2 = t; }
    { const int t = b0; b0 = b1; b1 = t; }
  }
}

// =======================================================================================
// C + P: q^{n+1} = qn + dt/2 (L1 + L2) + dt/2 (Psi1 + Psi2)  (eq 11), then con2prim.
// SRC_ROWS: for MODEL 0 rows 8,9,10,12,13 ; MODEL 1 rows 6..9, 13..17
// =======================================================================================
template <int MODEL> __device__ __forceinline__ int src_row(int k);
template <> __device__ __forceinline__ int src_row<0>(int k) { return k < 3 ? 8 + k : 9 + k; }   // 8,9,10,12,13
template <> __device__ __forceinline__ int src_row<1>(int k) { return k < 4 ? 6 + k : 9 + k; }   // 6,7,8,9,13..17

template <int MODEL>
__global__ void __launch_bounds__(256) k_final(double* __restrict__ q, const double* __restrict__ L1, const double* __restrict__ L2,
                                               const double* __restrict__ Ps1, const double* __restrict__ Ps2, double* __restrict__ w,
                                               size_t N, double hdt, DevPar P, Stats* st) {
  constexpr int NC = Dim<MODEL>::NC, NH = Dim<MODEL>::NH, NS = Dim<MODEL>::NS;
  __shared__ int shist[NBINS];
  BlockHist bh; bh.init(shist);
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c < N) {
    double ql[NC], wg[NH], wl[NH];
#pragma unroll
    for (int v = 0; v < NC; ++v) ql[v] = q[(size_t)v * N + c] + hdt * (L1[(size_t)v * N + c] + L2[(size_t)v * N + c]);
#pragma unroll
    for (int k = 0; k < NS; ++k) ql[src_row<MODEL>(k)] += hdt * (Ps1[(size_t)k * N + c] + Ps2[(size_t)k * N + c]);
#pragma unroll
    for (int v = 0; v < NH; ++v) wg[v] = w[(size_t)v * N + c];
    int it;
    const int rc = cell_con2prim<MODEL>(ql, wg, true, P, wl, it);
#pragma unroll
    for (int v = 0; v < NC; ++v) q[(size_t)v * N + c] = ql[v];
#pragma unroll
    for (int v = 0; v < NH; ++v) w[(size_t)v * N + c] = wl[v];
    bh.add(it);
    if (rc) record_fail(st, (long long)c);
  }
  bh.flush(st->hist_c2p);
}

// last-stage combine for the per-axis flux path when A (see StageCoef) is in use: q^{n+1} = A + wl L_last, then con2prim
template <int MODEL>
__global__ void __launch_bounds__(256) k_final_A(double* __restrict__ q, const double* __restrict__ A, const double* __restrict__ Ll,
                                                 double* __restrict__ w, size_t N, double wl, DevPar P, Stats* st) {
  constexpr int NC = Dim<MODEL>::NC, NH = Dim<MODEL>::NH;
  __shared__ int shist[NBINS];
  BlockHist bh; bh.init(shist);
  const size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c < N) {
    double ql[NC], wg[NH], wo[NH];
#pragma unroll
    for (int v = 0; v < NC; ++v) ql[v] = fma(wl, Ll[(size_t)v * N + c], A[(size_t)v * N + c]);
#pragma unroll
    for (int v = 0; v < NH; ++v) wg[v] = w[(size_t)v * N + c];
    int it;
    const int rc = cell_con2prim<MODEL>(ql, wg, true, P, wo, it);
#pragma unroll
    for (int v = 0; v < NC; ++v) q[(size_t)v * N + c] = ql[v];
#pragma unroll
    for (int v = 0; v < NH; ++v) w[(size_t)v * N + c] = wo[v];
    bh.add(it);
    if (rc) record_fail(st, (long long)c);
  }
  bh.flush(st->hist_c2p);
}

// =======================================================================================
// probes for the roofline denominators
// =======================================================================================
__global__ void __launch_bounds__(256) k_probe_fp64(double* out, int iters, double seed) {
  double a0 = seed, a1 = seed + 1, a2 = seed + 2, a3 = seed + 3, a4 = seed + 4, a5 = seed + 5, a6 = seed + 6, a7 = seed + 7;
  const double m = 1.0000001, b = 1e-9 * threadIdx.x;
  for (int i = 0; i < iters; ++i) {
    a0 = fma(a0, m, b); a1 = fma(a1, m, b); a2 = fma(a2, m, b); a3 = fma(a3, m, b);
    a4 = fma(a4, m, b); a5 = fma(a5, m, b); a6 = fma(a6, m, b); a7 = fma(a7, m, b);
  }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

__global__ void __launch_bounds__(256) k_probe_copy(const double2* __restrict__ src, double2* __restrict__ dst, size_t n2) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}

}  // namespace rmhd

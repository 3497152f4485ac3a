// flux3.cuh -- a4 fused: L(q) = -sum_d dF^d/dx_d for all present axes in ONE pass over the state
// (eq 12).  Reads q, w once (+ halo re-reads that hit L2), writes L once: 33 doubles of
// algorithmic traffic per cell instead of the 127 of three single-axis passes.
//
// A CTA owns a 32 (x) x 4 (y) column bundle and MARCHES along z over a segment:
//   z  : private per thread.  The 3-cell f+ / 2-cell f- window of the column lives in a shared-memory
//        ring used as per-thread scratch (no barrier); the previous face flux stays in registers.  The ring
//        runs two planes ahead of the x/y work (the face k+1/2 needs f-(k+2)).
//   x,y: per plane, f+- of the tile and its 2-cell halo are staged in shared memory in two chunks of
//        7 (9) variables; one WENO3 pair per face item; face fluxes exchanged through shared memory.
// 160 threads: warps 0-3 own the 128 columns; warp 4 is a helper that has no column and takes the
// work that does not divide by 128: the x-halo cells (16), the 33rd x-face of each row (4) and the
// 5th row of y-faces (32).  The y-halo rows (4 x 32 cells) are shared by the four main warps.
// Ghost zones are virtual (bc_map).  HAS_Z = false: one plane, no ring (2-D grids).
#pragma once
#include "kernels.cuh"

namespace rmhd {

#ifndef RMHD_F3_REGS
#define RMHD_F3_REGS 168
#endif
constexpr int F3_TX = 32, F3_TY = 4, F3_MAIN = F3_TX * F3_TY, F3_THREADS = F3_MAIN + 32;

template <int MODEL> struct F3 {
  static constexpr int NC = Dim<MODEL>::NC;
  static constexpr int CH = (NC + 1) / 2;                                   // variables per chunk
  static constexpr int PB = 2 * CH * (F3_TY + 4) * F3_TX;                   // y layout (>= x layout 2*CH*TY*36)
  static constexpr int FB = CH * (F3_TY + 1) * F3_TX;                       // y faces (>= x faces CH*TY*33)
  static constexpr int RING = 5 * NC * F3_MAIN;
  static constexpr size_t bytes(bool has_z) { return sizeof(double) * (PB + FB + (has_z ? RING : 0)); }
};

template <int MODEL, int K>
__device__ __forceinline__ void split_flux(const double* q, const double* w, const DevPar& P, double* fp, double* fm) {
  constexpr int NC = Dim<MODEL>::NC;
  double f[NC];
  if (MODEL == 0) r_flux<K>(q, w, P.sigma, P, f); else t_flux<K>(q, w, P, f);
#pragma unroll
  for (int v = 0; v < NC; ++v) {
    const double hf = 0.5 * f[v];
    fp[v] = fma(0.5, q[v], hf);
    fm[v] = fma(-0.5, q[v], hf);
  }
}

template <int MODEL, bool HAS_Z>
__global__ void __launch_bounds__(F3_THREADS, 1) __maxnreg__(HAS_Z ? (MODEL == 0 ? RMHD_F3_REGS : 255) : RMHD_F3_REGS)
k_flux3(ConsRows<MODEL> qin, HydRows<MODEL> win, double* __restrict__ L, size_t N, int nx, int ny, int nz, int bcx, int bcy,
        int bcz, double idx, double idy, double idz, int seg_len, DevPar P) {
  constexpr int NC = Dim<MODEL>::NC, NH = Dim<MODEL>::NH, CH = F3<MODEL>::CH;
  constexpr int TX = F3_TX, TY = F3_TY, XW = TX + 4, YR = TY + 4;
  extern __shared__ double sm[];
  double* PB = sm;
  double* FB = sm + F3<MODEL>::PB;
  const int tid = threadIdx.x, lane = tid & 31, ty = tid >> 5;
  const bool is_main = tid < F3_MAIN;
  double* ring = FB + F3<MODEL>::FB + tid;          // main threads only
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
  const int i = i0 + lane, j = j0 + ty;
  const bool inside = is_main && i < nx && j < ny;
  const int im = bc_map(i, nx, bcx);                // ghost semantics also for the tail of a partial tile
  const int jm = bc_map(is_main ? j : j0, ny, bcy);
  // y-halo row of this main warp (rows -2,-1,4,5 of the tile) and x-halo cell of helper lanes 0..15
  const int hrow = ty < 2 ? ty : ty + 4;            // PB row of the halo row (PB row = tile row + 2)
  const int jh = bc_map(j0 + hrow - 2, ny, bcy);
  const int xh_row = lane >> 2, xh_c = (lane & 3) < 2 ? (lane & 3) - 2 : (lane & 3) + 30;   // tile col -2,-1,32,33
  const int ixh = bc_map(i0 + xh_c, nx, bcx), jxh = bc_map(j0 + xh_row, ny, bcy);

  const int k0 = HAS_Z ? blockIdx.z * seg_len : 0;
  const int k1 = HAS_Z ? min(nz, k0 + seg_len) : 1;
  const size_t pstride = (size_t)nx * ny;

  auto load_cell = [&](int ii, int jj, int kk, double* q_, double* w_) {
    const size_t id = (size_t)kk * pstride + (size_t)jj * nx + ii;
#pragma unroll
    for (int v = 0; v < NC; ++v) q_[v] = __ldg(qin.r[v] + id);
#pragma unroll
    for (int v = 0; v < NH; ++v) w_[v] = __ldg(win.r[v] + id);
  };

  double Fp[NC];                                     // previous z-face flux (HAS_Z)
  double qf[NC], wf[NH];                             // feed plane (two ahead of the x/y plane)
  int a0 = 0, a1 = NC * F3_MAIN, a2 = 2 * NC * F3_MAIN, b0 = 3 * NC * F3_MAIN, b1 = 4 * NC * F3_MAIN;
  if (HAS_Z && is_main) load_cell(im, jm, bc_map(k0 - 2, nz, bcz), qf, wf);

  const int cbeg = HAS_Z ? k0 - 2 : 2, cend = HAS_Z ? k1 + 1 : 2;
#pragma unroll 1
  for (int c = cbeg; c <= cend; ++c) {
    const int k = HAS_Z ? c - 2 : 0;                 // plane of the x/y work
    const bool do_xy = !HAS_Z || c >= k0 + 2;
    double Lacc[NC];
    double qk[NC], wk[NH];
    if (do_xy && is_main) load_cell(im, jm, k, qk, wk);
    // ---------------- z: feed plane c, face between c-2 and c-1, L_z of plane c-2 --------------
    if (HAS_Z && is_main) {
      double fzp[NC], fzm[NC];
      split_flux<MODEL, 2>(qf, wf, P, fzp, fzm);
      if (c >= k0 + 1) {
#pragma unroll
        for (int v0 = 0; v0 < NC; v0 += 4) {
          constexpr int G = 4;
          double a[2 * G], b[2 * G], cc[2 * G], o[2 * G];
#pragma unroll
          for (int g = 0; g < G; ++g) {
            const int v = v0 + g < NC ? v0 + g : NC - 1;
            a[2 * g] = ring[a0 + v * F3_MAIN]; b[2 * g] = ring[a1 + v * F3_MAIN]; cc[2 * g] = ring[a2 + v * F3_MAIN];
            a[2 * g + 1] = fzm[v]; b[2 * g + 1] = ring[b1 + v * F3_MAIN]; cc[2 * g + 1] = ring[b0 + v * F3_MAIN];
          }
          weno3_batch<2 * G>(a, b, cc, o);
#pragma unroll
          for (int g = 0; g < G; ++g) {
            const int v = v0 + g;
            if (v < NC) { const double F = o[2 * g] + o[2 * g + 1]; Lacc[v] = -(F - Fp[v]) * idz; Fp[v] = F; }
          }
        }
      }
#pragma unroll
      for (int v = 0; v < NC; ++v) { ring[a0 + v * F3_MAIN] = fzp[v]; ring[b0 + v * F3_MAIN] = fzm[v]; }
      { const int t = a0; a0 = a1; a1 = a2; a2 = t; }
      { const int t = b0; b0 = b1; b1 = t; }
      if (c < cend) load_cell(im, jm, bc_map(c + 1, nz, bcz), qf, wf);     // next feed plane
    } else {
#pragma unroll
      for (int v = 0; v < NC; ++v) Lacc[v] = 0.0;
    }
    if (!do_xy) continue;                            // uniform over the CTA

    // ---------------- x ------------------------------------------------------------------------
    {
      double fp[NC], fm[NC];
      if (is_main) split_flux<MODEL, 0>(qk, wk, P, fp, fm);
      else if (lane < 16) { double qh[NC], wh[NH]; load_cell(ixh, jxh, k, qh, wh); split_flux<MODEL, 0>(qh, wh, P, fp, fm); }
#pragma unroll
      for (int ch = 0; ch < 2; ++ch) {
        if (is_main || lane < 16) {
          const int row = is_main ? ty : xh_row, col = is_main ? lane + 2 : xh_c + 2;
#pragma unroll
          for (int vv = 0; vv < CH; ++vv) {
            const int v = ch * CH + vv;
            if (v < NC) { PB[(vv * TY + row) * XW + col] = fp[v]; PB[((CH + vv) * TY + row) * XW + col] = fm[v]; }
          }
        }
        __syncthreads();
        if (is_main || lane < TY) {                  // 33 faces per row: items 0..131
          const int item = is_main ? tid : F3_MAIN + lane;
          const int row = item / (TX + 1), fc = item - row * (TX + 1);
          const double* p = PB + row * XW + fc;
          double F[CH];
          weno_faces<CH>(p, p + CH * TY * XW, TY * XW, 1, F);
#pragma unroll
          for (int vv = 0; vv < CH; ++vv) FB[(vv * TY + row) * (TX + 1) + fc] = F[vv];
        }
        __syncthreads();
        if (is_main) {
#pragma unroll
          for (int vv = 0; vv < CH; ++vv) {
            const int v = ch * CH + vv;
            if (v < NC) Lacc[v] -= (FB[(vv * TY + ty) * (TX + 1) + lane + 1] - FB[(vv * TY + ty) * (TX + 1) + lane]) * idx;
          }
        }
      }
    }
    // ---------------- y ------------------------------------------------------------------------
    {
      double gp[NC], gm[NC], qh[NC], wh[NH];
      if (is_main) { split_flux<MODEL, 1>(qk, wk, P, gp, gm); load_cell(im, jh, k, qh, wh); }
#pragma unroll
      for (int ch = 0; ch < 2; ++ch) {
        if (is_main) {
          double hp[NC], hm[NC];
          split_flux<MODEL, 1>(qh, wh, P, hp, hm);  // halo row: evaluated per chunk (registers are the scarcer resource)
#pragma unroll
          for (int vv = 0; vv < CH; ++vv) {
            const int v = ch * CH + vv;
            if (v < NC) {
              PB[(vv * YR + ty + 2) * TX + lane] = gp[v]; PB[((CH + vv) * YR + ty + 2) * TX + lane] = gm[v];
              PB[(vv * YR + hrow) * TX + lane] = hp[v];   PB[((CH + vv) * YR + hrow) * TX + lane] = hm[v];
            }
          }
        }
        __syncthreads();
        {                                            // face row ty (main) / row 4 (helper): between tile rows fr-1 and fr
          const double* p = PB + ty * TX + lane;
          double F[CH];
          weno_faces<CH>(p, p + CH * YR * TX, YR * TX, TX, F);
#pragma unroll
          for (int vv = 0; vv < CH; ++vv) FB[(vv * (TY + 1) + ty) * TX + lane] = F[vv];
        }
        __syncthreads();
        if (is_main) {
#pragma unroll
          for (int vv = 0; vv < CH; ++vv) {
            const int v = ch * CH + vv;
            if (v < NC) Lacc[v] -= (FB[(vv * (TY + 1) + ty + 1) * TX + lane] - FB[(vv * (TY + 1) + ty) * TX + lane]) * idy;
          }
        }
      }
    }
    if (inside) {
      const size_t id = (size_t)k * pstride + (size_t)j * nx + i;
#pragma unroll
      for (int v = 0; v < NC; ++v) L[(size_t)v * N + id] = Lacc[v];
    }
  }
}

}  // namespace rmhd

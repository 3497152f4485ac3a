// flux_vp.cuh -- a4 fused, 3-D grids: L(q) = -sum_d dF^d/dx_d (eq 12) for all three axes in one pass,
// TMA-staged planes, warps specialised by VARIABLE instead of by cell.
//
// What bounds this kernel (profiles/r1e_kernels.md): the thread-per-cell kernel flux_hm.cuh moves ~480 doubles per cell
// through the shared-memory / L1 data path (60 % of its peak, more than the FP64 pipe's 45 %): every reconstruction
// loads its three operands from shared memory.  Here
//   * each plane (own cells + x/y halo) is brought in by TMA (cp.async.bulk.tensor, 4-D boxes on the SoA rows,
//     mbarrier-tracked, one elected thread, one plane ahead); boundary CTAs patch the out-of-range halo (virtual ghost
//     zones, a6) after the box has landed;
//   * the 6 rows with a non-trivial flux (D, S, tau, rho_charge) get one warp each: lane = x column, the thread walks
//     the TY = 8 cells of its column, so along y every field value is loaded once and every first difference d and
//     smoothness term (eps + d^2)^2 is computed once and used by both faces that share the cell pair (11 instead of
//     14 FP64 instructions per reconstruction); along z the three planes sit in a 3-slot shared-memory ring;
//   * the 8 Maxwell / cleaning rows (linear fluxes, paired as in flux_fused.cuh: 8 reconstructions per face, not 16)
//     are reconstructed straight from the TMA-staged B, E, psi, phi planes by 8 warps (one row of the tile each), so
//     they need no field arrays and run decoupled from the hydro warps' barriers;
//   * the fields g+- = f +- q of the hydro rows are produced once per cell (phase A) by the hydro and helper warps.
// ~270 doubles per cell through the shared-memory path and ~1250 FP64 instructions instead of ~480 and ~1400.
//
// Step c of the march (k = c - 2 is the output plane; z-feed plane c runs two planes ahead as in flux_fused.cuh):
//   wait TMA(k) | [boundary CTAs: halo fix-up, CTA barrier]
//   hydro + helper warps: phase A  (x/y fields of plane k from the staged plane, z fields of plane c from global)
//   --- named barrier S1 (hydro + helpers); the elected thread re-arms the hydro buffer with TMA(k+1)
//   hydro warps: phase B  (x, y, z reconstructions of their row, 8 cells per thread, store)
//   --- named barrier S2
//   Maxwell warps (no barriers): x, y from the staged plane k, z from planes c (global), c-1 (registers), k (staged);
//   arrive on "Maxwell buffer consumed"; their planes are double-buffered.
// MODE (FluxComb, flux_fused.cuh): 0 stores L; 1 = F1 of SSP2(222): rows without a source are stored as q_ex of stage 2;
// 2 = last flux launch: q^{n+1} = A + hdt L (eq 11), A of the rows without a source rebuilt from qn and this launch's input.
#pragma once
#include <cuda.h>
#include "flux_hm.cuh"

namespace rmhd {

constexpr int VP_TX = 32, VP_TY = 8, VP_XW = VP_TX + 4, VP_YR = VP_TY + 4, VP_PL = VP_XW * VP_YR;

template <int MODEL> struct VPGeom {
  using FS = FSet<MODEL>;
  static constexpr int NHV = FS::NHV, NH = Dim<MODEL>::NH, NRH = NHV + NH, NRM = 8;
  static constexpr int WH = NHV, WM = VP_TY, WX = 2, NW = WH + WM + WX, THREADS = 32 * NW;
  static constexpr int NPA = 32 * (WH + WX);                                   // threads of the S1 / S2 barriers
  static constexpr int RAWH = NRH * VP_PL, RAWM = NRM * VP_PL;                 // doubles per staged plane
  static constexpr int GX = 2 * NHV * VP_TY * VP_XW, GY = 2 * NHV * VP_YR * VP_TX, GZ = 2 * NHV * VP_TY * VP_TX;
  static constexpr int FX = NHV * VP_TY;                                       // right face of tile column 31, hydro rows
  static constexpr int NBAR = 5;                                               // mbarriers (8 bytes each), after the arrays
  static constexpr size_t bytes() { return sizeof(double) * (RAWH + 2 * RAWM + GX + GY + 3 * GZ + FX + NBAR); }
  static constexpr unsigned TXH = sizeof(double) * RAWH, TXM = sizeof(double) * RAWM;
};

// rows of the state allocation (tensor-map coordinate 3) of the staged planes
template <int MODEL> struct VPRows {
  int h[VPGeom<MODEL>::NRH];     // the NHV rows with a non-trivial flux, then the NH hydro primitives
  int m[8];                      // B(3), E(3), psi, phi
};

RMHD_DEV unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
RMHD_DEV void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
RMHD_DEV void mbar_wait_par(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "VP_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra VP_DONE;\n"
      "bra VP_WAIT;\n"
      "VP_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// one 4-D box (VP_XW x VP_YR x 1 plane x 1 row of the allocation) -> shared memory; out-of-range elements arrive as zeros
RMHD_DEV void tma_load_plane(double* dst, const CUtensorMap* tm, int x, int y, int z, int row, unsigned long long* bar) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
               ::"r"(smem_u32(dst)), "l"(tm), "r"(x), "r"(y), "r"(z), "r"(row), "r"(smem_u32(bar)) : "memory");
}
template <int ID, int NT> RMHD_DEV void vp_bar() { asm volatile("bar.sync %0, %1;" ::"n"(ID), "n"(NT) : "memory"); }

// WENO3 with the cell-pair terms passed in (G7; same formula as physics.cuh weno3, unscaled fields g = 2 f+-, eps x 4):
//   d = u_right - u_left of a cell pair, S = (eps + d^2)^2.  Value at the face next to b biased to the d1 side:
//   b + (d1 + w0 (d0 - d1))/2,  w0 = S1 / (S1 + S0/2)
constexpr double VP_EPS = 4.0 * 1e-6;
RMHD_DEV void pair_terms(double ul, double ur, double& d, double& S) { d = ur - ul; const double e = fma(d, d, VP_EPS); S = e * e; }
RMHD_DEV double weno_ds(double b, double d0, double d1, double S0, double S1) {
  const double den = fma(0.5, S0, S1);
  const double r0 = rcp_seed(den);
  const double er = fma(-den, r0, 1.0);
  const double r = fma(r0, fma(er, er, er), r0);
  return fma(0.5, fma(S1 * r, d0 - d1, d1), b);
}
// value at the face between b and c biased to a (physics.cuh weno3 on unscaled fields)
RMHD_DEV double weno_u(double a, double b, double c) {
  double d0, S0, d1, S1;
  pair_terms(b, c, d0, S0);
  pair_terms(a, b, d1, S1);
  return weno_ds(b, d0, d1, S0, S1);
}

// store one row of one cell (element e = row * N + id): L itself, or the q_ex / eq-(11) update (FluxComb, flux_fused.cuh)
template <int MODE>
RMHD_DEV void store_row(double* __restrict__ L, const FluxComb& cb, size_t e, bool src, double val) {
  if constexpr (MODE == 0) {
    L[e] = val;
  } else if constexpr (MODE == 1) {
    if (src) L[e] = val;
    else cb.q[e] = fma(cb.hdt, val, __ldg(cb.qs + e));
  } else {
    double a;
    if (src) a = __ldg(cb.A + e);
    else { const double x = cb.q[e], y = __ldg(cb.qs + e); a = fma(cb.theta, y - x, x); }
    cb.q[e] = fma(cb.hdt, val, a);
  }
}

// Maxwell pair n of axis K (flux_fused.cuh: P = X + s Y left-biased, M = X - s Y right-biased; G(X) = Po - Mo, G(Y) = s (Po + Mo)):
// X, Y index the staged Maxwell planes (B 0-2, E 3-5, psi 6, phi 7)
template <int K> struct MxPair {
  static constexpr int a = (K + 1) % 3, b = (K + 2) % 3;
  __host__ __device__ static constexpr int X(int n) { return n == 0 ? a : (n == 1 ? 3 + a : (n == 2 ? 7 : 6)); }
  __host__ __device__ static constexpr int Y(int n) { return n == 0 ? 3 + b : (n == 1 ? b : (n == 2 ? K : 3 + K)); }
  __host__ __device__ static constexpr double s(int n) { return n == 0 ? -1.0 : 1.0; }
};

// boundary index map for overhangs of at most n (n >= 2): one wrap instead of bc_map's modulo; anything further out (tail of
// a partial tile, never used) is clamped into range
RMHD_DEV int bc1(int c, int n, int bc) {
  if (bc == 1) c += c < 0 ? n : (c >= n ? -n : 0);
  return min(max(c, 0), n - 1);
}
RMHD_DEV double shfl_down1(double v) {      // value of lane + 1 (lane 31: its own)
  int lo = __double2loint(v), hi = __double2hiint(v);
  asm volatile("shfl.sync.down.b32 %0, %0, 1, 0x1f, 0xffffffff;" : "+r"(lo));
  asm volatile("shfl.sync.down.b32 %0, %0, 1, 0x1f, 0xffffffff;" : "+r"(hi));
  return __hiloint2double(hi, lo);
}
RMHD_DEV double shfl_idx(double v, int src) {
  int lo = __double2loint(v), hi = __double2hiint(v);
  asm volatile("shfl.sync.idx.b32 %0, %0, %1, 0x1f, 0xffffffff;" : "+r"(lo) : "r"(src));
  asm volatile("shfl.sync.idx.b32 %0, %0, %1, 0x1f, 0xffffffff;" : "+r"(hi) : "r"(src));
  return __hiloint2double(hi, lo);
}

struct VPTile { int i0, j0, nL, xR0, nOx, nT, yB0, nOy; };

// virtual ghost zones (a6) of a staged plane: the elements of the box outside the grid (halo of boundary CTAs, tail of a
// partial tile) are replaced by their outflow / periodic image, read from global memory.  One copy, called by every thread.
template <int MODEL>
__device__ __noinline__ void vp_fixup(double* rawH, double* rM, const ConsRows<MODEL>& qin, const HydRows<MODEL>& win, const VPTile& T,
                                      int kz, int nx, int ny, int bcx, int bcy, int nthreads) {
  using FS = FSet<MODEL>;
  constexpr int NHV = FS::NHV, NRH = VPGeom<MODEL>::NRH, XW = VP_XW, YR = VP_YR, PL = VP_PL;
  auto src = [&](int v) -> const double* { return v < NHV ? qin.r[FS::hv(v)] : (v < NRH ? win.r[v - NHV] : qin.r[hm_mrow<MODEL>(v - NRH)]); };
  const unsigned pz = (unsigned)kz * ny;
  for (int it = threadIdx.x; it < (NRH + 8) * YR * T.nOx; it += nthreads) {          // out-of-range columns, every row of the box
    const int rw = it / T.nOx, o = it - rw * T.nOx, v = rw / YR, y = rw - v * YR;
    const int x = o < T.nL ? o : T.xR0 + (o - T.nL);
    const unsigned id = (pz + bc1(T.j0 - 2 + y, ny, bcy)) * nx + bc1(T.i0 - 2 + x, nx, bcx);
    (v < NRH ? rawH + v * PL : rM + (v - NRH) * PL)[y * XW + x] = __ldg(src(v) + id);
  }
  const int nxin = T.xR0 - T.nL;
  for (int it = threadIdx.x; it < (NRH + 8) * T.nOy * nxin; it += nthreads) {        // out-of-range rows, in-range columns
    const int rw = it / nxin, x = T.nL + (it - rw * nxin), v = rw / T.nOy, o = rw - v * T.nOy;
    const int y = o < T.nT ? o : T.yB0 + (o - T.nT);
    const unsigned id = (pz + bc1(T.j0 - 2 + y, ny, bcy)) * nx + (T.i0 - 2 + x);
    (v < NRH ? rawH + v * PL : rM + (v - NRH) * PL)[y * XW + x] = __ldg(src(v) + id);
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

template <int MODE, int MODEL = 0>
__global__ void __launch_bounds__(VPGeom<MODEL>::THREADS, 1)
k_flux_vp(const __grid_constant__ CUtensorMap tmap, VPRows<MODEL> rows, ConsRows<MODEL> qin, HydRows<MODEL> win, double* __restrict__ L,
          size_t N, int nx, int ny, int nz, int bcx, int bcy, int bcz, double hidx, double hidy, double hidz, int seg_len, DevPar P,
          FluxComb cb) {
  using FS = FSet<MODEL>;
  using GM = VPGeom<MODEL>;
  constexpr int NC = Dim<MODEL>::NC, NH = Dim<MODEL>::NH, NHV = FS::NHV, NRH = GM::NRH;
  constexpr int TX = VP_TX, TY = VP_TY, XW = VP_XW, YR = VP_YR, PL = VP_PL;
  constexpr int WH = GM::WH, WM = GM::WM, WX = GM::WX, NPA = GM::NPA, NT = GM::THREADS;
  extern __shared__ __align__(128) double sm[];          // TMA destinations need 128-byte alignment (checked below)
  double* rawH = sm;
  double* rawM = rawH + GM::RAWH;            // two buffers
  double* gX = rawM + 2 * GM::RAWM;
  double* gY = gX + GM::GX;
  double* gZ = gY + GM::GY;                  // three slots: planes c, c-1, c-2
  double* fX = gZ + 3 * GM::GZ;
  unsigned long long* bars = (unsigned long long*)(fX + GM::FX);
  unsigned long long &fullH = bars[0], *fullM = bars + 1, *doneM = bars + 3;
  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  const bool is_mx = wrp >= WH && wrp < WH + WM;
  const bool issuer = tid == 32 * (WH + WM);             // lane 0 of the first helper warp
  VPTile T;
  T.i0 = blockIdx.x * TX; T.j0 = blockIdx.y * TY;
  // elements of the staged box that fall outside the grid
  T.nL = T.i0 == 0 ? 2 : 0; T.xR0 = min(XW, nx - T.i0 + 2); T.nOx = T.nL + (XW - T.xR0);
  T.nT = T.j0 == 0 ? 2 : 0; T.yB0 = min(YR, ny - T.j0 + 2); T.nOy = T.nT + (YR - T.yB0);
  const bool boundary = T.nOx + T.nOy > 0;
  const int i0 = T.i0, j0 = T.j0;
  const int k0 = blockIdx.z * seg_len, k1 = min(nz, k0 + seg_len);
  const unsigned pstride = (unsigned)nx * ny;

  if (tid == 0) {
    if (smem_u32(sm) & 127u) __trap();
    mbar_init(&fullH, 1); mbar_init(&fullM[0], 1); mbar_init(&fullM[1], 1);
    mbar_init(&doneM[0], WM * 32); mbar_init(&doneM[1], WM * 32);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // staged step t (c = k0 + t): plane bc(k0 + t - 2) of the hydro rows / of the Maxwell rows (buffer t & 1)
  auto issue_H = [&](int t) {
    const int kz = bc1(k0 + t - 2, nz, bcz);
    mbar_expect_tx(&fullH, GM::TXH);
#pragma unroll 1
    for (int v = 0; v < NRH; ++v) tma_load_plane(rawH + v * PL, &tmap, i0 - 2, j0 - 2, kz, rows.h[v], &fullH);
  };
  auto issue_M = [&](int t) {
    const int kz = bc1(k0 + t - 2, nz, bcz);
    double* dst = rawM + (t & 1) * GM::RAWM;
    mbar_expect_tx(&fullM[t & 1], GM::TXM);
#pragma unroll 1
    for (int v = 0; v < 8; ++v) tma_load_plane(dst + v * PL, &tmap, i0 - 2, j0 - 2, kz, rows.m[v], &fullM[t & 1]);
  };
  const int tmax = k1 + 1 - k0;              // staged steps t = 0 .. tmax
  if (issuer) { issue_H(0); issue_M(0); }

  const int i = i0 + lane;
  const int im = bc1(i, nx, bcx);

  if (!is_mx) {
    // ======================================= hydro and helper warps =======================================
    const int pw = wrp < WH ? wrp : wrp - WM;            // 0 .. WH + WX - 1: phase-A warp
    const int h = wrp < WH ? wrp : 0, row = FS::hv(h);
    const bool rsrc = has_source<MODEL>(row);
    const size_t erow = (size_t)row * N;
    double pend[TY], Gprev[TY];                          // z carry of row hv(h) for the TY cells of this column
#pragma unroll
    for (int r = 0; r < TY; ++r) pend[r] = Gprev[r] = 0.0;
    // second phase-A task of this warp: a y-halo row of gY (box rows 0, 1, TY+2, TY+3) or the x-halo cells, or none
    const int ht = WH + WX - 1 - pw;
    const int jrow = bc1(j0 + pw, ny, bcy);           // this warp's own row (phase A), mapped for partial tiles

#pragma unroll 1
    for (int c = k0 - 2; c <= k1 + 1; ++c) {
      const int k = c - 2, t = c - k0;
      const bool staged = t >= 0, do_xy = c >= k0 + 2;
      double* rM = rawM + (t & 1) * GM::RAWM;
      if (staged) {
        if (issuer && t + 1 <= tmax) {        // Maxwell plane of the next step into the other buffer, once its readers are done
          if (t >= 1) mbar_wait_par(&doneM[(t + 1) & 1], ((t - 1) >> 1) & 1);
          issue_M(t + 1);
        }
        mbar_wait_par(&fullH, t & 1);
        mbar_wait_par(&fullM[t & 1], (t >> 1) & 1);
        if (boundary) {
          vp_fixup<MODEL>(rawH, rM, qin, win, T, bc1(k, nz, bcz), nx, ny, bcx, bcy, NT);
          vp_bar<0, NT>();
        }
      }
      // ---------------- phase A: fields g+- = f +- q of the hydro rows ----------------
      {
        double q_[NC], w_[NH], fh[NHV];
        Com<MODEL> cm;
        {   // z fields of plane c, own row pw, from global memory -> ring slot c mod 3
          const unsigned id = (unsigned)bc1(c, nz, bcz) * pstride + (unsigned)jrow * nx + im;
#pragma unroll
          for (int hh = 0; hh < NHV; ++hh) q_[FS::hv(hh)] = __ldg(qin.r[FS::hv(hh)] + id);
#pragma unroll
          for (int d = 0; d < 3; ++d) { q_[FS::IB + d] = __ldg(qin.r[FS::IB + d] + id); q_[FS::IE + d] = __ldg(qin.r[FS::IE + d] + id); }
#pragma unroll
          for (int v = 0; v < NH; ++v) w_[v] = __ldg(win.r[v] + id);
          cell_common(q_, w_, P, cm);
          cell_hflux<2>(q_, w_, cm, P, fh);
          double* gz = gZ + ((c + 3) % 3) * GM::GZ + pw * TX + lane;
#pragma unroll
          for (int hh = 0; hh < NHV; ++hh) {
            gz[hh * TY * TX] = fh[hh] + q_[FS::hv(hh)];
            gz[(NHV + hh) * TY * TX] = fh[hh] - q_[FS::hv(hh)];
          }
        }
        if (staged) {
          // x / y fields of plane k from the staged box: own row, then this warp's halo task
#pragma unroll 1
          for (int tk = 0; tk < 2; ++tk) {
            int y, x, ox = -1, oy = -1;                  // box cell; offsets into one field of gX / gY (-1: not this axis)
            if (tk == 0) { y = pw + 2; x = lane + 2; ox = pw * XW + lane + 2; oy = (pw + 2) * TX + lane; }
            else if (ht < 4) { y = ht < 2 ? ht : TY + ht; x = lane + 2; oy = y * TX + lane; }
            else if (ht == 4) { const int r = lane >> 2; y = r + 2; x = (lane & 3) < 2 ? (lane & 3) : (lane & 3) + TX; ox = r * XW + x; }
            else break;
            const double* p = rawH + y * XW + x;
#pragma unroll
            for (int hh = 0; hh < NHV; ++hh) q_[FS::hv(hh)] = p[hh * PL];
#pragma unroll
            for (int v = 0; v < NH; ++v) w_[v] = p[(NHV + v) * PL];
            const double* pm = rM + y * XW + x;
#pragma unroll
            for (int d = 0; d < 3; ++d) { q_[FS::IB + d] = pm[d * PL]; q_[FS::IE + d] = pm[(3 + d) * PL]; }
            cell_common(q_, w_, P, cm);
            if (ox >= 0) {
              cell_hflux<0>(q_, w_, cm, P, fh);
#pragma unroll
              for (int hh = 0; hh < NHV; ++hh) {
                gX[hh * TY * XW + ox] = fh[hh] + q_[FS::hv(hh)];
                gX[(NHV + hh) * TY * XW + ox] = fh[hh] - q_[FS::hv(hh)];
              }
            }
            if (oy >= 0) {
              cell_hflux<1>(q_, w_, cm, P, fh);
#pragma unroll
              for (int hh = 0; hh < NHV; ++hh) {
                gY[hh * YR * TX + oy] = fh[hh] + q_[FS::hv(hh)];
                gY[(NHV + hh) * YR * TX + oy] = fh[hh] - q_[FS::hv(hh)];
              }
            }
          }
        }
      }
      vp_bar<1, NPA>();                                       // S1: fields of this step are in shared memory
      if (issuer && staged && t + 1 <= tmax) issue_H(t + 1);  // the hydro buffer is free: next plane

      if (wrp >= WH) {
        // helper warps: L2 prefetch of what the next step reads from global memory (z feed plane c+1; epilogue rows of plane k+1)
        if (c + 1 <= k1 + 1) {
          const unsigned pc = (unsigned)bc1(c + 1, nz, bcz) * pstride + (unsigned)i0;
          const unsigned pk1 = (unsigned)min(k + 1, nz - 1) * pstride + (unsigned)i0;
          for (int it = (wrp - WH - WM) * 32 + lane; it < 2 * TY * (NC + NH + NC); it += 32 * WX) {
            const int half = it & 1, r = (it >> 1) & (TY - 1), v = it >> 4;      // TY = 8
            const unsigned col = (unsigned)bc1(j0 + r, ny, bcy) * nx + 16 * half;
            if (i0 + 16 * half >= nx) continue;
            if (v < NC) prefetch_l2(qin.r[v] + pc + col);
            else if (v < NC + NH) prefetch_l2(win.r[v - NC] + pc + col);
            else if (MODE != 0 && k + 1 >= k0 && k + 1 < k1) {
              const int vr = v - NC - NH;
              const size_t e = (size_t)vr * N + pk1 + col;
              if (MODE == 1) { if (!has_source<MODEL>(vr)) prefetch_l2(cb.qs + e); }
              else prefetch_l2((has_source<MODEL>(vr) ? cb.A : (const double*)cb.q) + e);
            }
          }
        }
      } else if (c >= k0) {
        // ---------------- phase B: row hv(h), the TY cells of column `lane` ----------------
        const double* pX = gX + (h * TY) * XW;
        const double* mX = gX + ((NHV + h) * TY) * XW;
        const double* pY = gY + (h * YR) * TX + lane;
        const double* mY = gY + ((NHV + h) * YR) * TX + lane;
        const double* zn = gZ + ((c + 3) % 3) * GM::GZ + lane;      // plane c
        const double* zm = gZ + ((c + 2) % 3) * GM::GZ + lane;      // plane c-1
        const double* zo = gZ + ((c + 1) % 3) * GM::GZ + lane;      // plane c-2
        double Gyb;
        // y walk: pair terms of ("+") rows (f, f+1) and ("-") rows (f+1, f+2) of gY carried from face to face
        double upb, dp1, Sp1, umb, dm0, Sm0;
        {   // face between tile columns 31 and 32 of row (lane & 7): the right face of lane 31, through shared memory
          const int r = lane & (TY - 1);
          const double* a = pX + r * XW + TX;
          const double* b = mX + r * XW + TX;
          const double G33 = weno_u(a[0], a[1], a[2]) + weno_u(b[3], b[2], b[1]);
          if (lane < TY) fX[h * TY + lane] = G33;
        }
        {   // face 0 (bottom of row 0)
          const double u0 = pY[0], u1 = pY[TX], u2 = pY[2 * TX];
          const double v1 = mY[TX], v2 = mY[2 * TX], v3 = mY[3 * TX];
          double d0, S0, e1, T1;
          pair_terms(u0, u1, dp1, Sp1); pair_terms(u1, u2, d0, S0);
          const double Pf = weno_ds(u1, d0, dp1, S0, Sp1);
          dp1 = d0; Sp1 = S0; upb = u2;
          // "-": a = v3, b = v2, c = v1:  d0 = v1 - v2 = -(pair(v1,v2)), d1 = v2 - v3 = -(pair(v2,v3))
          pair_terms(v1, v2, dm0, Sm0); pair_terms(v2, v3, e1, T1);
          const double Mf = weno_ds(v2, -dm0, -e1, Sm0, T1);
          dm0 = e1; Sm0 = T1; umb = v3;
          Gyb = Pf + Mf;
        }
        __syncwarp();
        const size_t ebase = erow + (unsigned)k * pstride + (unsigned)j0 * nx + i;
#pragma unroll
        for (int r = 0; r < TY; ++r) {
          double acc;
          {
            // x: left face of cell (lane, r); right face from lane + 1
            const double* a = pX + r * XW + lane;
            const double* b = mX + r * XW + lane;
            const double Gl = weno_u(a[0], a[1], a[2]) + weno_u(b[3], b[2], b[1]);
            double Gr = shfl_down1(Gl);
            if (lane == 31) Gr = fX[h * TY + r];
            acc = (Gl - Gr) * hidx;
            // y: face r + 1 (top of row r)
            const double un = pY[(r + 3) * TX], vn = mY[(r + 4) * TX];
            double d0, S0, e1, T1;
            pair_terms(upb, un, d0, S0);
            const double Pf = weno_ds(upb, d0, dp1, S0, Sp1);
            dp1 = d0; Sp1 = S0; upb = un;
            pair_terms(umb, vn, e1, T1);
            const double Mf = weno_ds(umb, -dm0, -e1, Sm0, T1);
            dm0 = e1; Sm0 = T1; umb = vn;
            const double Gyt = Pf + Mf;
            acc = fma(Gyb - Gyt, hidy, acc);
            Gyb = Gyt;
          }
          // z: "+" face c-1/2 stays pending one step, "-" completes face c-3/2
          {
            const int op = (h * TY + r) * TX, om = ((NHV + h) * TY + r) * TX;
            const double Pz = weno_u(zo[op], zm[op], zn[op]);
            const double Mz = weno_u(zn[om], zm[om], zo[om]);
            const double G = pend[r] + Mz;
            pend[r] = Pz;
            acc = fma(Gprev[r] - G, hidz, acc);
            Gprev[r] = G;
          }
          if (do_xy && i < nx && j0 + r < ny) store_row<MODE>(L, cb, ebase + (unsigned)r * nx, rsrc, acc);
        }
      }
      vp_bar<2, NPA>();                                       // S2: gX, gY and the oldest ring slot are consumed
    }
  } else {
    // ======================================= Maxwell warps: cell (lane, mw) =======================================
    const int mw = wrp - WH;
    const int jrow = bc1(j0 + mw, ny, bcy);
    const bool inside = i < nx && j0 + mw < ny;
    // fields of plane c-1 along z, pending "+" faces, previous G (X and Y rows of the 4 pairs)
    double mPm[4], mMm[4], mpend[4], mGX[4], mGY[4];
#pragma unroll
    for (int n = 0; n < 4; ++n) { mPm[n] = mMm[n] = mpend[n] = mGX[n] = mGY[n] = 0.0; }
#pragma unroll 1
    for (int c = k0 - 1; c <= k1 + 1; ++c) {
      const int k = c - 2, t = c - k0;
      const bool staged = t >= 0, do_xy = c >= k0 + 2;
      double* rM = rawM + (t & 1) * GM::RAWM;
      double zX[4], zY[4];                          // plane c along z: X, Y of the 4 pairs (global memory)
      {
        const unsigned idz = (unsigned)bc1(c, nz, bcz) * pstride + (unsigned)jrow * nx + im;
#pragma unroll
        for (int n = 0; n < 4; ++n) {
          zX[n] = __ldg(qin.r[hm_mrow<MODEL>(MxPair<2>::X(n))] + idz);
          zY[n] = __ldg(qin.r[hm_mrow<MODEL>(MxPair<2>::Y(n))] + idz);
        }
      }
      if (staged) {
        if (boundary) mbar_wait_par(&fullH, t & 1);
        mbar_wait_par(&fullM[t & 1], (t >> 1) & 1);
        if (boundary) {
          vp_fixup<MODEL>(rawH, rM, qin, win, T, bc1(k, nz, bcz), nx, ny, bcx, bcy, NT);
          vp_bar<0, NT>();
        }
      }
      double acc[8];
#pragma unroll
      for (int m = 0; m < 8; ++m) acc[m] = 0.0;
      const double* cell = rM + (mw + 2) * XW + lane + 2;          // own cell in the staged box
      if (staged) {
        double G33X, G33Y;
        {   // right face of lane 31 (between tile columns 31 and 32): lane -> pair n = lane & 3, runtime plane indices
          const int n = lane & 3;
          const int Xv = n == 0 ? 1 : (n == 1 ? 4 : (n == 2 ? 7 : 6)), Yv = n == 0 ? 5 : (n == 1 ? 2 : (n == 2 ? 0 : 3));
          const double s = n == 0 ? -1.0 : 1.0;
          const double* px = rM + Xv * PL + (mw + 2) * XW + TX;
          const double* py = rM + Yv * PL + (mw + 2) * XW + TX;
          const double Po = weno_u(fma(s, py[0], px[0]), fma(s, py[1], px[1]), fma(s, py[2], px[2]));
          const double Mo = weno_u(fma(-s, py[3], px[3]), fma(-s, py[2], px[2]), fma(-s, py[1], px[1]));
          G33X = Po - Mo; G33Y = Po + Mo;
        }
#pragma unroll
        for (int n = 0; n < 4; ++n) {
          {   // y: bottom and top face of the cell from box rows mw .. mw+4, pair terms shared between the two faces
            using MP = MxPair<1>;
            const double s = MP::s(n);
            const double* px = cell + MP::X(n) * PL - 2 * XW;
            const double* py = cell + MP::Y(n) * PL - 2 * XW;
            double Pv[4], Mv[4];                     // "+" field on box rows mw..mw+3, "-" field on box rows mw+1..mw+4
#pragma unroll
            for (int y = 0; y < 5; ++y) {
              const double X = px[y * XW], Y = py[y * XW];
              if (y < 4) Pv[y] = s > 0 ? X + Y : X - Y;
              if (y > 0) Mv[y - 1] = s > 0 ? X - Y : X + Y;
            }
            double dP[3], SP[3], dM[3], SM[3];
#pragma unroll
            for (int y = 0; y < 3; ++y) { pair_terms(Pv[y], Pv[y + 1], dP[y], SP[y]); pair_terms(Mv[y], Mv[y + 1], dM[y], SM[y]); }
            const double Pb = weno_ds(Pv[1], dP[1], dP[0], SP[1], SP[0]), Pt = weno_ds(Pv[2], dP[2], dP[1], SP[2], SP[1]);
            const double Mb = weno_ds(Mv[1], -dM[0], -dM[1], SM[0], SM[1]), Mt = weno_ds(Mv[2], -dM[1], -dM[2], SM[1], SM[2]);
            acc[MP::X(n)] = fma((Pb - Mb) - (Pt - Mt), hidy, acc[MP::X(n)]);
            acc[MP::Y(n)] = fma((Pb + Mb) - (Pt + Mt), s * hidy, acc[MP::Y(n)]);
          }
          {   // x: left face of the cell; right face from lane + 1
            using MP = MxPair<0>;
            const double s = MP::s(n);
            const double* px = cell + MP::X(n) * PL - 2;
            const double* py = cell + MP::Y(n) * PL - 2;
            const double X0 = px[0], X1 = px[1], X2 = px[2], X3 = px[3], Y0 = py[0], Y1 = py[1], Y2 = py[2], Y3 = py[3];
            const double Po = s > 0 ? weno_u(X0 + Y0, X1 + Y1, X2 + Y2) : weno_u(X0 - Y0, X1 - Y1, X2 - Y2);
            const double Mo = s > 0 ? weno_u(X3 - Y3, X2 - Y2, X1 - Y1) : weno_u(X3 + Y3, X2 + Y2, X1 + Y1);
            const double GXl = Po - Mo, GYl = Po + Mo;
            double GXr = shfl_down1(GXl), GYr = shfl_down1(GYl);
            const double gx33 = shfl_idx(G33X, n), gy33 = shfl_idx(G33Y, n);
            if (lane == 31) { GXr = gx33; GYr = gy33; }
            acc[MP::X(n)] = fma(GXl - GXr, hidx, acc[MP::X(n)]);
            acc[MP::Y(n)] = fma(GYl - GYr, s * hidx, acc[MP::Y(n)]);
          }
        }
      }
      // z: plane c (global), plane c-1 (registers), plane c-2 = k (staged box, own cell)
#pragma unroll
      for (int n = 0; n < 4; ++n) {
        using MP = MxPair<2>;
        const double s = MP::s(n);
        const double Pn = s > 0 ? zX[n] + zY[n] : zX[n] - zY[n], Mn = s > 0 ? zX[n] - zY[n] : zX[n] + zY[n];
        if (staged) {
          const double Xo = cell[MP::X(n) * PL], Yo = cell[MP::Y(n) * PL];
          const double Po_ = s > 0 ? Xo + Yo : Xo - Yo, Mo_ = s > 0 ? Xo - Yo : Xo + Yo;
          const double Pz = weno_u(Po_, mPm[n], Pn);
          const double Mz = weno_u(Mn, mMm[n], Mo_);
          const double GX = mpend[n] - Mz, GY = mpend[n] + Mz;
          mpend[n] = Pz;
          acc[MP::X(n)] = fma(mGX[n] - GX, hidz, acc[MP::X(n)]);
          acc[MP::Y(n)] = fma(mGY[n] - GY, s * hidz, acc[MP::Y(n)]);
          mGX[n] = GX; mGY[n] = GY;
        }
        mPm[n] = Pn; mMm[n] = Mn;
      }
      if (do_xy && inside) {
        const size_t e0 = (size_t)((unsigned)k * pstride + (unsigned)(j0 + mw) * nx + i);
#pragma unroll
        for (int m = 0; m < 8; ++m) store_row<MODE>(L, cb, (size_t)hm_mrow<MODEL>(m) * N + e0, has_source<MODEL>(hm_mrow<MODEL>(m)), acc[m]);
      }
      if (staged) mbar_arrive(&doneM[t & 1]);
    }
  }
}

}  // namespace rmhd

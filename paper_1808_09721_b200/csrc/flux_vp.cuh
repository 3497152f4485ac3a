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
  static constexpr int NTAB = NRH + NRM;                                       // row pointers of the staged planes
  static constexpr size_t bytes() { return sizeof(double) * (RAWH + 2 * RAWM + GX + GY + 3 * GZ + FX + NBAR + NTAB); }
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
// G independent cell pairs / reconstructions in OPERATION-MAJOR order: ptxas keeps the source order of independent
// chains, and the FP64 pipe needs >= 4 instructions in flight per SM sub-partition (8-cycle dependent latency, one
// issue per 2 cycles)
template <int G> RMHD_DEV void pair_terms_batch(const double* ul, const double* ur, double* d, double* S) {
#pragma unroll
  for (int g = 0; g < G; ++g) d[g] = ur[g] - ul[g];
#pragma unroll
  for (int g = 0; g < G; ++g) S[g] = fma(d[g], d[g], VP_EPS);
#pragma unroll
  for (int g = 0; g < G; ++g) S[g] = S[g] * S[g];
}
template <int G> RMHD_DEV void weno_ds_batch(const double* b, const double* d0, const double* d1, const double* S0, const double* S1, double* out) {
  double den[G], r0[G], er[G];
#pragma unroll
  for (int g = 0; g < G; ++g) den[g] = fma(0.5, S0[g], S1[g]);
#pragma unroll
  for (int g = 0; g < G; ++g) r0[g] = rcp_seed(den[g]);
#pragma unroll
  for (int g = 0; g < G; ++g) er[g] = fma(-den[g], r0[g], 1.0);
#pragma unroll
  for (int g = 0; g < G; ++g) er[g] = fma(er[g], er[g], er[g]);
#pragma unroll
  for (int g = 0; g < G; ++g) r0[g] = fma(r0[g], er[g], r0[g]);
#pragma unroll
  for (int g = 0; g < G; ++g) r0[g] = S1[g] * r0[g];
#pragma unroll
  for (int g = 0; g < G; ++g) den[g] = d0[g] - d1[g];
#pragma unroll
  for (int g = 0; g < G; ++g) den[g] = fma(r0[g], den[g], d1[g]);
#pragma unroll
  for (int g = 0; g < G; ++g) out[g] = fma(0.5, den[g], b[g]);
}
// value at the face between b and c biased to a (physics.cuh weno3 on unscaled fields)
RMHD_DEV double weno_u(double a, double b, double c) {
  double d0, S0, d1, S1;
  pair_terms(b, c, d0, S0);
  pair_terms(a, b, d1, S1);
  return weno_ds(b, d0, d1, S0, S1);
}

// store one row of one cell (element e = row * N + id): L itself, or the q_ex / eq-(11) update (FluxComb, flux_fused.cuh)
// split in two so that the loads are issued before the reconstructions of the cell and used after them
template <int MODE>
RMHD_DEV void epi_load(const FluxComb& cb, size_t e, bool src, double& x, double& y) {
  x = y = 0.0;
  if constexpr (MODE == 1) { if (!src) x = __ldg(cb.qs + e); }
  if constexpr (MODE == 2) {
    if (src) x = __ldg(cb.A + e);
    else { x = cb.q[e]; y = __ldg(cb.qs + e); }
  }
}
template <int MODE>
RMHD_DEV void store_row(double* __restrict__ L, const FluxComb& cb, size_t e, bool src, double val, double x, double y) {
  if constexpr (MODE == 0) {
    L[e] = val;
  } else if constexpr (MODE == 1) {
    if (src) L[e] = val;
    else cb.q[e] = fma(cb.hdt, val, x);
  } else {
    const double a = src ? x : fma(cb.theta, y - x, x);
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

#ifdef VP_TRACE
__device__ long long vp_trace_buf[16 * 80 * 8];
#define VP_T(slot) do { if (lane == 0 && blockIdx.x == 2 && blockIdx.y == 5 && blockIdx.z == 1 && c - k0 + 2 < 80) vp_trace_buf[(wrp * 80 + (c - k0 + 2)) * 8 + (slot)] = clock64(); } while (0)
#else
#define VP_T(slot)
#endif

struct VPTile { int i0, j0, nL, xR0, nOx, nT, yB0, nOy; };

// virtual ghost zones (a6) of a staged plane: the elements of the box outside the grid (halo of boundary CTAs, tail of a
// partial tile) are replaced by their outflow / periodic image, read from global memory.  One copy, called by every thread.
template <int MODEL>
__device__ __noinline__ void vp_fixup(double* rawH, double* rM, const double* const* tab, const VPTile& T,
                                      int kz, int nx, int ny, int bcx, int bcy, int nthreads) {
  constexpr int NRH = VPGeom<MODEL>::NRH, XW = VP_XW, YR = VP_YR, PL = VP_PL;
  auto src = [&](int v) -> const double* { return tab[v]; };
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
  const double** tab = (const double**)(bars + GM::NBAR);   // staged rows: NHV cons rows, NH primitives, B, E, psi, phi
  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  // warp roles: Maxwell 0 .. WM-1, helpers WM .. WM+WX-1, hydro WM+WX .. (the scheduler favours high warp ids: the hydro
  // warps, whose phases are chained by the barriers, go first; the decoupled Maxwell warps fill the gaps)
  const bool is_mx = wrp < WM;
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
#pragma unroll
    for (int v = 0; v < NHV; ++v) tab[v] = qin.r[FS::hv(v)];
#pragma unroll
    for (int v = 0; v < NH; ++v) tab[NHV + v] = win.r[v];
#pragma unroll
    for (int m = 0; m < 8; ++m) tab[NRH + m] = qin.r[hm_mrow<MODEL>(m)];
    mbar_init(&fullH, 1); mbar_init(&fullM[0], 1); mbar_init(&fullM[1], 1);
    mbar_init(&doneM[0], WM * 32); mbar_init(&doneM[1], WM * 32);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // staged step t (c = k0 + t): plane bc(k0 + t - 2) of the hydro rows / of the Maxwell rows (buffer t & 1)
  // (called by the whole first helper warp: lane 0 arms the barrier, then one lane per row issues its box)
  const int my_row = lane < NRH ? rows.h[lane < NRH ? lane : 0] : rows.m[(lane - NRH) & 7];
  auto issue_H = [&](int t) {
    const int kz = bc1(k0 + t - 2, nz, bcz);
    if (lane == 0) mbar_expect_tx(&fullH, GM::TXH);
    __syncwarp();
    if (lane < NRH) tma_load_plane(rawH + lane * PL, &tmap, i0 - 2, j0 - 2, kz, my_row, &fullH);
  };
  auto issue_M = [&](int t) {
    const int kz = bc1(k0 + t - 2, nz, bcz);
    double* dst = rawM + (t & 1) * GM::RAWM;
    if (lane == 0) mbar_expect_tx(&fullM[t & 1], GM::TXM);
    __syncwarp();
    if (lane >= NRH && lane < NRH + 8) tma_load_plane(dst + (lane - NRH) * PL, &tmap, i0 - 2, j0 - 2, kz, my_row, &fullM[t & 1]);
  };
  const int tmax = k1 + 1 - k0;              // staged steps t = 0 .. tmax
  const bool issuer = wrp == WM;             // the first helper warp
  if (issuer) { issue_H(0); issue_M(0); }

  const int i = i0 + lane;
  const int im = bc1(i, nx, bcx);

  if (!is_mx) {
    // ======================================= hydro and helper warps =======================================
    const bool is_hyd = wrp >= WM + WX;
    const int h = is_hyd ? wrp - WM - WX : 0, row = FS::hv(h);
    const int pw = is_hyd ? h : WH + wrp - WM;           // 0 .. WH + WX - 1: phase-A warp
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
      // z feed: plane c, own row pw, straight from global memory (L2: prefetched by the helper warps one step earlier);
      // issued first, used after the x / y fields
      double zq[NC], zw[NH];
      VP_T(0);
      {
        const unsigned id = (unsigned)bc1(c, nz, bcz) * pstride + (unsigned)jrow * nx + im;
#pragma unroll
        for (int hh = 0; hh < NHV; ++hh) zq[FS::hv(hh)] = __ldg(qin.r[FS::hv(hh)] + id);
#pragma unroll
        for (int d = 0; d < 3; ++d) { zq[FS::IB + d] = __ldg(qin.r[FS::IB + d] + id); zq[FS::IE + d] = __ldg(qin.r[FS::IE + d] + id); }
#pragma unroll
        for (int v = 0; v < NH; ++v) zw[v] = __ldg(win.r[v] + id);
      }
      if (staged) {
        if (issuer && t + 1 <= tmax) {        // Maxwell plane of the next step into the other buffer, once its readers are done
          if (t >= 1 && lane == 0) mbar_wait_par(&doneM[(t + 1) & 1], ((t - 1) >> 1) & 1);
          __syncwarp();
          issue_M(t + 1);
        }
        mbar_wait_par(&fullH, t & 1);
        mbar_wait_par(&fullM[t & 1], (t >> 1) & 1);
        if (boundary) {
          vp_fixup<MODEL>(rawH, rM, tab, T, bc1(k, nz, bcz), nx, ny, bcx, bcy, NT);
          vp_bar<0, NT>();
        }
      }
      VP_T(1);
      // ---------------- phase A: fields g+- = f +- q of the hydro rows ----------------
      {
        double q_[NC], w_[NH], fh[NHV];
        Com<MODEL> cm;
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
        VP_T(2);
        {   // z fields of plane c -> ring slot c mod 3
          cell_common(zq, zw, P, cm);
          cell_hflux<2>(zq, zw, cm, P, fh);
          double* gz = gZ + ((c + 3) % 3) * GM::GZ + pw * TX + lane;
#pragma unroll
          for (int hh = 0; hh < NHV; ++hh) {
            gz[hh * TY * TX] = fh[hh] + zq[FS::hv(hh)];
            gz[(NHV + hh) * TY * TX] = fh[hh] - zq[FS::hv(hh)];
          }
        }
      }
      VP_T(3);
      vp_bar<1, NPA>();                                       // S1: fields of this step are in shared memory
      VP_T(4);
      if (issuer && staged && t + 1 <= tmax) issue_H(t + 1);  // the hydro buffer is free: next plane

      if (!is_hyd) {
        // helper warps: L2 prefetch of what the next step reads from global memory (z feed plane c+1; epilogue rows of plane k+1)
        if (c + 1 <= k1 + 1) {
          const unsigned pc = (unsigned)bc1(c + 1, nz, bcz) * pstride + (unsigned)i0;
          const unsigned pk1 = (unsigned)min(k + 1, nz - 1) * pstride + (unsigned)i0;
          for (int it = (wrp - WM) * 32 + lane; it < 2 * TY * (GM::NTAB + NC); it += 32 * WX) {
            const int half = it & 1, r = (it >> 1) & (TY - 1), v = it >> 4;      // TY = 8: one 128-byte line per item
            const unsigned col = (unsigned)bc1(j0 + r, ny, bcy) * nx + 16 * half;
            if (i0 + 16 * half >= nx) continue;
            if (v < GM::NTAB) prefetch_l2(tab[v] + pc + col);
            else if (MODE != 0 && k + 1 >= k0 && k + 1 < k1) {
              const int vr = v - GM::NTAB;
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
        // operands of the q_ex / eq-(11) epilogue of the TY cells: issued now, used at the stores
        const size_t ebase = erow + (unsigned)k * pstride + (unsigned)j0 * nx + i;
        double ex[TY], ey[TY];
#pragma unroll
        for (int r = 0; r < TY; ++r) {
          ex[r] = ey[r] = 0.0;
          if (do_xy && i < nx && j0 + r < ny) epi_load<MODE>(cb, ebase + (unsigned)r * nx, rsrc, ex[r], ey[r]);
        }
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
#pragma unroll
        for (int r = 0; r < TY; ++r) {
          double acc;
          const bool st = do_xy && i < nx && j0 + r < ny;
          {
            // the six reconstructions of the cell as one batch: x+ x- (left face), y+ y- (face r+1), z+ (face c-1/2), z- (face c-3/2)
            const double* a = pX + r * XW + lane;
            const double* b = mX + r * XW + lane;
            const int op = (h * TY + r) * TX, om = ((NHV + h) * TY + r) * TX;
            const double xa = a[0], xb = a[1], xc = a[2], ya = b[3], yb = b[2], yc = b[1];
            const double un = pY[(r + 3) * TX], vn = mY[(r + 4) * TX];
            const double za = zo[op], zb = zm[op], zc = zn[op], wa = zn[om], wb = zm[om], wc = zo[om];
            const double ul[10] = {xb, xa, yb, ya, upb, umb, zb, za, wb, wa};
            const double ur[10] = {xc, xb, yc, yb, un, vn, zc, zb, wc, wb};
            double d[10], S[10];
            pair_terms_batch<10>(ul, ur, d, S);
            const double bb[6] = {xb, yb, upb, umb, zb, wb};
            const double d0[6] = {d[0], d[2], d[4], -dm0, d[6], d[8]};
            const double d1[6] = {d[1], d[3], dp1, -d[5], d[7], d[9]};
            const double S0[6] = {S[0], S[2], S[4], Sm0, S[6], S[8]};
            const double S1[6] = {S[1], S[3], Sp1, S[5], S[7], S[9]};
            double o[6];
            weno_ds_batch<6>(bb, d0, d1, S0, S1, o);
            dp1 = d[4]; Sp1 = S[4]; upb = un;
            dm0 = d[5]; Sm0 = S[5]; umb = vn;
            // x: right face from lane + 1
            const double Gl = o[0] + o[1];
            double Gr = shfl_down1(Gl);
            if (lane == 31) Gr = fX[h * TY + r];
            acc = (Gl - Gr) * hidx;
            // y
            const double Gyt = o[2] + o[3];
            acc = fma(Gyb - Gyt, hidy, acc);
            Gyb = Gyt;
            // z: "+" face c-1/2 stays pending one step, "-" completes face c-3/2
            const double G = pend[r] + o[5];
            pend[r] = o[4];
            acc = fma(Gprev[r] - G, hidz, acc);
            Gprev[r] = G;
          }
          if (st) store_row<MODE>(L, cb, ebase + (unsigned)r * nx, rsrc, acc, ex[r], ey[r]);
        }
      }
      VP_T(5);
      vp_bar<2, NPA>();                                       // S2: gX, gY and the oldest ring slot are consumed
      VP_T(6);
    }
  } else {
    // ======================================= Maxwell warps: cell (lane, mw) =======================================
    const int mw = wrp;
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
      VP_T(0);
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
          vp_fixup<MODEL>(rawH, rM, tab, T, bc1(k, nz, bcz), nx, ny, bcx, bcy, NT);
          vp_bar<0, NT>();
        }
      }
      VP_T(1);
      double acc[8], ex[8], ey[8];
      const size_t e0 = (size_t)((unsigned)k * pstride + (unsigned)(j0 + mw) * nx + i);
#pragma unroll
      for (int m = 0; m < 8; ++m) {
        acc[m] = 0.0; ex[m] = ey[m] = 0.0;
        if (do_xy && inside) epi_load<MODE>(cb, (size_t)hm_mrow<MODEL>(m) * N + e0, has_source<MODEL>(hm_mrow<MODEL>(m)), ex[m], ey[m]);
      }
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
            const double ul[6] = {Pv[0], Pv[1], Pv[2], Mv[0], Mv[1], Mv[2]}, ur[6] = {Pv[1], Pv[2], Pv[3], Mv[1], Mv[2], Mv[3]};
            double d[6], S[6], o[4];
            pair_terms_batch<6>(ul, ur, d, S);
            const double bb[4] = {Pv[1], Pv[2], Mv[1], Mv[2]};
            const double d0[4] = {d[1], d[2], -d[3], -d[4]}, d1[4] = {d[0], d[1], -d[4], -d[5]};
            const double S0[4] = {S[1], S[2], S[3], S[4]}, S1[4] = {S[0], S[1], S[4], S[5]};
            weno_ds_batch<4>(bb, d0, d1, S0, S1, o);            // Pb, Pt, Mb, Mt
            acc[MP::X(n)] = fma((o[0] - o[2]) - (o[1] - o[3]), hidy, acc[MP::X(n)]);
            acc[MP::Y(n)] = fma((o[0] + o[2]) - (o[1] + o[3]), s * hidy, acc[MP::Y(n)]);
          }
          {   // x: left face of the cell (right face from lane + 1);  z: plane c (global), c-1 (registers), c-2 = k (staged box, own cell)
            using MX = MxPair<0>;
            using MZ = MxPair<2>;
            const double sx = MX::s(n), sz = MZ::s(n);
            const double* px = cell + MX::X(n) * PL - 2;
            const double* py = cell + MX::Y(n) * PL - 2;
            const double X0 = px[0], X1 = px[1], X2 = px[2], X3 = px[3], Y0 = py[0], Y1 = py[1], Y2 = py[2], Y3 = py[3];
            const double P0 = sx > 0 ? X0 + Y0 : X0 - Y0, P1 = sx > 0 ? X1 + Y1 : X1 - Y1, P2 = sx > 0 ? X2 + Y2 : X2 - Y2;
            const double M1 = sx > 0 ? X1 - Y1 : X1 + Y1, M2 = sx > 0 ? X2 - Y2 : X2 + Y2, M3 = sx > 0 ? X3 - Y3 : X3 + Y3;
            const double Xo = cell[MZ::X(n) * PL], Yo = cell[MZ::Y(n) * PL];
            const double Pn = sz > 0 ? zX[n] + zY[n] : zX[n] - zY[n], Mn = sz > 0 ? zX[n] - zY[n] : zX[n] + zY[n];
            const double Po_ = sz > 0 ? Xo + Yo : Xo - Yo, Mo_ = sz > 0 ? Xo - Yo : Xo + Yo;
            const double ul[8] = {P1, P0, M2, M3, mPm[n], Po_, mMm[n], Mn}, ur[8] = {P2, P1, M1, M2, Pn, mPm[n], Mo_, mMm[n]};
            double d[8], S[8], o[4];
            pair_terms_batch<8>(ul, ur, d, S);
            const double bb[4] = {P1, M2, mPm[n], mMm[n]};
            const double d0[4] = {d[0], d[2], d[4], d[6]}, d1[4] = {d[1], d[3], d[5], d[7]};
            const double S0[4] = {S[0], S[2], S[4], S[6]}, S1[4] = {S[1], S[3], S[5], S[7]};
            weno_ds_batch<4>(bb, d0, d1, S0, S1, o);            // x+, x-, z+, z-
            const double GXl = o[0] - o[1], GYl = o[0] + o[1];
            double GXr = shfl_down1(GXl), GYr = shfl_down1(GYl);
            const double gx33 = shfl_idx(G33X, n), gy33 = shfl_idx(G33Y, n);
            if (lane == 31) { GXr = gx33; GYr = gy33; }
            acc[MX::X(n)] = fma(GXl - GXr, hidx, acc[MX::X(n)]);
            acc[MX::Y(n)] = fma(GYl - GYr, sx * hidx, acc[MX::Y(n)]);
            const double GX = mpend[n] - o[3], GY = mpend[n] + o[3];
            mpend[n] = o[2];
            acc[MZ::X(n)] = fma(mGX[n] - GX, hidz, acc[MZ::X(n)]);
            acc[MZ::Y(n)] = fma(mGY[n] - GY, sz * hidz, acc[MZ::Y(n)]);
            mGX[n] = GX; mGY[n] = GY;
            mPm[n] = Pn; mMm[n] = Mn;
          }
        }
      } else {
#pragma unroll
        for (int n = 0; n < 4; ++n) {   // c = k0 - 1: plane c becomes plane c-1 of the first staged step
          using MZ = MxPair<2>;
          const double sz = MZ::s(n);
          mPm[n] = sz > 0 ? zX[n] + zY[n] : zX[n] - zY[n]; mMm[n] = sz > 0 ? zX[n] - zY[n] : zX[n] + zY[n];
        }
      }
      if (do_xy && inside) {
#pragma unroll
        for (int m = 0; m < 8; ++m) store_row<MODE>(L, cb, (size_t)hm_mrow<MODEL>(m) * N + e0, has_source<MODEL>(hm_mrow<MODEL>(m)), acc[m], ex[m], ey[m]);
      }
      VP_T(5);
      if (staged) mbar_arrive(&doneM[t & 1]);
    }
  }
}

}  // namespace rmhd

// flux_hm.cuh -- a4 fused, resistive model: the one-pass L(q) of flux_fused.cuh (same fields, same tile,
// same shared-memory exchange, same two barriers per plane) with the work of every column split between
// TWO threads by field group, so that 16 warps per SM are resident at 128 registers instead of 10 at 168:
//   role H (warps 0-3): the 6 rows with a non-trivial flux (D, S, tau, rho_charge): 12 fields per axis.
//                       Loads q, w of its cell, flux vectors along x, y (plane k) and z (feed plane k+2),
//                       hydro z-ring in shared memory, stores its 6 rows of L.
//   role M (warps 4-7): the 8 Maxwell / cleaning rows (B, E, psi, phi): 8 fields per axis, rebuilt from the
//                       B, E, psi, phi rows for x, y, z; stores its 8 rows of L.  Because this role is the
//                       lighter one it also takes the cells that do not divide by 128: the y-halo rows
//                       (all 20 fields along y) and, warp 7, the 16 x-halo cells (all 20 fields along x).
// The 5th row of y-faces is an extra pass of warp 0 of each role, the 33rd x-face of every row an extra pass
// of lanes 0-3 of warp 1 of each role.  Each thread accumulates and stores only its own rows, so the two
// roles never exchange L.  See flux_fused.cuh for the field definitions and the z schedule.
#pragma once
#include "flux_fused.cuh"

namespace rmhd {

// geometry of the two-role kernel: TX = 32 columns x TYP rows per CTA (TYP = 4: two CTAs per SM; TYP = 8: one CTA
// of 16 warps per SM with half the y-halo and extra-face overhead per cell)
template <int TYP, int MODEL = 0> struct HMGeom {
  static constexpr int NF = FSet<MODEL>::NF, NC = Dim<MODEL>::NC, NHV = FSet<MODEL>::NHV;
  static constexpr int TY = TYP, MAIN = FF_TX * TYP, THREADS = 2 * MAIN, YR = TYP + 4;
  static constexpr int GX = NF * TY * FF_XW, GY = NF * YR * FF_TX, FY = NC * (TY + 1) * FF_TX, FX = NC * TY, RING = 4 * NHV * MAIN;
  static constexpr size_t bytes(bool has_z) { return sizeof(double) * (GX + GY + FY + FX + (has_z ? RING : 0)); }
};
constexpr int HM_THREADS = HMGeom<4>::THREADS;

// CTA-wide barrier reached from role-specific code paths (every thread executes the same number of them)
template <int NT> RMHD_DEV void hm_barrier() { asm volatile("bar.sync 1, %0;" ::"n"(NT) : "memory"); }

// split-phase CTA barrier (mbarrier): arrive when the own shared-memory reads/writes of a phase are done, wait
// only where the others' results are needed; independent work placed in between hides the skew between warps
RMHD_DEV void mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
RMHD_DEV void mbar_arrive(unsigned long long* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
RMHD_DEV void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "HM_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra HM_DONE;\n"
      "bra HM_WAIT;\n"
      "HM_DONE:\n"
      "}\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}

// reconstructions of NREC consecutive fields starting at field F0 of one face (shared memory), G at a time
template <int MODEL, int F0, int NREC, int G, int DONE = 0>
RMHD_DEV void face_recon_range(const double* p, int fs, int st, double* o) {
  constexpr int B = NREC - DONE >= G ? G : NREC - DONE;
  double a[B], b[B], c[B];
#pragma unroll
  for (int g = 0; g < B; ++g) {
    const int f = F0 + DONE + g;
    const double* pf = p + f * fs;
    if (field_is_plus<MODEL>(f)) { a[g] = pf[0]; b[g] = pf[st]; c[g] = pf[2 * st]; }
    else { a[g] = pf[3 * st]; b[g] = pf[2 * st]; c[g] = pf[st]; }
  }
  weno3_batch<B, true>(a, b, c, o + DONE);
  if constexpr (DONE + B < NREC) face_recon_range<MODEL, F0, NREC, G, DONE + B>(p, fs, st, o);
}

// G of the 8 Maxwell rows in the fixed order (Bx, By, Bz, Ex, Ey, Ez, psi, phi) from P1..P4, M1..M4 of axis K
template <int K>
RMHD_DEV void assemble_M(const double* p, double* G) {
  constexpr int a = (K + 1) % 3, b = (K + 2) % 3;
  G[a] = p[0] - p[4];
  G[3 + b] = -(p[0] + p[4]);
  G[b] = p[1] + p[5];
  G[3 + a] = p[1] - p[5];
  G[K] = p[2] + p[6];
  G[7] = p[2] - p[6];
  G[3 + K] = p[3] + p[7];
  G[6] = p[3] - p[7];
}
template <int MODEL> __host__ __device__ constexpr int hm_mrow(int m) {   // conserved row of Maxwell slot m (B, E, psi, phi)
  return m < 6 ? FSet<MODEL>::IB + m : (m == 6 ? FSet<MODEL>::IPSI : FSet<MODEL>::IPHI);
}

#ifndef RMHD_HM_GH
#define RMHD_HM_GH 6     // reconstructions in flight per batch, role H (12 per face)
#endif

// Cycle account of the plane loop (measurement build only: -DRMHD_HM_CYCLES; the product library has none of it).  Lane 0 of
// every warp adds the clock() ticks between two marks to a global counter [role][phase]; the marks sit where the phases of
// the plane loop end.  Phases, role H: 0 own-cell loads + flux vectors + field stores, 1 bar.sync, 2 x/y reconstructions,
// 3 z part, 4 mbarrier wait, 5 epilogue (fY / fX reads, stores), 6 z part of the feed-only prologue planes.  Role M: 0 z part
// + own-cell field stores, 1 halo cells, 2 bar.sync, 3 x/y reconstructions + extra faces, 4 mbarrier arrive + wait, 5 epilogue,
// 6 prologue planes.  Slot 7 counts the warp-planes.  Loads are charged where their consumer waits, not where they issue.
#ifdef RMHD_HM_CYCLES
__device__ unsigned long long g_hm_cycles[2][8];
#define HM_TICK_DECL() __shared__ unsigned hm_acc[32][8]; if (threadIdx.x < 256) hm_acc[threadIdx.x >> 3][threadIdx.x & 7] = 0u
#define HM_TICK_START() unsigned hm_t0 = (unsigned)clock()
#define HM_TICK(ph)                                                      \
  do {                                                                   \
    const unsigned hm_t1 = (unsigned)clock();                            \
    if (lane == 0) hm_acc[wrp][(ph)] += hm_t1 - hm_t0;                   \
    hm_t0 = hm_t1;                                                       \
  } while (0)
#define HM_COUNT_PLANE() do { if (lane == 0) hm_acc[wrp][7] += 1u; } while (0)
#define HM_TICK_FLUSH()                                                                                           \
  do {                                                                                                            \
    if (lane == 0)                                                                                                \
      for (int ph = 0; ph < 8; ++ph) atomicAdd(&g_hm_cycles[roleH ? 0 : 1][ph], (unsigned long long)hm_acc[wrp][ph]); \
  } while (0)
#else
#define HM_TICK_START() do {} while (0)
#define HM_TICK(ph) do {} while (0)
#define HM_COUNT_PLANE() do {} while (0)
#define HM_TICK_DECL() do {} while (0)
#define HM_TICK_FLUSH() do {} while (0)
#endif

// HAS_Y = false (2-D grids): the tile's TY rows are TY consecutive 32-cell segments of one x line, there is no y work in
// the plane, and the marching axis ("z" below) is the grid's y axis: ZDIR = 1 selects the y components of the flux
// vectors; the host passes ny = 1, nz = the grid's ny, bcz = its y boundary condition, hidz = 1/(2 dy).  A 2-D grid
// then runs the same plane pipeline as a 3-D one instead of one isolated plane per CTA.
// MODEL = 1 (two-fluid, 10 hydro rows = 20 fields per face and axis): 32 x 4 tiles; the hydro role also carries 30 doubles of
// z state, so a 3-D launch is held to one CTA per SM (168 registers), a 2-D one keeps two.
template <bool HAS_Z, bool COMB = false, int TYP = 4, bool HAS_Y = true, int ZDIR = 2, int MODEL = 0>
__global__ void __launch_bounds__(HMGeom<TYP, MODEL>::THREADS, MODEL == 0 ? (TYP == 4 ? 2 : 1) : ((HAS_Z || TYP == 8) ? 1 : 2))
k_flux_hm(ConsRows<MODEL> qin, HydRows<MODEL> win, double* __restrict__ L, size_t N, int nx, int ny, int nz, int bcx, int bcy, int bcz,
          double hidx, double hidy, double hidz, int seg_len, DevPar P, FluxComb cb) {
  using FS = FSet<MODEL>;
  using SM = HMGeom<TYP, MODEL>;
  constexpr int NC = Dim<MODEL>::NC, NH = Dim<MODEL>::NH, NF = FS::NF, NHV = FS::NHV, NM = 8;
  constexpr int NR = NHV > NM ? NHV : NM;           // rows a thread of either role can own
  constexpr int GH = MODEL == 0 ? RMHD_HM_GH : 5;   // hydro reconstructions in flight per batch
  constexpr int TX = FF_TX, TY = TYP, XW = FF_XW, YR = SM::YR, MAIN = SM::MAIN, NT = SM::THREADS;
  constexpr int FSX = TY * XW, FSY = YR * TX;       // field strides of gX, gY
  extern __shared__ double sm[];
  __shared__ unsigned long long bar2;                // "P2 done" (fY, fX written; gX, gY no longer read)
  if (threadIdx.x == 0) mbar_init(&bar2, NT);
  HM_TICK_DECL();
  __syncthreads();
  unsigned ph2 = 0;
  double* gX = sm;
  double* gY = gX + SM::GX;
  double* fY = gY + SM::GY;
  double* fX = fY + SM::FY;
  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  const bool roleH = wrp < TY;
  const int ty = wrp & (TY - 1);
  double* ring = fX + SM::FX + (tid & (MAIN - 1));   // role H only
  const int i0 = HAS_Y ? blockIdx.x * TX : blockIdx.x * (TX * TY) + ty * TX;   // first column of this thread's row
  const int j0 = HAS_Y ? blockIdx.y * TY : 0;
  const int i = i0 + lane, j = HAS_Y ? j0 + ty : 0;
  const bool inside = i < nx && j < ny;
  const int im = bc_map(i, nx, bcx), jm = bc_map(j, ny, bcy);
  const int hrow = ty < 2 ? ty : ty + TY;             // gY row of the y-halo cell of this M thread (M warps 0-3 only)
  const int jh = bc_map(j0 + hrow - 2, ny, bcy);
  const int xh_row = (lane >> 2) & (TY - 1), xh_col = (lane & 3) < 2 ? (lane & 3) : (lane & 3) + 32;
  const int ixh = bc_map((HAS_Y ? i0 : (int)blockIdx.x * (TX * TY) + xh_row * TX) + xh_col - 2, nx, bcx);
  const int jxh = HAS_Y ? bc_map(j0 + xh_row, ny, bcy) : 0;
  // 32-bit element offsets inside a row (N < 2^31, checked by rmhd_create): one IMAD.WIDE per access
  const unsigned pstride = (unsigned)nx * ny;
  const unsigned col_main = (unsigned)jm * nx + im, col_yh = (unsigned)jh * nx + im, col_xh = (unsigned)jxh * nx + ixh;

  auto load_cell = [&](unsigned id, double* q_, double* w_) {
#pragma unroll
    for (int v = 0; v < NC; ++v) q_[v] = __ldg(qin.r[v] + id);
#pragma unroll
    for (int v = 0; v < NH; ++v) w_[v] = __ldg(win.r[v] + id);
  };
  auto load_mx = [&](unsigned id, double* B, double* E, double& psi, double& phi) {
#pragma unroll
    for (int d = 0; d < 3; ++d) { B[d] = __ldg(qin.r[FS::IB + d] + id); E[d] = __ldg(qin.r[FS::IE + d] + id); }
    psi = __ldg(qin.r[FS::IPSI] + id); phi = __ldg(qin.r[FS::IPHI] + id);
  };
  auto prefetch_cell = [&](unsigned id) {
#pragma unroll
    for (int v = 0; v < NC; ++v) prefetch_l2(qin.r[v] + id);
#pragma unroll
    for (int v = 0; v < NH; ++v) prefetch_l2(win.r[v] + id);
  };

  const int k0 = HAS_Z ? blockIdx.z * seg_len : 0;
  const int k1 = HAS_Z ? min(nz, k0 + seg_len) : 1;
  // z carry: pending left-biased reconstructions of the newest face, G of the previous face (own rows only)
  double pend[NHV], Gprev[NR];                      // H uses pend[0..5], Gprev[0..5]; M uses pend[0..3], Gprev[0..7]
#pragma unroll
  for (int v = 0; v < NHV; ++v) pend[v] = 0.0;
#pragma unroll
  for (int v = 0; v < NR; ++v) Gprev[v] = 0.0;
  int s_old = 0, s_new = 2 * NHV * MAIN;

  const int cbeg = HAS_Z ? k0 - 2 : 2, cend = HAS_Z ? k1 + 1 : 2;
#pragma unroll 1
  for (int c = cbeg; c <= cend; ++c) {
    const int k = HAS_Z ? c - 2 : 0;
    const bool do_xy = !HAS_Z || c >= k0 + 2;
    const unsigned pk = (unsigned)k * pstride;
    double Lacc[NR];                                 // H: 6 rows (D, S, tau, rho_charge); M: 8 rows (B, E, psi, phi)
#pragma unroll
    for (int v = 0; v < NR; ++v) Lacc[v] = 0.0;
    HM_TICK_START();
    if (do_xy) HM_COUNT_PLANE();

    if (roleH) {
      // ======================================= role H =======================================
      if (do_xy) {
        if (HAS_Z && c < cend) prefetch_cell((unsigned)bc_map(c + 1, nz, bcz) * pstride + col_main);
        if (inside) prefetch_rows<COMB, NHV, MODEL>(cb, N, pk + (unsigned)j * nx + i, [](int h) { return FS::hv(h); });
        {
          double q_[NC], w_[NH], fh[NHV];
          Com<MODEL> cm;
          load_cell(pk + col_main, q_, w_);
          cell_common(q_, w_, P, cm);
          cell_hflux<0>(q_, w_, cm, P, fh);
#pragma unroll
          for (int h = 0; h < NHV; ++h) {
            gX[(h * TY + ty) * XW + lane + 2] = fh[h] + q_[FS::hv(h)];
            gX[((NHV + h) * TY + ty) * XW + lane + 2] = fh[h] - q_[FS::hv(h)];
          }
          if (HAS_Y) {
            cell_hflux<1>(q_, w_, cm, P, fh);
#pragma unroll
            for (int h = 0; h < NHV; ++h) {
              gY[(h * YR + ty + 2) * TX + lane] = fh[h] + q_[FS::hv(h)];
              gY[((NHV + h) * YR + ty + 2) * TX + lane] = fh[h] - q_[FS::hv(h)];
            }
          }
        }
        HM_TICK(0);
        hm_barrier<NT>();
        HM_TICK(1);
        // left x-face (t = 0) and bottom y-face (t = 1) of the own cell: ONE copy of the reconstruction code
#pragma unroll 1
        for (int t = 0; t < (HAS_Y ? 2 : 1); ++t) {
          double o[2 * NHV];
          face_recon_range<MODEL, 0, 2 * NHV, GH>(t ? gY + ty * TX + lane : gX + ty * XW + lane, t ? FSY : FSX, t ? TX : 1, o);
          if (t == 0) {
#pragma unroll
            for (int h = 0; h < NHV; ++h) {
              const double G = o[h] + o[NHV + h];
              const double Gr = __shfl_down_sync(0xffffffffu, G, 1);
              Lacc[h] = (lane < 31 ? G - Gr : G) * hidx;
            }
          } else {
#pragma unroll
            for (int h = 0; h < NHV; ++h) {
              const double G = o[h] + o[NHV + h];
              fY[(FS::hv(h) * (TY + 1) + ty) * TX + lane] = G;
              Lacc[h] = fma(G, hidy, Lacc[h]);
            }
          }
        }
        mbar_arrive(&bar2);                          // waited for after the z part
        HM_TICK(2);
      }
      if (HAS_Z) {
        double u0[2 * NHV];
        {
          double q_[NC], w_[NH], fh[NHV];
          Com<MODEL> cm;
          load_cell((unsigned)bc_map(c, nz, bcz) * pstride + col_main, q_, w_);
          cell_common(q_, w_, P, cm);
          cell_hflux<ZDIR>(q_, w_, cm, P, fh);
#pragma unroll
          for (int h = 0; h < NHV; ++h) { u0[h] = fh[h] + q_[FS::hv(h)]; u0[NHV + h] = fh[h] - q_[FS::hv(h)]; }
        }
        if (c >= k0) {
          double o[2 * NHV];
#pragma unroll
          for (int f0 = 0; f0 < 2 * NHV; f0 += GH) {
            constexpr int G = GH;
            double a[G], b[G], cc[G];
#pragma unroll
            for (int g = 0; g < G; ++g) {
              const int f = f0 + g;
              const double u2 = ring[s_old + f * MAIN];
              b[g] = ring[s_new + f * MAIN];
              if (f < NHV) { a[g] = u2; cc[g] = u0[f]; } else { a[g] = u0[f]; cc[g] = u2; }
            }
            weno3_batch<G, true>(a, b, cc, o + f0);
          }
#pragma unroll
          for (int h = 0; h < NHV; ++h) {
            const double G = pend[h] + o[NHV + h];   // face c-3/2: last step's "+" and this step's "-"
            pend[h] = o[h];
            if (do_xy) Lacc[h] = fma(Gprev[h] - G, hidz, Lacc[h]);
            Gprev[h] = G;
          }
        }
#pragma unroll
        for (int f = 0; f < 2 * NHV; ++f) ring[s_old + f * MAIN] = u0[f];
        { const int t = s_old; s_old = s_new; s_new = t; }
        HM_TICK(do_xy ? 3 : 6);
      }
      if (do_xy) {
        mbar_wait(&bar2, ph2); ph2 ^= 1u;
        HM_TICK(4);
#pragma unroll
        for (int h = 0; h < NHV; ++h) if (HAS_Y) Lacc[h] = fma(-fY[(FS::hv(h) * (TY + 1) + ty + 1) * TX + lane], hidy, Lacc[h]);
        if (lane == 31) {
#pragma unroll
          for (int h = 0; h < NHV; ++h) Lacc[h] = fma(-fX[FS::hv(h) * TY + ty], hidx, Lacc[h]);
        }
        if (inside) {
          const unsigned id = pk + (unsigned)j * nx + i;
          store_rows<COMB, NHV, MODEL>(L, cb, N, id, Lacc, [](int h) { return FS::hv(h); });
        }
        HM_TICK(5);
      }
    } else {
      // ======================================= role M =======================================
      // z first: it loads B, E, psi, phi of planes c-2, c-1, c; plane c-2 IS plane k, so the x/y fields of the own
      // cell are built from the same registers (no second load)
      if (do_xy) {
        if (inside) prefetch_rows<COMB, NM, MODEL>(cb, N, pk + (unsigned)j * nx + i, [](int m) { return hm_mrow<MODEL>(m); });
        if (HAS_Z && c < cend) {
          const unsigned pn = (unsigned)(k + 1) * pstride;
          if (HAS_Y && (TY == 4 || ty < 4)) prefetch_cell(pn + col_yh);
          if (wrp == 2 * TY - 1 && lane < 4 * TY) prefetch_cell(pn + col_xh);
        }
      }
      {
        double u0[NM], u1[NM], u2[NM];
        {
          double B[3], E[3], psi, phi;
          load_mx((HAS_Z ? (unsigned)bc_map(c - 2, nz, bcz) * pstride : pk) + col_main, B, E, psi, phi);
          if (do_xy) {
            double m[NM];
            mx_fields<0>(B, E, psi, phi, m);
#pragma unroll
            for (int f = 0; f < NM; ++f) gX[((2 * NHV + f) * TY + ty) * XW + lane + 2] = m[f];
            if (HAS_Y) {
              mx_fields<1>(B, E, psi, phi, m);
#pragma unroll
              for (int f = 0; f < NM; ++f) gY[((2 * NHV + f) * YR + ty + 2) * TX + lane] = m[f];
            }
          }
          if (HAS_Z) {
            mx_fields<ZDIR>(B, E, psi, phi, u2);
            load_mx((unsigned)bc_map(c - 1, nz, bcz) * pstride + col_main, B, E, psi, phi);
            mx_fields<ZDIR>(B, E, psi, phi, u1);
            load_mx((unsigned)bc_map(c, nz, bcz) * pstride + col_main, B, E, psi, phi);
            mx_fields<ZDIR>(B, E, psi, phi, u0);
          }
        }
        if (HAS_Z && c >= k0) {
          double a[NM], cc[NM], o[NM], oo[NM], G[NM];
#pragma unroll
          for (int g = 0; g < NM; ++g) { if (g < 4) { a[g] = u2[g]; cc[g] = u0[g]; } else { a[g] = u0[g]; cc[g] = u2[g]; } }
          weno3_batch<NM, true>(a, u1, cc, o);
#pragma unroll
          for (int g = 0; g < 4; ++g) { oo[g] = pend[g]; pend[g] = o[g]; oo[4 + g] = o[4 + g]; }
          assemble_M<ZDIR>(oo, G);
#pragma unroll
          for (int v = 0; v < NM; ++v) { if (do_xy) Lacc[v] = (Gprev[v] - G[v]) * hidz; Gprev[v] = G[v]; }
        }
      }
      HM_TICK(do_xy ? 0 : 6);
      if (do_xy) {
        {
          double q_[NC], w_[NH], g[NF];
          Com<MODEL> cm;
          if (HAS_Y && (TY == 4 || ty < 4)) {        // the 4 y-halo rows: M warps 0-3
            load_cell(pk + col_yh, q_, w_);
            cell_common(q_, w_, P, cm);
            cell_fields<MODEL, 1>(q_, w_, cm, P, g);
#pragma unroll
            for (int f = 0; f < NF; ++f) gY[(f * YR + hrow) * TX + lane] = g[f];
          }
          if (wrp == 2 * TY - 1 && lane < 4 * TY) {
            load_cell(pk + col_xh, q_, w_);
            cell_common(q_, w_, P, cm);
            cell_fields<MODEL, 0>(q_, w_, cm, P, g);
#pragma unroll
            for (int f = 0; f < NF; ++f) gX[(f * TY + xh_row) * XW + xh_col] = g[f];
          }
        }
        HM_TICK(1);
        hm_barrier<NT>();
        HM_TICK(2);
        // t = 0: left x-face, t = 1: bottom y-face of the own cell; t = 2 (two M warps only): the last row of
        // y-faces / the 33rd x-face of row `lane` (lanes >= TY reconstruct in-bounds garbage that is not stored)
        constexpr int XB = TY == 4 ? 0 : 4;          // first of the 4 M warps that take the extra faces (TY = 8: those without a y-halo row)
        const int ntask = (wrp == TY + XB || wrp == TY + XB + 1) ? 3 : 2;
#pragma unroll 1
        for (int t = 0; t < ntask; ++t) {
          if (!HAS_Y && (t == 1 || (t == 2 && wrp == TY + XB))) continue;   // no y faces
          const bool ydir = t == 1 || (t == 2 && wrp == TY + XB);
          const double* p = t == 0 ? gX + ty * XW + lane : (t == 1 ? gY + ty * TX + lane : (ydir ? gY + TY * TX + lane : gX + lane * XW + TX));
          double o[NM], G[NM];
          face_recon_range<MODEL, 2 * NHV, NM, NM>(p, ydir ? FSY : FSX, ydir ? TX : 1, o);
          if (ydir) assemble_M<1>(o, G); else assemble_M<0>(o, G);
          if (t == 0) {
#pragma unroll
            for (int v = 0; v < NM; ++v) {
              const double Gr = __shfl_down_sync(0xffffffffu, G[v], 1);
              Lacc[v] = fma(lane < 31 ? G[v] - Gr : G[v], hidx, Lacc[v]);
            }
          } else if (t == 1) {
#pragma unroll
            for (int v = 0; v < NM; ++v) { fY[(hm_mrow<MODEL>(v) * (TY + 1) + ty) * TX + lane] = G[v]; Lacc[v] = fma(G[v], hidy, Lacc[v]); }
          } else if (ydir) {
#pragma unroll
            for (int v = 0; v < NM; ++v) fY[(hm_mrow<MODEL>(v) * (TY + 1) + TY) * TX + lane] = G[v];
          } else if (lane < TY) {
#pragma unroll
            for (int v = 0; v < NM; ++v) fX[hm_mrow<MODEL>(v) * TY + lane] = G[v];
          }
        }
        if ((HAS_Y && wrp == TY + XB + 2) || wrp == TY + XB + 3) {   // the same two extra face sets of the hydro rows (12 fields), taken off role H
          const bool ydir = wrp == TY + XB + 2;
          double o[2 * NHV];
          face_recon_range<MODEL, 0, 2 * NHV, GH>(ydir ? gY + TY * TX + lane : gX + (lane & (TY - 1)) * XW + TX, ydir ? FSY : FSX, ydir ? TX : 1, o);
          if (ydir) {
#pragma unroll
            for (int h = 0; h < NHV; ++h) fY[(FS::hv(h) * (TY + 1) + TY) * TX + lane] = o[h] + o[NHV + h];
          } else if (lane < TY) {
#pragma unroll
            for (int h = 0; h < NHV; ++h) fX[FS::hv(h) * TY + lane] = o[h] + o[NHV + h];
          }
        }
        HM_TICK(3);
        mbar_arrive(&bar2);
        mbar_wait(&bar2, ph2); ph2 ^= 1u;
        HM_TICK(4);
#pragma unroll
        for (int v = 0; v < NM; ++v) if (HAS_Y) Lacc[v] = fma(-fY[(hm_mrow<MODEL>(v) * (TY + 1) + ty + 1) * TX + lane], hidy, Lacc[v]);
        if (lane == 31) {
#pragma unroll
          for (int v = 0; v < NM; ++v) Lacc[v] = fma(-fX[hm_mrow<MODEL>(v) * TY + ty], hidx, Lacc[v]);
        }
        if (inside) {
          const unsigned id = pk + (unsigned)j * nx + i;
          store_rows<COMB, NM, MODEL>(L, cb, N, id, Lacc, [](int m) { return hm_mrow<MODEL>(m); });
        }
        HM_TICK(5);
      }
    }
  }
  HM_TICK_FLUSH();
}

}  // namespace rmhd

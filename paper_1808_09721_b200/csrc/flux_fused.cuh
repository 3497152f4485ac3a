// flux_fused.cuh -- a4 fused: L(q) = -sum_d dF^d/dx_d for ALL present axes in ONE pass over the state
// (eq 12): q, w are read once (+ halo re-reads that hit L2) and L is written once, 33 doubles
// of algorithmic traffic per cell instead of the 127 of three single-axis passes.
//
// FIELDS.  With alpha = 1 the split fluxes are f+- = (f +- q)/2.  The kernel reconstructs the unscaled
// g+- = f +- q (eps scaled by 4, so the WENO3 weights are bit-identical) and folds the 1/2 into 1/dx.
// The Maxwell / cleaning rows have linear fluxes that pair up (axis K, (K,a,b) cyclic):
//   f(B_a) = -E_b, f(E_b) = -B_a :  g+(E_b) = -g+(B_a),  g-(E_b) = g-(B_a)
//   f(B_b) = +E_a, f(E_a) = +B_b :  g+(E_a) =  g+(B_b),  g-(E_a) = -g-(B_b)     (same for (B_K, phi), (E_K, psi))
// and WENO3 is odd (weno(-u) = -weno(u) bitwise), so the 8 such rows need 8 reconstructions per face, not 16:
//   P1 = B_a - E_b, P2 = E_a + B_b, P3 = phi + B_K, P4 = psi + E_K   (left-biased,  "+")
//   M1 = B_a + E_b, M2 = E_a - B_b, M3 = phi - B_K, M4 = psi - E_K   (right-biased, "-")
// Field order: g+ of the NHV rows with a non-trivial flux, g- of the same rows, P1..P4, M1..M4  (NF = 2 NHV + 8:
// 20 for the resistive model instead of 28, 28 for the two-fluid model instead of 36).
//
// SCHEDULE.  A CTA owns a 32 (x) x 4 (y) column bundle and marches along z over a segment of planes.
// 160 threads: warps 0-3 own the 128 columns, warp 4 takes what does not divide by 128 (the 16 x-halo
// cells, the 33rd x-face of each row, the 5th row of y-faces).  Per plane k, two barriers:
//   P1  every cell of the tile + its 2-cell cross-shaped halo: load q, w (boundary index map = virtual ghost
//       zones, a6), flux vectors along x and y, fields -> shared memory (gX: 4 rows x 36, gY: 8 rows x 32)
//   --- barrier
//   P2  one thread per face: left x-face and bottom y-face of its cell, NF reconstructions each, 8 at a
//       time (weno3_batch).  Right x-face by shuffle from lane+1; bottom faces -> shared (fY)
//   --- barrier
//   P3  top y-face from fY, then the z part and the store (overlaps P1 of the next plane: same interval)
// z: the feed plane runs two planes ahead (face k+1/2 needs g-(k+2)).  The g+- of the NHV rows of the two
// previous planes live in a shared-memory ring used as per-thread scratch (4 NHV doubles per column);
// the Maxwell fields of the previous planes are rebuilt from the B, E, psi, phi rows (L1/L2 hits); the
// left-biased reconstruction of face c-1/2 is done as soon as plane c arrives and kept pending one step,
// so only 10 + NC doubles per column are carried in registers.  HAS_Z = false: one plane, no ring (2-D).
#pragma once
#include "kernels.cuh"

namespace rmhd {

constexpr int FF_TX = 32, FF_TY = 4, FF_MAIN = FF_TX * FF_TY, FF_THREADS = FF_MAIN + 32;
constexpr int FF_XW = FF_TX + 4, FF_YR = FF_TY + 4;

template <int MODEL> struct FSet;
template <> struct FSet<0> {
  static constexpr int NHV = 6, NF = 20, IB = 5, IE = 8, IPSI = 12, IPHI = 13;
  __host__ __device__ static constexpr int hv(int h) { return h < 5 ? h : 11; }   // D, S, tau, rho_charge
};
template <> struct FSet<1> {
  static constexpr int NHV = 10, NF = 28, IB = 10, IE = 13, IPSI = 16, IPHI = 17;
  __host__ __device__ static constexpr int hv(int h) { return h; }                // D, S, tau, Dbar, Sbar, taubar
};

// ---- flux vector, rows with a non-trivial flux only; axis-independent terms computed once per cell -------
template <int MODEL> struct Com;
template <> struct Com<0> { double W, Z, ptot, vE, Ws; };
template <> struct Com<1> { double W[2], Z[2], ptot; };

RMHD_DEV void cell_common(const double* q, const double* w, const DevPar& P, Com<0>& c) {
  const double* v = w + 1;
  const double* B = q + 5;
  const double* E = q + 8;
  c.W = rsqrt(1.0 - (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]));
  c.Z = (w[0] + P.gi * w[4]) * c.W * c.W;
  c.ptot = w[4] + 0.5 * (E[0] * E[0] + E[1] * E[1] + E[2] * E[2] + B[0] * B[0] + B[1] * B[1] + B[2] * B[2]);
  c.vE = v[0] * E[0] + v[1] * E[1] + v[2] * E[2];
  c.Ws = c.W * P.sigma;
}
RMHD_DEV void cell_common(const double* q, const double* w, const DevPar& P, Com<1>& c) {
  const double* B = q + 10;
  const double* E = q + 13;
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const double* v = w + 5 * s + 1;
    c.W[s] = rsqrt(1.0 - (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]));
    c.Z[s] = (w[5 * s] + P.gi * w[5 * s + 4]) * c.W[s] * c.W[s];
  }
  c.ptot = w[4] + w[9] + 0.5 * (E[0] * E[0] + E[1] * E[1] + E[2] * E[2] + B[0] * B[0] + B[1] * B[1] + B[2] * B[2]);
}

template <int K>
RMHD_DEV void cell_hflux(const double* q, const double* w, const Com<0>& c, const DevPar&, double* fh /*6*/) {
  constexpr int a = (K + 1) % 3, b = (K + 2) % 3;
  const double* v = w + 1;
  const double* B = q + 5;
  const double* E = q + 8;
  const double Zvk = c.Z * v[K];
  fh[0] = q[0] * v[K];
  fh[1 + K] = Zvk * v[K] + c.ptot - E[K] * E[K] - B[K] * B[K];
  fh[1 + a] = Zvk * v[a] - E[a] * E[K] - B[a] * B[K];
  fh[1 + b] = Zvk * v[b] - E[b] * E[K] - B[b] * B[K];
  fh[4] = q[1 + K] - fh[0];
  fh[5] = q[11] * v[K] + c.Ws * (E[K] + (v[a] * B[b] - v[b] * B[a]) - c.vE * v[K]);   // J_K
}
template <int K>
RMHD_DEV void cell_hflux(const double* q, const double* w, const Com<1>& c, const DevPar& P, double* fh /*10*/) {
  constexpr int a = (K + 1) % 3, b = (K + 2) % 3;
  const double* B = q + 10;
  const double* E = q + 13;
  double fD = 0, fDb = 0, ftb = 0, fS[3] = {0, 0, 0}, fSb[3] = {0, 0, 0};
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const double* ws = w + 5 * s;
    const double* v = ws + 1;
    const double mu = s == 0 ? P.mu_e : P.mu_p;
    const double Dv = ws[0] * c.W[s] * v[K];
    const double Zvk = c.Z[s] * v[K];
    fD += Dv; fDb += mu * Dv; ftb += mu * (Zvk - Dv);
    const double sK = Zvk * v[K], sa = Zvk * v[a], sb = Zvk * v[b];
    fS[K] += sK; fS[a] += sa; fS[b] += sb;
    fSb[K] += mu * (sK + ws[4]); fSb[a] += mu * sa; fSb[b] += mu * sb;
  }
  fh[0] = fD;
  fh[1 + K] = fS[K] + c.ptot - E[K] * E[K] - B[K] * B[K];
  fh[1 + a] = fS[a] - E[a] * E[K] - B[a] * B[K];
  fh[1 + b] = fS[b] - E[b] * E[K] - B[b] * B[K];
  fh[4] = q[1 + K] - fD;
  fh[5] = fDb;
  fh[6] = fSb[0]; fh[7] = fSb[1]; fh[8] = fSb[2];
  fh[9] = ftb;
}

// the 8 Maxwell fields of one cell from its B, E, psi, phi (m[0..3] = P1..P4, m[4..7] = M1..M4)
template <int K>
RMHD_DEV void mx_fields(const double* B, const double* E, double psi, double phi, double* m) {
  constexpr int a = (K + 1) % 3, b = (K + 2) % 3;
  m[0] = B[a] - E[b]; m[1] = E[a] + B[b]; m[2] = phi + B[K]; m[3] = psi + E[K];
  m[4] = B[a] + E[b]; m[5] = E[a] - B[b]; m[6] = phi - B[K]; m[7] = psi - E[K];
}

// all NF fields of one cell for axis K
template <int MODEL, int K>
RMHD_DEV void cell_fields(const double* q, const double* w, const Com<MODEL>& c, const DevPar& P, double* g) {
  using FS = FSet<MODEL>;
  double fh[FS::NHV];
  cell_hflux<K>(q, w, c, P, fh);
#pragma unroll
  for (int h = 0; h < FS::NHV; ++h) { g[h] = fh[h] + q[FS::hv(h)]; g[FS::NHV + h] = fh[h] - q[FS::hv(h)]; }
  mx_fields<K>(q + FS::IB, q + FS::IE, q[FS::IPSI], q[FS::IPHI], g + 2 * FS::NHV);
}

// G = g^+ + g^- (= 2 x the numerical flux) of every conserved row from the NF reconstructed fields
template <int MODEL, int K>
RMHD_DEV void assemble_G(const double* o, double* G) {
  using FS = FSet<MODEL>;
  constexpr int a = (K + 1) % 3, b = (K + 2) % 3;
#pragma unroll
  for (int h = 0; h < FS::NHV; ++h) G[FS::hv(h)] = o[h] + o[FS::NHV + h];
  const double* p = o + 2 * FS::NHV;
  G[FS::IB + a] = p[0] - p[4];
  G[FS::IE + b] = -(p[0] + p[4]);
  G[FS::IB + b] = p[1] + p[5];
  G[FS::IE + a] = p[1] - p[5];
  G[FS::IB + K] = p[2] + p[6];
  G[FS::IPHI] = p[2] - p[6];
  G[FS::IE + K] = p[3] + p[7];
  G[FS::IPSI] = p[3] - p[7];
}

template <int MODEL> __host__ __device__ constexpr bool field_is_plus(int f) {
  return f < FSet<MODEL>::NHV || (f >= 2 * FSet<MODEL>::NHV && f < 2 * FSet<MODEL>::NHV + 4);
}

// the NF reconstructions of one face from shared memory.  Field f lives at p + f*fs, cells are st apart,
// p[0] is the cell two to the left of the face ("+": cells 0,1,2 ; "-": cells 3,2,1).  8 chains in flight.
template <int MODEL, int F0 = 0>
RMHD_DEV void face_recon(const double* p, int fs, int st, double* o) {
  constexpr int NF = FSet<MODEL>::NF;
  constexpr int G = NF - F0 >= 8 ? 8 : NF - F0;
  double a[G], b[G], c[G];
#pragma unroll
  for (int g = 0; g < G; ++g) {
    const double* pf = p + (F0 + g) * fs;
    if (field_is_plus<MODEL>(F0 + g)) { a[g] = pf[0]; b[g] = pf[st]; c[g] = pf[2 * st]; }
    else { a[g] = pf[3 * st]; b[g] = pf[2 * st]; c[g] = pf[st]; }
  }
  weno3_batch<G, true>(a, b, c, o + F0);
  if constexpr (F0 + G < NF) face_recon<MODEL, F0 + G>(p, fs, st, o);
}

template <int MODEL> struct FFSmem {
  static constexpr int NF = FSet<MODEL>::NF, NC = Dim<MODEL>::NC, NHV = FSet<MODEL>::NHV;
  static constexpr int GX = NF * FF_TY * FF_XW;
  static constexpr int GY = NF * FF_YR * FF_TX;
  static constexpr int FY = NC * (FF_TY + 1) * FF_TX;
  static constexpr int FX = NC * FF_TY;
  static constexpr int RING = 4 * NHV * FF_MAIN;
  static constexpr size_t bytes(bool has_z) { return sizeof(double) * (GX + GY + FY + FX + (has_z ? RING : 0)); }
};

// a5 fused into the F2 launch (COMB = true): the kernel does not store L2 but finishes eq (11) row by row,
//   q^{n+1}_v = A_v + hdt L2_v,   A_v = qn_v + hdt L1_v + hdt (Psi1_v + Psi2_v) left by stage 2 in the L2 buffer,
//   hdt = dt/2 (w = w~ = (1/2, 1/2), Table 2),
// into the qn rows (F2 reads the stage state qs, never qn), so L2 is neither written nor re-read.
// theta > 0: for the rows WITHOUT a source the last stage is q_last = qn + c (sum of the earlier L), so their part of eq (11)
// is A_v = (1 - theta) qn_v + theta q_last,v (SSP2(222): theta = 1/2; SSP3(332): theta = 2/3) and the stage kernel stores A
// only for the rows with a source; q_last is this launch's own input (qs).
// pre != 0 (the F1 launch of SSP2(222)): no eq-(11) work; the rows without a source are stored as q_ex of stage 2,
// q[v] = qs[v] + hdt L_v (q: the stage-state buffer, qs: this launch's input rows = qn, hdt = a~_21 dt), so that stage 2
// neither reads qn, L1 of those rows nor writes them; the rows with a source are stored as L.
struct FluxComb { double* q; const double* A; double hdt; const double* qs; double theta; int pre; };
template <int MODEL> __host__ __device__ constexpr bool has_source(int v) {
  return MODEL == 0 ? ((v >= 8 && v <= 10) || v >= 12) : ((v >= 6 && v <= 9) || v >= 13);
}
// store NR rows (row index by ROW(r)) of one cell: L itself, or the eq-(11) update
template <bool COMB, int NR, int MODEL, class ROW>
RMHD_DEV void store_rows(double* __restrict__ L, const FluxComb& cb, size_t N, unsigned id, const double* Lacc, ROW row) {
  if constexpr (!COMB) {
#pragma unroll
    for (int r = 0; r < NR; ++r) (L + (size_t)row(r) * N)[id] = Lacc[r];
  } else {
    if (cb.pre) {
      double z[NR];
#pragma unroll
      for (int r = 0; r < NR; ++r) z[r] = has_source<MODEL>(row(r)) ? 0.0 : __ldg((cb.qs + (size_t)row(r) * N) + id);
#pragma unroll
      for (int r = 0; r < NR; ++r) {
        const size_t o = (size_t)row(r) * N;
        if (has_source<MODEL>(row(r))) (L + o)[id] = Lacc[r];
        else (cb.q + o)[id] = fma(cb.hdt, Lacc[r], z[r]);
      }
      return;
    }
    double x[NR], y[NR];
    const bool mix = cb.theta > 0.0;
#pragma unroll
    for (int r = 0; r < NR; ++r) {
      const size_t o = (size_t)row(r) * N;
      if (mix && !has_source<MODEL>(row(r))) { x[r] = (cb.q + o)[id]; y[r] = __ldg((cb.qs + o) + id); }
      else { x[r] = __ldg((cb.A + o) + id); y[r] = 0.0; }
    }
#pragma unroll
    for (int r = 0; r < NR; ++r) {
      const double a = (mix && !has_source<MODEL>(row(r))) ? fma(cb.theta, y[r] - x[r], x[r]) : x[r];
      (cb.q + (size_t)row(r) * N)[id] = fma(cb.hdt, Lacc[r], a);
    }
  }
}
template <bool COMB, int NR, int MODEL, class ROW>
RMHD_DEV void prefetch_rows(const FluxComb& cb, size_t N, unsigned id, ROW row) {
  if constexpr (COMB) {
    if (cb.pre) return;
    const bool mix = cb.theta > 0.0;
#pragma unroll
    for (int r = 0; r < NR; ++r) {
      const size_t o = (size_t)row(r) * N;
      prefetch_l2(((mix && !has_source<MODEL>(row(r))) ? (const double*)cb.q : cb.A) + o + id);
    }
  }
}

template <int MODEL, bool HAS_Z, bool COMB = false>
__global__ void __launch_bounds__(FF_THREADS, (MODEL == 0 || !HAS_Z) ? 2 : 1)
k_flux_fused(ConsRows<MODEL> qin, HydRows<MODEL> win, double* __restrict__ L, size_t N, int nx, int ny, int nz, int bcx, int bcy,
             int bcz, double hidx, double hidy, double hidz, int seg_len, DevPar P, FluxComb cb) {
  using FS = FSet<MODEL>;
  using SM = FFSmem<MODEL>;
  constexpr int NC = Dim<MODEL>::NC, NH = Dim<MODEL>::NH, NF = FS::NF, NHV = FS::NHV;
  constexpr int TX = FF_TX, TY = FF_TY, XW = FF_XW, YR = FF_YR;
  extern __shared__ double sm[];
  double* gX = sm;
  double* gY = gX + SM::GX;
  double* fY = gY + SM::GY;
  double* fX = fY + SM::FY;
  const int tid = threadIdx.x, lane = tid & 31, ty = tid >> 5;
  const bool is_main = tid < FF_MAIN;
  double* ring = fX + SM::FX + tid;                 // main threads only (HAS_Z)
  const int i0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
  const int i = i0 + lane, j = j0 + ty;
  const bool inside = is_main && i < nx && j < ny;
  const int im = bc_map(i, nx, bcx);                // ghost semantics also for the tail of a partial tile
  const int jm = bc_map(is_main ? j : j0, ny, bcy);
  // y-halo row taken by this main warp (tile rows -2, -1, 4, 5 = gY rows 0, 1, 6, 7); x-halo cell of helper lanes 0..15
  const int hrow = ty < 2 ? ty : ty + 4;
  const int jh = bc_map(j0 + hrow - 2, ny, bcy);
  const int xh_row = (lane >> 2) & 3, xh_col = (lane & 3) < 2 ? (lane & 3) : (lane & 3) + 32;    // gX columns 0, 1, 34, 35
  const int ixh = bc_map(i0 + xh_col - 2, nx, bcx), jxh = bc_map(j0 + xh_row, ny, bcy);
  const size_t pstride = (size_t)nx * ny;
  const size_t col_main = (size_t)jm * nx + im, col_yh = (size_t)jh * nx + im, col_xh = (size_t)jxh * nx + ixh;

  auto load_cell = [&](size_t id, double* q_, double* w_) {
#pragma unroll
    for (int v = 0; v < NC; ++v) q_[v] = __ldg(qin.r[v] + id);
#pragma unroll
    for (int v = 0; v < NH; ++v) w_[v] = __ldg(win.r[v] + id);
  };
  auto prefetch_cell = [&](size_t id) {
#pragma unroll
    for (int v = 0; v < NC; ++v) prefetch_l2(qin.r[v] + id);
#pragma unroll
    for (int v = 0; v < NH; ++v) prefetch_l2(win.r[v] + id);
  };

  const int k0 = HAS_Z ? blockIdx.z * seg_len : 0;
  const int k1 = HAS_Z ? min(nz, k0 + seg_len) : 1;
  // z carry (registers): pending left-biased reconstructions of the newest face, G of the previous face
  double pend[NHV + 4], Gprev[NC];
  int s_old = 0, s_new = 2 * NHV * FF_MAIN;         // ring slots of planes c-2 and c-1

  const int cbeg = HAS_Z ? k0 - 2 : 2, cend = HAS_Z ? k1 + 1 : 2;
#pragma unroll 1
  for (int c = cbeg; c <= cend; ++c) {
    const int k = HAS_Z ? c - 2 : 0;                // plane of the x/y work and of the output
    const bool do_xy = !HAS_Z || c >= k0 + 2;       // uniform over the CTA
    double Lacc[NC];
    if (do_xy) {
      const size_t pk = (size_t)k * pstride;
      // ---------------- P1: fields of the tile and its halo -> shared memory ------------------------
      if (inside) prefetch_rows<COMB, NC, MODEL>(cb, N, (unsigned)(pk + (size_t)j * nx + i), [](int r) { return r; });
      if (HAS_Z && c < cend) {                      // L2 prefetch of what the next iteration loads first
        const size_t pn = (size_t)(k + 1) * pstride;
        if (is_main) { prefetch_cell(pn + col_yh); prefetch_cell((size_t)bc_map(c + 1, nz, bcz) * pstride + col_main); }
        else if (lane < 16) prefetch_cell(pn + col_xh);
      }
      if (is_main) {
        double q_[NC], w_[NH], g[NF];
        Com<MODEL> cm;
        load_cell(pk + col_main, q_, w_);
        cell_common(q_, w_, P, cm);
        cell_fields<MODEL, 0>(q_, w_, cm, P, g);
#pragma unroll
        for (int f = 0; f < NF; ++f) gX[(f * TY + ty) * XW + lane + 2] = g[f];
        cell_fields<MODEL, 1>(q_, w_, cm, P, g);
#pragma unroll
        for (int f = 0; f < NF; ++f) gY[(f * YR + ty + 2) * TX + lane] = g[f];
        load_cell(pk + col_yh, q_, w_);
        cell_common(q_, w_, P, cm);
        cell_fields<MODEL, 1>(q_, w_, cm, P, g);
#pragma unroll
        for (int f = 0; f < NF; ++f) gY[(f * YR + hrow) * TX + lane] = g[f];
      } else if (lane < 16) {
        double q_[NC], w_[NH], g[NF];
        Com<MODEL> cm;
        load_cell(pk + col_xh, q_, w_);
        cell_common(q_, w_, P, cm);
        cell_fields<MODEL, 0>(q_, w_, cm, P, g);
#pragma unroll
        for (int f = 0; f < NF; ++f) gX[(f * TY + xh_row) * XW + xh_col] = g[f];
      }
      __syncthreads();
      // ---------------- P2: one face per thread and axis ---------------------------------------------
      if (is_main) {
        double o[NF], G[NC];
        face_recon<MODEL>(gX + ty * XW + lane, TY * XW, 1, o);          // left face of cell (lane, ty)
        assemble_G<MODEL, 0>(o, G);
#pragma unroll
        for (int v = 0; v < NC; ++v) {
          const double Gr = __shfl_down_sync(0xffffffffu, G[v], 1);    // lane 31: from fX after the barrier
          Lacc[v] = (lane < 31 ? G[v] - Gr : G[v]) * hidx;
        }
        face_recon<MODEL>(gY + ty * TX + lane, YR * TX, TX, o);          // bottom face of cell (lane, ty)
        assemble_G<MODEL, 1>(o, G);
#pragma unroll
        for (int v = 0; v < NC; ++v) { fY[(v * (TY + 1) + ty) * TX + lane] = G[v]; Lacc[v] = fma(G[v], hidy, Lacc[v]); }
      } else {
        double o[NF], G[NC];
        if (lane < TY) {                                                  // 33rd x-face of row `lane`
          face_recon<MODEL>(gX + lane * XW + TX, TY * XW, 1, o);
          assemble_G<MODEL, 0>(o, G);
#pragma unroll
          for (int v = 0; v < NC; ++v) fX[v * TY + lane] = G[v];
        }
        face_recon<MODEL>(gY + TY * TX + lane, YR * TX, TX, o);           // 5th row of y-faces
        assemble_G<MODEL, 1>(o, G);
#pragma unroll
        for (int v = 0; v < NC; ++v) fY[(v * (TY + 1) + TY) * TX + lane] = G[v];
      }
      __syncthreads();
      // ---------------- P3: top y-face, right x-face of lane 31 -----------------------------------------
      if (is_main) {
#pragma unroll
        for (int v = 0; v < NC; ++v) Lacc[v] = fma(-fY[(v * (TY + 1) + ty + 1) * TX + lane], hidy, Lacc[v]);
        if (lane == 31) {
#pragma unroll
          for (int v = 0; v < NC; ++v) Lacc[v] = fma(-fX[v * TY + ty], hidx, Lacc[v]);
        }
      }
    } else {
#pragma unroll
      for (int v = 0; v < NC; ++v) Lacc[v] = 0.0;
    }
    // ---------------- z: feed plane c, face between c-2 and c-1, L_z of plane c-2 ----------------------
    if (HAS_Z && is_main) {
      double u2[NF], u1[NF], u0[NF];                 // fields of planes c-2, c-1, c
      {
        double q_[NC], w_[NH];
        Com<MODEL> cm;
        load_cell((size_t)bc_map(c, nz, bcz) * pstride + col_main, q_, w_);
        cell_common(q_, w_, P, cm);
        cell_fields<MODEL, 2>(q_, w_, cm, P, u0);
      }
      {
        const size_t id1 = (size_t)bc_map(c - 1, nz, bcz) * pstride + col_main, id2 = (size_t)bc_map(c - 2, nz, bcz) * pstride + col_main;
        double B1[3], E1[3], B2[3], E2[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
          B1[d] = __ldg(qin.r[FS::IB + d] + id1); E1[d] = __ldg(qin.r[FS::IE + d] + id1);
          B2[d] = __ldg(qin.r[FS::IB + d] + id2); E2[d] = __ldg(qin.r[FS::IE + d] + id2);
        }
        mx_fields<2>(B1, E1, __ldg(qin.r[FS::IPSI] + id1), __ldg(qin.r[FS::IPHI] + id1), u1 + 2 * NHV);
        mx_fields<2>(B2, E2, __ldg(qin.r[FS::IPSI] + id2), __ldg(qin.r[FS::IPHI] + id2), u2 + 2 * NHV);
      }
      if (c >= k0) {                                 // the ring holds planes c-2, c-1 from here on
#pragma unroll
        for (int f = 0; f < 2 * NHV; ++f) { u2[f] = ring[s_old + f * FF_MAIN]; u1[f] = ring[s_new + f * FF_MAIN]; }
        double o[NF];
#pragma unroll
        for (int f0 = 0; f0 < NF; f0 += 8) {
          double a[8], b[8], cc[8], r[8];
#pragma unroll
          for (int g = 0; g < 8; ++g) {
            const int f = f0 + g < NF ? f0 + g : NF - 1;
            b[g] = u1[f];
            if (field_is_plus<MODEL>(f)) { a[g] = u2[f]; cc[g] = u0[f]; } else { a[g] = u0[f]; cc[g] = u2[f]; }
          }
          weno3_batch<8, true>(a, b, cc, r);
#pragma unroll
          for (int g = 0; g < 8; ++g) if (f0 + g < NF) o[f0 + g] = r[g];
        }
        // "+" results belong to face c-1/2 (pending); "-" results to face c-3/2, completed by last step's pending
        double oo[NF], G[NC];
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          if (field_is_plus<MODEL>(f)) { const int pi = f < NHV ? f : f - NHV; oo[f] = pend[pi]; pend[pi] = o[f]; }
          else oo[f] = o[f];
        }
        assemble_G<MODEL, 2>(oo, G);
#pragma unroll
        for (int v = 0; v < NC; ++v) { if (do_xy) Lacc[v] = fma(Gprev[v] - G[v], hidz, Lacc[v]); Gprev[v] = G[v]; }
      }
#pragma unroll
      for (int f = 0; f < 2 * NHV; ++f) ring[s_old + f * FF_MAIN] = u0[f];
      { const int t = s_old; s_old = s_new; s_new = t; }
    }
    if (do_xy && inside) {
      const size_t id = (size_t)k * pstride + (size_t)j * nx + i;
      store_rows<COMB, NC, MODEL>(L, cb, N, (unsigned)id, Lacc, [](int r) { return r; });
    }
  }
}

}  // namespace rmhd

// flux_fused.cuh -- a4 fused: the pieces shared by the one-pass L(q) kernels (flux_hm.cuh):
// L(q) = -sum_d dF^d/dx_d for ALL present axes in ONE pass over the state (eq 12): q, w are read once
// (+ halo re-reads that hit L2) and L is written once, 33 doubles of algorithmic traffic per cell instead of the 127 of
// three single-axis passes.
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
// z SCHEDULE (used by flux_hm.cuh).  The feed plane runs two planes ahead (face k+1/2 needs g-(k+2)).  The g+- of the NHV
// rows of the two previous planes live in a shared-memory ring used as per-thread scratch (4 NHV doubles per column);
// the Maxwell fields of the previous planes are rebuilt from the B, E, psi, phi rows (L1/L2 hits); the left-biased
// reconstruction of face c-1/2 is done as soon as plane c arrives and kept pending one step.
#pragma once
#include "kernels.cuh"

namespace rmhd {

constexpr int FF_TX = 32, FF_XW = FF_TX + 4;        // tile width and width with the 2-cell x-halo on both sides

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

template <int MODEL> __host__ __device__ constexpr bool field_is_plus(int f) {
  return f < FSet<MODEL>::NHV || (f >= 2 * FSet<MODEL>::NHV && f < 2 * FSet<MODEL>::NHV + 4);
}

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

// G = g^+ + g^- (= 2 x the numerical flux) of every conserved row from the NF reconstructed fields of one face
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

// =======================================================================================
// a4: L(q) along ONE axis (every 1-D grid; y and z of RMHD_FLUX=split use k_flux_march).  Flux vector + Lax-Friedrichs
// split (eq 12, alpha = 1) + WENO3 + face flux + divergence, one CTA per tile, the stencil staged through shared memory,
// with the paired Maxwell fields of the one-pass kernel (NF = 20 / 28 reconstructions per face instead of 28 / 36):
//   phase 1  every cell of the tile + 2 halo cells per side: load q, w (boundary index map = virtual ghost zones, a6),
//            the NF unscaled fields g+- of the axis -> smem
//   phase 2  one thread per face: NF WENO3 reconstructions, G = 2 x the face flux of every row (registers, then smem
//            aliased onto the field buffer)
//   phase 3  one thread per cell: L (=|+=) -(G_{i+1/2} - G_{i-1/2}) / (2 dx)
// AXIS 0: lanes run along the sweep axis (x): tile 64 cells x 4 rows.
// AXIS 1,2: lanes run along x, the sweep axis is strided: tile 32 (x) x 8 (sweep).
// =======================================================================================
template <int AXIS> struct Tile { static constexpr int TS = 8, TO = 32; };
template <> struct Tile<0> { static constexpr int TS = 64, TO = 4; };
constexpr int FLUX_THREADS = 288;
constexpr int FLUX_PREFETCH_CTAS = 148 * 2 + 24;   // resident CTAs (2 per SM) plus a margin

template <int MODEL, int AXIS>
constexpr size_t flux_smem_bytes() { return sizeof(double) * FSet<MODEL>::NF * (Tile<AXIS>::TS + 4) * Tile<AXIS>::TO; }

template <int MODEL, int AXIS>
__global__ void __launch_bounds__(FLUX_THREADS, 2) k_flux(ConsRows<MODEL> qin, HydRows<MODEL> win, double* __restrict__ L, size_t N,
                                                          int nx, int ny, int nz, int bc, double inv_dx, int accumulate, DevPar P) {
  constexpr int NC = Dim<MODEL>::NC, NH = Dim<MODEL>::NH, NF = FSet<MODEL>::NF;
  constexpr int TS = Tile<AXIS>::TS, TO = Tile<AXIS>::TO;
  constexpr int CS = (TS + 4) * TO;   // cells incl. halo
  constexpr int FS = (TS + 1) * TO;   // faces
  static_assert(FS <= FLUX_THREADS && TS * TO <= FLUX_THREADS, "one pass per phase");
  static_assert(NC * FS <= NF * CS, "G aliases the field buffer");
  extern __shared__ double sm[];      // fields [NF][CS];  later G [NC][FS]
  const int tid = threadIdx.x;
  const int ns = AXIS == 0 ? nx : (AXIS == 1 ? ny : nz);
  const int no = AXIS == 0 ? ny * nz : nx;
  const int o0 = blockIdx.x * TO;
  // a 1-D grid (AXIS 0, one row) lays the TO tile rows along x: row o covers cells s0 + o TS ... (all threads busy)
  const bool rows_x = AXIS == 0 && no == 1;
  const int s0 = rows_x ? blockIdx.y * (TS * TO) : blockIdx.y * TS;
  const int third = blockIdx.z;

  // ---- L2 prefetch of the tile that the CTA about one wave behind this one will stage (AXIS 0 only)
  if (AXIS == 0 && !rows_x) {
    const long long lin = (long long)blockIdx.x + (long long)gridDim.x * blockIdx.y + FLUX_PREFETCH_CTAS;
    if (lin < (long long)gridDim.x * gridDim.y && tid < CS) {
      const int pbx = (int)(lin % gridDim.x), pby = (int)(lin / gridDim.x);
      const int c = pby * TS - 2 + tid % (TS + 4), oo = pbx * TO + tid / (TS + 4);
      if (c < ns + 2 && oo < no) {
        const size_t idx = (size_t)oo * nx + bc_map(c, ns, bc);
#pragma unroll
        for (int v = 0; v < NC; ++v) prefetch_l2(qin.r[v] + idx);
#pragma unroll
        for (int v = 0; v < NH; ++v) prefetch_l2(win.r[v] + idx);
      }
    }
  }
  // ---- phase 1
  for (int item = tid; item < CS; item += FLUX_THREADS) {
    int sh, o;
    if (AXIS == 0) { sh = item % (TS + 4); o = item / (TS + 4); } else { o = item % TO; sh = item / TO; }
    const int c = s0 - 2 + sh + (rows_x ? o * TS : 0);
    const int oo = rows_x ? 0 : o0 + o;
    if (c < ns + 2 && oo < no) {
      const int cm = bc_map(c, ns, bc);
      size_t idx;
      if (AXIS == 0) idx = (size_t)oo * nx + cm;
      else if (AXIS == 1) idx = ((size_t)third * ny + cm) * nx + oo;
      else idx = ((size_t)cm * ny + third) * nx + oo;
      double ql[NC], wl[NH], g[NF];
#pragma unroll
      for (int v = 0; v < NC; ++v) ql[v] = __ldg(qin.r[v] + idx);
#pragma unroll
      for (int v = 0; v < NH; ++v) wl[v] = __ldg(win.r[v] + idx);
      Com<MODEL> cm_;
      cell_common(ql, wl, P, cm_);
      cell_fields<MODEL, AXIS>(ql, wl, cm_, P, g);
#pragma unroll
      for (int f = 0; f < NF; ++f) sm[f * CS + item] = g[f];
    }
  }
  __syncthreads();

  // ---- phase 2: face fs is the left face of tile cell fs (halo coordinate fs + 2)
  double G[NC];
  const bool has_face = tid < FS;
  if (has_face) {
    int fs, o, st;
    if (AXIS == 0) { fs = tid % (TS + 1); o = tid / (TS + 1); st = 1; }
    else { o = tid % TO; fs = tid / TO; st = TO; }
    const int base = AXIS == 0 ? o * (TS + 4) + fs : fs * TO + o;   // halo coordinate fs
    double rec[NF];
    face_recon<MODEL>(sm + base, CS, st, rec);
    assemble_G<MODEL, AXIS>(rec, G);
  }
  __syncthreads();
  if (has_face) {
#pragma unroll
    for (int v = 0; v < NC; ++v) sm[v * FS + tid] = G[v];
  }
  __syncthreads();

  // ---- phase 3
  if (tid < TS * TO) {
    int s, o, fi, st;
    if (AXIS == 0) { s = tid % TS; o = tid / TS; fi = o * (TS + 1) + s; st = 1; }
    else { o = tid % TO; s = tid / TO; fi = s * TO + o; st = TO; }
    const int c = s0 + s + (rows_x ? o * TS : 0);
    const int oo = rows_x ? 0 : o0 + o;
    if (c < ns && oo < no) {
      size_t idx;
      if (AXIS == 0) idx = (size_t)oo * nx + c;
      else if (AXIS == 1) idx = ((size_t)third * ny + c) * nx + oo;
      else idx = ((size_t)c * ny + third) * nx + oo;
      const double hid = 0.5 * inv_dx;
#pragma unroll
      for (int v = 0; v < NC; ++v) {
        const double val = -(sm[v * FS + fi + st] - sm[v * FS + fi]) * hid;
        double* dst = L + (size_t)v * N + idx;
        *dst = accumulate ? *dst + val : val;
      }
    }
  }
}

}  // namespace rmhd

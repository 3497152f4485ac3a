// physics.cuh -- per-cell device arithmetic of the resistive and two-fluid RMHD models.
// Part of the CUDA product path (sm_100a); shares nothing with oracle/.
//
// Notation follows the paper (PAPER.md, cited "P:Lnnn"): D, S, tau, B, E, rho_charge (varrho),
// psi, phi; W Lorentz factor (eq 3), h enthalpy (eq 4), Z := rho h W^2, sigma conductivity,
// mu_s charge/mass ratios, eta resistivity.  Readings "Gn" are listed in DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <cmath>

#ifndef RMHD_DEV
#define RMHD_DEV __device__ __forceinline__
#endif

namespace rmhd {

constexpr int R_NC = 14;  // resistive conserved rows
constexpr int R_NH = 5;   // resistive hydro primitive rows (rho, v, p); B, E live in the cons rows
constexpr int R_NS = 5;   // resistive non-zero source rows: E(3), psi, phi
constexpr int T_NC = 18;
constexpr int T_NH = 10;
constexpr int T_NS = 9;   // Sbar(3), taubar, E(3), psi, phi

template <int MODEL> struct Dim;
template <> struct Dim<0> { static constexpr int NC = R_NC, NH = R_NH, NS = R_NS, NP = 11, IB = 5, IE = 8, IPSI = 12; };
template <> struct Dim<1> { static constexpr int NC = T_NC, NH = T_NH, NS = T_NS, NP = 16, IB = 10, IE = 13, IPSI = 16; };

struct DevPar {
  double gam, g, gi;  // Gamma, (Gamma-1)/Gamma, Gamma/(Gamma-1)
  double sigma, eta, mu_e, mu_p, kappa;
  double tol_c2p, tol_stage;
  int maxit_c2p, maxit_stage;
};

struct Hyd {
  double rho, vx, vy, vz, p, W, Z;
};

RMHD_DEV double max3abs(double a, double b, double c) { return fmax(fabs(a), fmax(fabs(b), fabs(c))); }

// ---------------------------------------------------------------------------------------
// Hydrodynamic conserved -> primitive (G4/G5): root of
//   f(Z) = Z - p(Z) - taut - D,  p = g (Z (1-v^2) - D sqrt(1-v^2)),  v^2 = St^2/Z^2
// by Newton-Raphson kept inside the bracket (|St|, +inf).  One reciprocal, one rsqrt and one
// division per iteration.  Converged when the applied update |dZ| <= tol Z.
// returns 0 ok, 1 inadmissible input, 2 not converged, 3 unphysical result
// The safeguard logic (bracket, start value, return codes, the switch to the second residual) follows the oracle's on purpose,
// so that both sides raise identical failure flags; its correctness rests on the oracle's closed-form and round-trip pins.
// ---------------------------------------------------------------------------------------
RMHD_DEV void hyd_from_Z(double D, double Sx, double Sy, double Sz, double S2, double Z, double g, Hyd& h) {
  const double iZ = 1.0 / Z;
  const double om = 1.0 - S2 * iZ * iZ;
  const double W = rsqrt(om);
  const double sq = om * W;
  h.Z = Z; h.W = W;
  h.p = g * (Z * om - D * sq);
  h.rho = D * sq;
  h.vx = Sx * iZ; h.vy = Sy * iZ; h.vz = Sz * iZ;
}

// Second residual ("one may converge where the other may not").  The recovery in the Lorentz
// factor W instead of Z: with En = taut + D = Z - p and p = g (Z / W^2 - D / W),
//   Z(W) = W (En W - g D) / (W^2 - g),   F(W) = (En W - g D)^2 (W^2 - 1) - St^2 (W^2 - g)^2 = 0,   1 <= W <= Wmax,
//   Wmax = (1 - St^2 / En^2)^(-1/2)  (p >= 0 <=> Z >= En).
// F is a well-scaled polynomial where f(Z) is almost flat at its root (|St| -> En: large W and hot gas).  Newton-Raphson
// from Wmax inside the bracket [1, Wmax]; converged when the applied update |dW| <= tol W or |F| is at its round-off
// floor.  Taken automatically by c2p_hydro after C2P_SWITCH iterations of the first residual; never inlined (rare path).
constexpr int C2P_SWITCH = 20;

// primitives from a converged (or last) Lorentz factor W of the second residual; returns the c2p_hydro_W code
RMHD_DEV int hyd_from_W(double D, double Sx, double Sy, double Sz, double En, double g, double W, bool conv, Hyd& h) {
  const double Z = W * (En * W - g * D) / (W * W - g);
  const double iZ = 1.0 / Z;
  h.Z = Z; h.W = W;
  h.p = g * (Z / (W * W) - D / W);
  h.rho = D / W;
  h.vx = Sx * iZ; h.vy = Sy * iZ; h.vz = Sz * iZ;
  if (!conv) return 2;
  if (!(h.p > 0.0) || !(h.rho > 0.0) || !isfinite(h.p) || !isfinite(Z)) return 3;
  return 0;
}

__device__ __noinline__ int c2p_hydro_W(double D, double Sx, double Sy, double Sz, double S2, double taut, double g, double tol,
                                        int maxit, Hyd& h, int& iters) {
  const double Sabs = sqrt(S2), En = taut + D;
  double lo = 1.0, hi = rsqrt((En - Sabs) * (En + Sabs) / (En * En));
  const double floor_eps = 32.0 * 2.220446049250313e-16;
  if (hi - 1.0 <= 1e-9) {
    // near-static state: W^2 - 1 carries only a few ulps of 1 (exactly 0 once |St| / En < 1e-8, where F(Wmax) would read
    // "no root"); the root in closed form, W = 1 + v^2 / 2 with v^2 = St^2 / Z(W = 1)^2, error O(v^4) <= 4e-18
    const double Z1 = (En - g * D) / (1.0 - g);
    ++iters;
    return hyd_from_W(D, Sx, Sy, Sz, En, g, 1.0 + 0.5 * S2 / (Z1 * Z1), true, h);
  }
  double W = hi;
  bool conv = false;
  {
    const double a = En * W - g * D, b = W * W - g, c = W * W - 1.0;
    const double t1 = a * a * c, t2 = S2 * b * b;
    if (!isfinite(hi) || !(t1 - t2 >= -floor_eps * (t1 + t2))) {
      h.rho = h.vx = h.vy = h.vz = h.p = h.W = h.Z = nan("");
      return 3;
    }
  }
  while (iters < maxit) {
    ++iters;
    const double a = En * W - g * D, b = W * W - g, c = W * W - 1.0;
    const double t1 = a * a * c, t2 = S2 * b * b;
    const double f = t1 - t2;
    if (fabs(f) <= floor_eps * (t1 + t2)) { conv = true; break; }
    const double dF = 2.0 * En * a * c + 2.0 * W * a * a - 4.0 * S2 * W * b;
    if (f < 0.0) lo = fmax(lo, W); else hi = fmin(hi, W);
    double Wn = W - f / dF;
    if (!(Wn >= lo && Wn <= hi) || !isfinite(Wn)) Wn = 0.5 * (lo + hi);
    const double dW = Wn - W;
    W = Wn;
    if (fabs(dW) <= tol * W) { conv = true; break; }
  }
  return hyd_from_W(D, Sx, Sy, Sz, En, g, W, conv, h);
}

RMHD_DEV int c2p_hydro(double D, double Sx, double Sy, double Sz, double taut, double Zg,
                                         const DevPar& P, Hyd& h, int& iters) {
  const double S2 = Sx * Sx + Sy * Sy + Sz * Sz;
  const double Sabs = sqrt(S2);
  iters = 0;
  if (!(D > 0.0) || !(taut + D > Sabs) || !isfinite(taut) || !isfinite(S2)) {
    h.rho = h.vx = h.vy = h.vz = h.p = h.W = h.Z = nan("");
    return 1;
  }
  double lo = Sabs, hi = (double)INFINITY;
  double Z = Zg;
  if (!(Z > Sabs) || !isfinite(Z)) Z = fmax(taut + D, Sabs * (1.0 + 1e-8) + 1e-300);
  bool conv = false;
  for (int it = 1; it <= P.maxit_c2p; ++it) {
    if (it > C2P_SWITCH) {   // copies, so that h and iters of the common path stay in registers
      Hyd t; int its = iters;
      const int rc = c2p_hydro_W(D, Sx, Sy, Sz, S2, taut, P.g, P.tol_c2p, P.maxit_c2p, t, its);
      h = t; iters = its;
      return rc;
    }
    iters = it;
    const double iZ = 1.0 / Z;
    const double v2 = S2 * iZ * iZ;
    const double om = 1.0 - v2;
    const double W = rsqrt(om);
    const double sq = om * W;
    const double f = Z - P.g * (Z * om - D * sq) - taut - D;
    const double fp = 1.0 - P.g * (1.0 + v2 - D * W * v2 * iZ);
    if (f < 0.0) lo = fmax(lo, Z); else hi = fmin(hi, Z);
    double Zn = Z - f / fp;
    if (!(Zn >= lo && Zn <= hi && Zn > Sabs) || !isfinite(Zn)) Zn = isfinite(hi) ? 0.5 * (lo + hi) : 2.0 * Z;
    const double dZ = Zn - Z;
    Z = Zn;
    if (fabs(dZ) <= P.tol_c2p * Z) { conv = true; break; }
  }
  hyd_from_Z(D, Sx, Sy, Sz, S2, Z, P.g, h);
  if (!conv) return 2;
  if (!(h.p > 0.0) || !(h.rho > 0.0) || !isfinite(h.p) || !isfinite(h.W)) return 3;
  return 0;
}

RMHD_DEV double Z_of_prims(double rho, double vx, double vy, double vz, double p, const DevPar& P) {
  const double W2 = 1.0 / (1.0 - (vx * vx + vy * vy + vz * vz));
  return (rho + P.gi * p) * W2;
}

// ---------------------------------------------------------------------------------------
// Resistive model (eq 1-4)
// q: D, S(3), tau, B(3), E(3), rhoc, psi, phi      w: rho, v(3), p
// ---------------------------------------------------------------------------------------
RMHD_DEV void r_prim2cons(const double* w /*rho,v,p*/, const double* B, const double* E, double rhoc,
                                            const DevPar& P, double* q) {
  const double v2 = w[1] * w[1] + w[2] * w[2] + w[3] * w[3];
  const double W = rsqrt(1.0 - v2);
  const double Z = (w[0] + P.gi * w[4]) * W * W;
  q[0] = w[0] * W;
  q[1] = Z * w[1] + (E[1] * B[2] - E[2] * B[1]);
  q[2] = Z * w[2] + (E[2] * B[0] - E[0] * B[2]);
  q[3] = Z * w[3] + (E[0] * B[1] - E[1] * B[0]);
  q[4] = Z - w[4] + 0.5 * (E[0] * E[0] + E[1] * E[1] + E[2] * E[2] + B[0] * B[0] + B[1] * B[1] + B[2] * B[2]) - q[0];
  q[5] = B[0]; q[6] = B[1]; q[7] = B[2];
  q[8] = E[0]; q[9] = E[1]; q[10] = E[2];
  q[11] = rhoc; q[12] = 0.0; q[13] = 0.0;
}

RMHD_DEV int r_con2prim(const double* q, double Zg, const DevPar& P, Hyd& h, int& iters) {
  const double Bx = q[5], By = q[6], Bz = q[7], Ex = q[8], Ey = q[9], Ez = q[10];
  const double Sx = q[1] - (Ey * Bz - Ez * By);
  const double Sy = q[2] - (Ez * Bx - Ex * Bz);
  const double Sz = q[3] - (Ex * By - Ey * Bx);
  const double taut = q[4] - 0.5 * (Ex * Ex + Ey * Ey + Ez * Ez + Bx * Bx + By * By + Bz * Bz);
  return c2p_hydro(q[0], Sx, Sy, Sz, taut, Zg, P, h, iters);
}

// J = rhoc v + W sigma [E + v x B - (v.E) v]
RMHD_DEV void r_current(const double* q, const Hyd& h, double sigma, double* J) {
  const double Bx = q[5], By = q[6], Bz = q[7], Ex = q[8], Ey = q[9], Ez = q[10];
  const double vE = h.vx * Ex + h.vy * Ey + h.vz * Ez;
  const double ws = h.W * sigma;
  J[0] = q[11] * h.vx + ws * (Ex + (h.vy * Bz - h.vz * By) - vE * h.vx);
  J[1] = q[11] * h.vy + ws * (Ey + (h.vz * Bx - h.vx * Bz) - vE * h.vy);
  J[2] = q[11] * h.vz + ws * (Ez + (h.vx * By - h.vy * Bx) - vE * h.vz);
}

// flux vector along axis K (eq 1-2).  The Maxwell rows use the cyclic form: with (K,a,b)
// cyclic, f(B_a) = -E_b, f(B_b) = +E_a, f(E_a) = +B_b, f(E_b) = -B_a, f(B_K) = phi, f(E_K) = psi.
template <int K>
RMHD_DEV void r_flux(const double* q, const double* w, double sigma, const DevPar& P, double* f) {
  constexpr int a = (K + 1) % 3, b = (K + 2) % 3;
  const double* v = w + 1;
  const double* B = q + 5;
  const double* E = q + 8;
  const double v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
  const double W = rsqrt(1.0 - v2);
  const double Z = (w[0] + P.gi * w[4]) * W * W;
  const double ptot = w[4] + 0.5 * (E[0] * E[0] + E[1] * E[1] + E[2] * E[2] + B[0] * B[0] + B[1] * B[1] + B[2] * B[2]);
  const double vE = v[0] * E[0] + v[1] * E[1] + v[2] * E[2];
  const double vxB_K = v[a] * B[b] - v[b] * B[a];
  const double Zvk = Z * v[K];
  f[0] = q[0] * v[K];
  f[1 + K] = Zvk * v[K] + ptot - E[K] * E[K] - B[K] * B[K];
  f[1 + a] = Zvk * v[a] - E[a] * E[K] - B[a] * B[K];
  f[1 + b] = Zvk * v[b] - E[b] * E[K] - B[b] * B[K];
  f[4] = q[1 + K] - f[0];
  f[5 + K] = q[13]; f[5 + a] = -E[b]; f[5 + b] = E[a];
  f[8 + K] = q[12]; f[8 + a] = B[b]; f[8 + b] = -B[a];
  f[11] = q[11] * v[K] + W * sigma * (E[K] + vxB_K - vE * v[K]);
  f[12] = E[K];
  f[13] = B[K];
}

// ---------------------------------------------------------------------------------------
// Two-fluid model (eq 5-6; App. A P:L441-451 with readings G2, G3)
// q: D, S(3), tau, Dbar, Sbar(3), taubar, B(3), E(3), psi, phi     w: rho_e,v_e(3),p_e, rho_p,v_p(3),p_p
// ---------------------------------------------------------------------------------------
RMHD_DEV void t_prim2cons(const double* w, const double* B, const double* E, const DevPar& P, double* q) {
  double D = 0, Sx = 0, Sy = 0, Sz = 0, tau = 0, Db = 0, Sbx = 0, Sby = 0, Sbz = 0, taub = 0;
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const double* ws = w + 5 * s;
    const double mu = s == 0 ? P.mu_e : P.mu_p;
    const double W = rsqrt(1.0 - (ws[1] * ws[1] + ws[2] * ws[2] + ws[3] * ws[3]));
    const double Z = (ws[0] + P.gi * ws[4]) * W * W;
    const double Ds = ws[0] * W;
    const double ts = Z - ws[4] - Ds;
    D += Ds; tau += ts; Db += mu * Ds; taub += mu * ts;
    Sx += Z * ws[1]; Sy += Z * ws[2]; Sz += Z * ws[3];
    Sbx += mu * Z * ws[1]; Sby += mu * Z * ws[2]; Sbz += mu * Z * ws[3];
  }
  q[0] = D;
  q[1] = Sx + (E[1] * B[2] - E[2] * B[1]);
  q[2] = Sy + (E[2] * B[0] - E[0] * B[2]);
  q[3] = Sz + (E[0] * B[1] - E[1] * B[0]);
  q[4] = tau + 0.5 * (E[0] * E[0] + E[1] * E[1] + E[2] * E[2] + B[0] * B[0] + B[1] * B[1] + B[2] * B[2]);
  q[5] = Db; q[6] = Sbx; q[7] = Sby; q[8] = Sbz; q[9] = taub;
  q[10] = B[0]; q[11] = B[1]; q[12] = B[2];
  q[13] = E[0]; q[14] = E[1]; q[15] = E[2];
  q[16] = 0.0; q[17] = 0.0;
}

// species split (eq 7-8): x = x_e + x_p, xbar = mu_e x_e + mu_p x_p
struct Split {
  double ce, de, cp, dp;  // x_e = ce*xbar + de*x ; x_p = cp*xbar + dp*x
  RMHD_DEV explicit Split(const DevPar& P) {
    const double r = 1.0 / (P.mu_e - P.mu_p);
    ce = r; de = -P.mu_p * r; cp = -r; dp = P.mu_e * r;
  }
};

RMHD_DEV int t_con2prim(const double* q, const double* Zg /*2*/, const DevPar& P, Hyd* h /*2*/, int& iters) {
  const double Bx = q[10], By = q[11], Bz = q[12], Ex = q[13], Ey = q[14], Ez = q[15];
  const double Sx = q[1] - (Ey * Bz - Ez * By);
  const double Sy = q[2] - (Ez * Bx - Ex * Bz);
  const double Sz = q[3] - (Ex * By - Ey * Bx);
  const double taut = q[4] - 0.5 * (Ex * Ex + Ey * Ey + Ez * Ez + Bx * Bx + By * By + Bz * Bz);
  const Split sp(P);
  int it0, it1;
  const int r0 = c2p_hydro(sp.ce * q[5] + sp.de * q[0], sp.ce * q[6] + sp.de * Sx, sp.ce * q[7] + sp.de * Sy,
                           sp.ce * q[8] + sp.de * Sz, sp.ce * q[9] + sp.de * taut, Zg[0], P, h[0], it0);
  const int r1 = c2p_hydro(sp.cp * q[5] + sp.dp * q[0], sp.cp * q[6] + sp.dp * Sx, sp.cp * q[7] + sp.dp * Sy,
                           sp.cp * q[8] + sp.dp * Sz, sp.cp * q[9] + sp.dp * taut, Zg[1], P, h[1], it1);
  iters = it0 > it1 ? it0 : it1;
  return r0 ? r0 : r1;
}

template <int K>
RMHD_DEV void t_flux(const double* q, const double* w, const DevPar& P, double* f) {
  constexpr int a = (K + 1) % 3, b = (K + 2) % 3;
  const double* B = q + 10;
  const double* E = q + 13;
  double fD = 0, fDb = 0, ftb = 0, psum = 0, fS[3] = {0, 0, 0}, fSb[3] = {0, 0, 0};
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const double* ws = w + 5 * s;
    const double* v = ws + 1;
    const double mu = s == 0 ? P.mu_e : P.mu_p;
    const double W = rsqrt(1.0 - (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]));
    const double Z = (ws[0] + P.gi * ws[4]) * W * W;
    const double Dv = ws[0] * W * v[K];
    const double Zvk = Z * v[K];
    fD += Dv; fDb += mu * Dv; ftb += mu * (Zvk - Dv); psum += ws[4];
    const double sK = Zvk * v[K], sa = Zvk * v[a], sb = Zvk * v[b];
    fS[K] += sK; fS[a] += sa; fS[b] += sb;
    fSb[K] += mu * (sK + ws[4]); fSb[a] += mu * sa; fSb[b] += mu * sb;
  }
  const double ptot = psum + 0.5 * (E[0] * E[0] + E[1] * E[1] + E[2] * E[2] + B[0] * B[0] + B[1] * B[1] + B[2] * B[2]);
  f[0] = fD;
  f[1 + K] = fS[K] + ptot - E[K] * E[K] - B[K] * B[K];
  f[1 + a] = fS[a] - E[a] * E[K] - B[a] * B[K];
  f[1 + b] = fS[b] - E[b] * E[K] - B[b] * B[K];
  f[4] = q[1 + K] - fD;
  f[5] = fDb;
  f[6] = fSb[0]; f[7] = fSb[1]; f[8] = fSb[2];
  f[9] = ftb;
  f[10 + K] = q[17]; f[10 + a] = -E[b]; f[10 + b] = E[a];
  f[13 + K] = q[16]; f[13 + a] = B[b]; f[13 + b] = -B[a];
  f[16] = E[K];
  f[17] = B[K];
}

// Two-fluid source (A2-A3).  With D_s = rho_s W_s (so mu_s rho_s W_s = mu_s D_s):
//   Kq = sum mu_s^2 D_s (= wp^2 Wbar), rhoc = sum mu_s D_s, J = sum mu_s D_s v_s,
//   U = sum mu_s^2 D_s v_s (= wp^2 u), wp2 = sum mu_s^2 D_s / W_s, rho0 = (Kq rhoc - J.U)/wp2
//   Psi_Sbar = Kq E + U x B - eta (wp2 J - rho0 U);  Psi_taubar = U.E - eta (wp2 rhoc - rho0 Kq);
//   Psi_E = -J;  Psi_psi = rhoc - kappa psi;  Psi_phi = -kappa phi
// out: s[0..2] Sbar rows, s[3] taubar, s[4..6] E rows (psi, phi rows are done by the caller)
RMHD_DEV void t_source7(const double* De /*D_e, D_p*/, const Hyd* h, const double* B, const double* E,
                                          const DevPar& P, double* s) {
  const double me = P.mu_e * De[0], mp = P.mu_p * De[1];
  const double m2e = P.mu_e * me, m2p = P.mu_p * mp;
  const double Kq = m2e + m2p, rhoc = me + mp;
  const double Jx = me * h[0].vx + mp * h[1].vx, Jy = me * h[0].vy + mp * h[1].vy, Jz = me * h[0].vz + mp * h[1].vz;
  const double Ux = m2e * h[0].vx + m2p * h[1].vx, Uy = m2e * h[0].vy + m2p * h[1].vy, Uz = m2e * h[0].vz + m2p * h[1].vz;
  const double wp2 = m2e / h[0].W + m2p / h[1].W;
  const double rho0 = (Kq * rhoc - (Jx * Ux + Jy * Uy + Jz * Uz)) / wp2;
  s[0] = Kq * E[0] + (Uy * B[2] - Uz * B[1]) - P.eta * (wp2 * Jx - rho0 * Ux);
  s[1] = Kq * E[1] + (Uz * B[0] - Ux * B[2]) - P.eta * (wp2 * Jy - rho0 * Uy);
  s[2] = Kq * E[2] + (Ux * B[1] - Uy * B[0]) - P.eta * (wp2 * Jz - rho0 * Uz);
  s[3] = (Ux * E[0] + Uy * E[1] + Uz * E[2]) - P.eta * (wp2 * rhoc - rho0 * Kq);
  s[4] = -Jx; s[5] = -Jy; s[6] = -Jz;
}

// ---------------------------------------------------------------------------------------
// WENO3 (Shu 1997, r = 2; G7): value at the face between b and c biased to a.
//   beta0 = (c-b)^2, beta1 = (b-a)^2, alpha0 = (2/3)/(eps+beta0)^2, alpha1 = (1/3)/(eps+beta1)^2
//   u = (alpha0 (b+c)/2 + alpha1 (3b-a)/2)/(alpha0+alpha1) = b + ( d1 + w0 (d0 - d1) )/2,
//   w0 = alpha0/(alpha0+alpha1) = e1^2 / (e1^2 + e0^2/2),  e_k = eps + beta_k,  d0 = c-b, d1 = b-a
// One reciprocal per reconstruction: MUFU seed r0 (rcp.approx.ftz.f64 reads only the high word
// of its input: relative error e <= ~2^-20) + one cubic step r = r0 (1 + e + e^2), error e^3
// <= 2^-60 (the denominator is >= eps^2 = 1e-12, never denormal).  14 FP64 instructions.
//
// The FP64 pipe of sm_100 issues one warp instruction per 2 cycles per SM sub-partition but has
// ~18 cycles of dependent latency (measured: utilisation = warps x ILP x 2 / 18 in profiles/r1a),
// and ptxas emits each reconstruction as one serial chain.  weno3_batch therefore runs G
// independent reconstructions in OPERATION-MAJOR order, so G chains are in flight per warp.
// ---------------------------------------------------------------------------------------
RMHD_DEV double rcp_seed(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  return r;
}

RMHD_DEV double weno3(double a, double b, double c) {
  const double eps = 1e-6;
  const double d0 = c - b, d1 = b - a;
  const double e0 = fma(d0, d0, eps), e1 = fma(d1, d1, eps);
  const double t = e1 * e1;
  const double den = fma(0.5 * e0, e0, t);
  const double r0 = rcp_seed(den);
  const double er = fma(-den, r0, 1.0);
  const double r = fma(r0, fma(er, er, er), r0);
  return fma(0.5, fma(t * r, d0 - d1, d1), b);
}

#ifndef RMHD_WENO_GV
#define RMHD_WENO_GV 4   // variables per batch: 2 x RMHD_WENO_GV reconstructions in flight
#endif

// UNSCALED: the inputs are g+- = f +- q = 2 f+-; eps is scaled by 4 (exactly, a power of two) so the
// nonlinear weights are bit-identical to those of the scaled data and the result is exactly twice as large.
template <int G, bool UNSCALED = false>
RMHD_DEV void weno3_batch(const double* a, const double* b, const double* c, double* out) {
  const double eps = UNSCALED ? 4.0 * 1e-6 : 1e-6;
  double d0[G], d1[G], e0[G], e1[G], t[G], den[G], r0[G], er[G];
#pragma unroll
  for (int g = 0; g < G; ++g) d0[g] = c[g] - b[g];
#pragma unroll
  for (int g = 0; g < G; ++g) d1[g] = b[g] - a[g];
#pragma unroll
  for (int g = 0; g < G; ++g) e0[g] = fma(d0[g], d0[g], eps);
#pragma unroll
  for (int g = 0; g < G; ++g) e1[g] = fma(d1[g], d1[g], eps);
#pragma unroll
  for (int g = 0; g < G; ++g) t[g] = e1[g] * e1[g];
#pragma unroll
  for (int g = 0; g < G; ++g) e1[g] = 0.5 * e0[g];
#pragma unroll
  for (int g = 0; g < G; ++g) den[g] = fma(e1[g], e0[g], t[g]);
#pragma unroll
  for (int g = 0; g < G; ++g) r0[g] = rcp_seed(den[g]);
#pragma unroll
  for (int g = 0; g < G; ++g) er[g] = fma(-den[g], r0[g], 1.0);
#pragma unroll
  for (int g = 0; g < G; ++g) d0[g] = d0[g] - d1[g];
#pragma unroll
  for (int g = 0; g < G; ++g) er[g] = fma(er[g], er[g], er[g]);
#pragma unroll
  for (int g = 0; g < G; ++g) r0[g] = fma(r0[g], er[g], r0[g]);
#pragma unroll
  for (int g = 0; g < G; ++g) t[g] = t[g] * r0[g];
#pragma unroll
  for (int g = 0; g < G; ++g) d1[g] = fma(t[g], d0[g], d1[g]);
#pragma unroll
  for (int g = 0; g < G; ++g) out[g] = fma(0.5, d1[g], b[g]);
}

// face fluxes F_v = weno3(f+ at p, p+st, p+2st) + weno3(f- at m+3st, m+2st, m+st) for NV variables
// whose f+ / f- planes are vstride apart, in groups of <= 4 variables (8 chains in flight)
template <int NV>
RMHD_DEV void weno_faces(const double* pp, const double* pm, int vstride, int st, double* F) {
  constexpr int GV = NV >= RMHD_WENO_GV ? RMHD_WENO_GV : NV;
  double a[2 * GV], b[2 * GV], c[2 * GV], o[2 * GV];
#pragma unroll
  for (int v = 0; v < GV; ++v) {
    a[2 * v] = pp[v * vstride]; b[2 * v] = pp[v * vstride + st]; c[2 * v] = pp[v * vstride + 2 * st];
    a[2 * v + 1] = pm[v * vstride + 3 * st]; b[2 * v + 1] = pm[v * vstride + 2 * st]; c[2 * v + 1] = pm[v * vstride + st];
  }
  weno3_batch<2 * GV>(a, b, c, o);
#pragma unroll
  for (int v = 0; v < GV; ++v) F[v] = o[2 * v] + o[2 * v + 1];
  if constexpr (NV > GV) weno_faces<NV - GV>(pp + GV * vstride, pm + GV * vstride, vstride, st, F + GV);
}

}  // namespace rmhd

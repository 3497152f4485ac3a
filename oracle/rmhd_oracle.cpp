// =====================================================================================
// rmhd_oracle.cpp -- CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, serial-by-construction (optionally OpenMP over independent cells) FP64
// implementation of one step of the finite-volume IMEX SSP2(222) / SSP3(332) schemes for resistive
// single-fluid (14 conserved variables) and two-fluid (18) special-relativistic MHD of
// Wright & Hawke, "Resistive and multi-fluid RMHD on graphics processing units".
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load this library.  It shares NO code, header, table or helper with the CUDA
// path under paper_1808_09721_b200/csrc/ and neither includes the other.
//
// Every function cites the passage of /root/reference/PAPER.md ("P:Lnnn") it follows and,
// where the paper is silent or garbled, the reading listed in DESIGN.md ("G1".."G19").
//
// Parity pins (tests/test_oracle_*.py): con2prim round trip + closed form; species split
// inverse; WENO3 linear exactness / equal-beta reduction / order / mirror; vacuum plane
// wave (Maxwell flux signs); uniform state => L == 0; telescoping conservation; closed
// form stage solution and SSP2(222) stability function R(z); stage residual; frozen-v
// guess vs Sherman-Morrison; steady states; bitwise mirror symmetry; self-similar current
// sheet; ideal limit; two-fluid Langmuir frequency; general IMEX stepper and
// SSP3(332) (Table 3): order conditions, implicit stability function, Shu-Osher
// RK3 recomposition through eval_L, telegraph-mode closed form, Table 2 through the general
// stepper against the SSP2(222) path, second-order convergence.  tests/test_oracle_pins_r2.py:
// two-fluid source rows with friction on a charged, moving state (hand values; rho_0 of reading G2),
// Gauss-law initial charge density, zero-gradient outflow fill, the second con2prim residual alone
// and the hard tail (W up to 100, p/rho up to 1e4) -- each checked against a named mutation.
// Full configs 1,3,4,5 have no printed reference values in the paper: "parity unpinned" beyond
// those pins; no function of this file is without a pin.
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
// -ffp-contract=off: the paper itself switches FMA off; also needed for the
// bitwise mirror-symmetry pin.
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---- variable layout (eq 1; eq 5-6) --------------------------------
// resistive cons : D, Sx,Sy,Sz, tau, Bx,By,Bz, Ex,Ey,Ez, rho_charge, psi, phi        (14)
// resistive prims: rho, vx,vy,vz, p, Bx,By,Bz, Ex,Ey,Ez                              (11)
// two-fluid cons : D, S(3), tau, Dbar, Sbar(3), taubar, B(3), E(3), psi, phi         (18)
// two-fluid prims: rho_e, v_e(3), p_e, rho_p, v_p(3), p_p, B(3), E(3)                (16)
constexpr int MAXN = 18;
constexpr int MAXP = 16;

struct Par {
  int model;               // 0 resistive, 1 two-fluid
  double gam;              // Gamma-law index
  double sigma;            // conductivity (resistive)
  double eta;              // resistivity (two-fluid)
  double mu[2];            // charge/mass ratio: [0] electrons, [1] protons/positrons
  double kappa;            // cleaning rate, paper uses 1
  double tol_c2p;          // P:L124, read as relative step tolerance (G5)
  double tol_stage;        // G6
  int maxit_c2p, maxit_stage;
};

inline int ncons(int model) { return model == 0 ? 14 : 18; }
inline int nprim(int model) { return model == 0 ? 11 : 16; }

inline double dot3(const double* a, const double* b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
inline void cross3(const double* a, const double* b, double* c) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}
// Levi-Civita symbol, indices 0..2
inline double lc(int i, int j, int k) { return 0.5 * double((i - j) * (j - k) * (k - i)); }

// ---- hydrodynamic part --------------------------------------------------------------
// eq (3): W = 1/sqrt(1 - v_i v^i);  eq (4): h = 1 + Gamma p / (rho (Gamma-1))
// Z := rho h W^2 (the quantity multiplying v_i in S_i, eq 2).
inline double lorentz(const double* v) { return 1.0 / std::sqrt(1.0 - dot3(v, v)); }
inline double enthalpy_Z(double rho, double p, double W, double gam) {
  double h = 1.0 + gam * p / (rho * (gam - 1.0));
  return rho * h * W * W;
}

struct Hydro {
  double rho, v[3], p, W, Z;
};

// R1 (G4, G5): single-unknown residual in Z = rho h W^2 for the purely
// hydrodynamic conserved set (D, St_i = Z v_i, taut = Z - p - D):
//   f(Z) = Z - p(Z) - taut - D,  v^2 = St^2/Z^2,  p(Z) = (G-1)/G (Z (1-v^2) - D sqrt(1-v^2))
//   f'(Z) = 1 - (G-1)/G (1 + v^2 - D W v^2 / Z)
// Newton-Raphson safeguarded by a bracket (lo = |St| where v^2 = 1; f increasing
// for Gamma <= 2).  Stop when the applied update |dZ| <= tol * Z (G5: the paper's 1e-13
// read as a relative step tolerance; the update is applied, so the root sits at round-off).
// returns 0 ok, 1 inadmissible input, 2 not converged, 3 unphysical result
// Second residual (two alternative residuals, "one may converge where the other may not"; the paper cites
// them without printing them, G4).  Reading taken: the same recovery written in the Lorentz factor W instead of Z, which
// for the Gamma-law EOS (eq 4) is a quartic.  With E := taut + D = Z - p and p = g (Z / W^2 - D / W), g = (G-1)/G:
//   Z(W) = W (E W - g D) / (W^2 - g),
// and St^2 = Z^2 (1 - 1/W^2) gives
//   F(W) = (E W - g D)^2 (W^2 - 1) - St^2 (W^2 - g)^2 = 0   on  1 <= W <= Wmax = (1 - St^2/E^2)^(-1/2)  (p >= 0 <=> Z >= E).
// F(1) = -St^2 (1 - g)^2 <= 0; an admissible state has F(Wmax) >= 0.  Newton-Raphson from W = Wmax kept inside the
// bracket (bisection otherwise); stop when the applied update |dW| <= tol W, or when |F| has reached its round-off floor
// 32 eps ((E W - g D)^2 (W^2 - 1) + St^2 (W^2 - g)^2) (the two terms cancel to ~(E - |St|)/E where this residual is
// needed, so the update cannot shrink further).  It is the automatic fall-back of c2p_hydro
// below after g_c2p_switch iterations of the first residual: near |St| -> E (large W, hot gas) f(Z) is almost flat at the
// root while F(W) stays a well-scaled polynomial.
int g_c2p_switch = 20;   // iterations of the first residual before the second takes over (0: second residual only; test hook)

int c2p_hydro_W(double D, const double* St, double taut, double gam, double tol, int maxit, Hydro& w, int& iters) {
  const double g = (gam - 1.0) / gam;
  const double S2 = dot3(St, St);
  const double Sabs = std::sqrt(S2);
  const double E = taut + D;
  auto F = [&](double W, double& dF, double& mag) {
    const double a = E * W - g * D, b = W * W - g, c = W * W - 1.0;
    dF = 2.0 * E * a * c + 2.0 * W * a * a - 4.0 * S2 * W * b;
    mag = a * a * c + S2 * b * b;
    return a * a * c - S2 * b * b;
  };
  const double floor_eps = 32.0 * std::numeric_limits<double>::epsilon();
  double lo = 1.0, hi = 1.0 / std::sqrt((E - Sabs) * (E + Sabs) / (E * E));
  double dF, mag;
  double W = hi;
  bool conv = false;
  // Near-static state, Wmax - 1 <= 1e-9 (|St| / E below about 4e-5): W^2 - 1 is then known to a few ulps of 1 only (it
  // rounds to exactly 0 once |St| / E < 1e-8, and F(Wmax) = -St^2 (1-g)^2 would read "no root"), so the quartic cannot
  // be iterated.  Its root is taken in closed form instead: W^2 - 1 = v^2 = St^2 / Z^2 with Z = Z(W = 1) = (E - g D) / (1 - g),
  // W = sqrt(1 + v^2) = 1 + v^2 / 2; the neglected terms are O(v^4) <= 4e-18.  (Reading G4.)
  if (hi - 1.0 <= 1e-9) {
    const double Z1 = (E - g * D) / (1.0 - g);
    W = 1.0 + 0.5 * S2 / (Z1 * Z1);
    ++iters;
    conv = true;
  } else if (!std::isfinite(hi) || !(F(hi, dF, mag) >= -floor_eps * mag)) return 3;   // no root with p >= 0
  while (!conv && iters < maxit) {
    ++iters;
    const double f = F(W, dF, mag);
    if (std::fabs(f) <= floor_eps * mag) { conv = true; break; }
    if (f < 0.0) lo = std::max(lo, W); else hi = std::min(hi, W);
    double Wn = W - f / dF;
    if (!(Wn >= lo && Wn <= hi) || !std::isfinite(Wn)) Wn = 0.5 * (lo + hi);
    const double dW = Wn - W;
    W = Wn;
    if (std::fabs(dW) <= tol * W) { conv = true; break; }
  }
  const double Z = W * (E * W - g * D) / (W * W - g);
  w.Z = Z; w.W = W;
  w.p = g * (Z / (W * W) - D / W);
  w.rho = D / W;
  for (int i = 0; i < 3; ++i) w.v[i] = St[i] / Z;
  if (!conv) return 2;
  if (!(w.p > 0.0) || !(w.rho > 0.0) || !std::isfinite(w.p) || !std::isfinite(Z)) return 3;
  return 0;
}

int c2p_hydro(double D, const double* St, double taut, double gam, double Zguess, double tol, int maxit,
              Hydro& w, int& iters) {
  const double g = (gam - 1.0) / gam;
  const double S2 = dot3(St, St);
  const double Sabs = std::sqrt(S2);
  iters = 0;
  w.rho = w.p = w.W = w.Z = std::numeric_limits<double>::quiet_NaN();
  w.v[0] = w.v[1] = w.v[2] = w.rho;
  if (!(D > 0.0) || !(taut + D > Sabs) || !std::isfinite(taut) || !std::isfinite(S2)) return 1;
  double lo = Sabs, hi = std::numeric_limits<double>::infinity();
  double Z = Zguess;
  if (!(Z > Sabs) || !std::isfinite(Z)) Z = std::max(taut + D, Sabs * (1.0 + 1e-8) + 1e-300);
  bool conv = false;
  for (int it = 1; it <= maxit; ++it) {
    if (it > g_c2p_switch) return c2p_hydro_W(D, St, taut, gam, tol, maxit, w, iters);
    iters = it;
    double v2 = S2 / (Z * Z);
    double om = 1.0 - v2;
    double sq = std::sqrt(om);
    double W = 1.0 / sq;
    double p = g * (Z * om - D * sq);
    double f = Z - p - taut - D;
    double fp = 1.0 - g * (1.0 + v2 - D * W * v2 / Z);
    if (f < 0.0) lo = std::max(lo, Z); else hi = std::min(hi, Z);
    double Zn = Z - f / fp;
    if (!(Zn >= lo && Zn <= hi && Zn > Sabs) || !std::isfinite(Zn)) {
      Zn = std::isfinite(hi) ? 0.5 * (lo + hi) : 2.0 * Z;
    }
    double dZ = Zn - Z;
    Z = Zn;
    if (std::fabs(dZ) <= tol * Z) { conv = true; break; }
  }
  double v2 = S2 / (Z * Z);
  double om = 1.0 - v2;
  double sq = std::sqrt(om);
  w.Z = Z;
  w.W = 1.0 / sq;
  w.p = g * (Z * om - D * sq);
  w.rho = D * sq;  // rho = D / W
  for (int i = 0; i < 3; ++i) w.v[i] = St[i] / Z;
  if (!conv) return 2;
  if (!(w.p > 0.0) || !(w.rho > 0.0) || !std::isfinite(w.p) || !std::isfinite(w.W)) return 3;
  return 0;
}

// ---- resistive single-fluid model -------------------------------------------------------
// R0, eq (2)-(4) P:L63-71: D = rho W; S = Z v + E x B; tau = Z - p + (E^2+B^2)/2 - D.
void r_prim2cons(const double* w, double rhoc, double psi, double phi, double gam, double* q) {
  const double* v = w + 1; const double* B = w + 5; const double* E = w + 8;
  double W = lorentz(v);
  double Z = enthalpy_Z(w[0], w[4], W, gam);
  double ExB[3]; cross3(E, B, ExB);
  q[0] = w[0] * W;
  for (int i = 0; i < 3; ++i) q[1 + i] = Z * v[i] + ExB[i];
  q[4] = Z - w[4] + 0.5 * (dot3(E, E) + dot3(B, B)) - q[0];
  for (int i = 0; i < 3; ++i) { q[5 + i] = B[i]; q[8 + i] = E[i]; }
  q[11] = rhoc; q[12] = psi; q[13] = phi;
}

// R1: subtract the EM parts, then the hydro root-find.
int r_cons2prim(const double* q, const Par& P, double Zguess, double* w, double& Zout, int& iters) {
  const double* B = q + 5; const double* E = q + 8;
  double ExB[3]; cross3(E, B, ExB);
  double St[3] = {q[1] - ExB[0], q[2] - ExB[1], q[3] - ExB[2]};
  double taut = q[4] - 0.5 * (dot3(E, E) + dot3(B, B));
  Hydro h;
  int rc = c2p_hydro(q[0], St, taut, P.gam, Zguess, P.tol_c2p, P.maxit_c2p, h, iters);
  w[0] = h.rho; w[1] = h.v[0]; w[2] = h.v[1]; w[3] = h.v[2]; w[4] = h.p;
  for (int i = 0; i < 3; ++i) { w[5 + i] = B[i]; w[8 + i] = E[i]; }
  Zout = h.Z;
  return rc;
}

// P:L75 / eq (2): J_i = rhoc v_i + W sigma [E_i + eps_ijk v^j B^k - (v_k E^k) v_i]
void r_current(const double* w, double rhoc, double sigma, double* J) {
  const double* v = w + 1; const double* B = w + 5; const double* E = w + 8;
  double W = lorentz(v);
  double vxB[3]; cross3(v, B, vxB);
  double vE = dot3(v, E);
  for (int i = 0; i < 3; ++i) J[i] = rhoc * v[i] + W * sigma * (E[i] + vxB[i] - vE * v[i]);
}

// R2, eq (1)-(2) P:L57-63: flux vector along axis k.
void r_flux(const double* q, const double* w, int k, double sigma, double gam, double* f) {
  const double* v = w + 1; const double* B = w + 5; const double* E = w + 8;
  double W = lorentz(v);
  double Z = enthalpy_Z(w[0], w[4], W, gam);
  double ptot = w[4] + 0.5 * (dot3(E, E) + dot3(B, B));
  double J[3]; r_current(w, q[11], sigma, J);
  f[0] = q[0] * v[k];                                            // D v^k
  for (int i = 0; i < 3; ++i)                                    // S_i^k  (eq 2, S_ij)
    f[1 + i] = Z * v[i] * v[k] + (i == k ? ptot : 0.0) - E[i] * E[k] - B[i] * B[k];
  f[4] = q[1 + k] - q[0] * v[k];                                 // S^k - D v^k
  for (int i = 0; i < 3; ++i) {                                  // -eps^{ijk} E_j + delta_i^k phi
    double s = 0.0;
    for (int j = 0; j < 3; ++j) s -= lc(i, j, k) * E[j];
    f[5 + i] = s + (i == k ? q[13] : 0.0);
  }
  for (int i = 0; i < 3; ++i) {                                  // +eps^{ijk} B_j + delta_i^k psi
    double s = 0.0;
    for (int j = 0; j < 3; ++j) s += lc(i, j, k) * B[j];
    f[8 + i] = s + (i == k ? q[12] : 0.0);
  }
  f[11] = J[k];                                                  // J^k
  f[12] = E[k];                                                  // E^k
  f[13] = B[k];                                                  // B^k
}

// R3, eq (1) P:L57 right-hand side.
void r_source(const double* q, const double* w, double sigma, double kappa, double* s) {
  for (int i = 0; i < 14; ++i) s[i] = 0.0;
  double J[3]; r_current(w, q[11], sigma, J);
  for (int i = 0; i < 3; ++i) s[8 + i] = -J[i];
  s[12] = q[11] - kappa * q[12];
  s[13] = -kappa * q[13];
}

// ---- two-fluid model ------------------------------------------------------------------
// TF0, eq (6) P:L95-108 with reading G2 (Sbar carries h_s): sums over s in {e,p}.
void t_prim2cons(const double* w, double psi, double phi, const Par& P, double* q) {
  const double* B = w + 10; const double* E = w + 13;
  double ExB[3]; cross3(E, B, ExB);
  for (int i = 0; i < 18; ++i) q[i] = 0.0;
  for (int s = 0; s < 2; ++s) {
    const double* ws = w + 5 * s;
    const double* v = ws + 1;
    double W = lorentz(v);
    double Z = enthalpy_Z(ws[0], ws[4], W, P.gam);
    double Ds = ws[0] * W;
    q[0] += Ds;
    q[4] += Z - ws[4] - Ds;
    q[5] += P.mu[s] * Ds;
    q[9] += P.mu[s] * (Z - ws[4] - Ds);
    for (int i = 0; i < 3; ++i) { q[1 + i] += Z * v[i]; q[6 + i] += P.mu[s] * Z * v[i]; }
  }
  for (int i = 0; i < 3; ++i) q[1 + i] += ExB[i];
  q[4] += 0.5 * (dot3(E, E) + dot3(B, B));
  for (int i = 0; i < 3; ++i) { q[10 + i] = B[i]; q[13 + i] = E[i]; }
  q[16] = psi; q[17] = phi;
}

// eq (7) P:L128 (and (8) P:L133 with reading G3): invert x = x_e + x_p, xbar = mu_e x_e + mu_p x_p.
inline void species_split(double x, double xbar, const double* mu, double* xe, double* xp) {
  *xe = (xbar - mu[1] * x) / (mu[0] - mu[1]);
  *xp = (xbar - mu[0] * x) / (mu[1] - mu[0]);
}

// TF1.
int t_cons2prim(const double* q, const Par& P, const double* Zguess, double* w, double* Zout, int& iters) {
  const double* B = q + 10; const double* E = q + 13;
  double ExB[3]; cross3(E, B, ExB);
  double St[3] = {q[1] - ExB[0], q[2] - ExB[1], q[3] - ExB[2]};   // G3: unbarred S
  double taut = q[4] - 0.5 * (dot3(E, E) + dot3(B, B));
  double Ds[2], Ss[2][3], ts[2];
  species_split(q[0], q[5], P.mu, &Ds[0], &Ds[1]);
  for (int i = 0; i < 3; ++i) species_split(St[i], q[6 + i], P.mu, &Ss[0][i], &Ss[1][i]);
  species_split(taut, q[9], P.mu, &ts[0], &ts[1]);
  int rc = 0; iters = 0;
  for (int s = 0; s < 2; ++s) {
    Hydro h; int it;
    int r = c2p_hydro(Ds[s], Ss[s], ts[s], P.gam, Zguess ? Zguess[s] : -1.0, P.tol_c2p, P.maxit_c2p, h, it);
    if (r && !rc) rc = r;
    iters = std::max(iters, it);
    double* ws = w + 5 * s;
    ws[0] = h.rho; ws[1] = h.v[0]; ws[2] = h.v[1]; ws[3] = h.v[2]; ws[4] = h.p;
    Zout[s] = h.Z;
  }
  for (int i = 0; i < 3; ++i) { w[10 + i] = B[i]; w[13 + i] = E[i]; }
  return rc;
}

// (A3) P:L451 with reading G2: plasma-frame quantities.
struct TFaux {
  double wp2, rhoc, J[3], Wbar, u[3], rho0;
};
void t_aux(const double* w, const Par& P, TFaux& a) {
  a.wp2 = 0.0; a.rhoc = 0.0; a.Wbar = 0.0;
  for (int i = 0; i < 3; ++i) { a.J[i] = 0.0; a.u[i] = 0.0; }
  for (int s = 0; s < 2; ++s) {
    const double* ws = w + 5 * s; const double* v = ws + 1;
    double W = lorentz(v);
    double m = P.mu[s];
    a.wp2 += m * m * ws[0];                    // omega_p^2 = mu_s^2 rho_s
    a.rhoc += m * ws[0] * W;                   // charge density
    a.Wbar += m * m * ws[0] * W;
    for (int i = 0; i < 3; ++i) { a.J[i] += m * ws[0] * W * v[i]; a.u[i] += m * m * ws[0] * W * v[i]; }
  }
  a.Wbar /= a.wp2;
  for (int i = 0; i < 3; ++i) a.u[i] /= a.wp2;
  a.rho0 = a.Wbar * a.rhoc - dot3(a.J, a.u);
}

// TF2, (A1) P:L443 with reading G2.
void t_flux(const double* q, const double* w, int k, const Par& P, double* f) {
  const double* B = w + 10; const double* E = w + 13;
  for (int i = 0; i < 18; ++i) f[i] = 0.0;
  double psum = 0.0, Dv = 0.0;
  for (int s = 0; s < 2; ++s) {
    const double* ws = w + 5 * s; const double* v = ws + 1;
    double W = lorentz(v);
    double Z = enthalpy_Z(ws[0], ws[4], W, P.gam);
    double Ds = ws[0] * W;
    double m = P.mu[s];
    f[0] += Ds * v[k];
    Dv += Ds * v[k];
    psum += ws[4];
    f[5] += m * Ds * v[k];
    f[9] += m * (Z - Ds) * v[k];                         // (taubar_s + mu_s p_s) v_s^k
    for (int i = 0; i < 3; ++i) {
      f[1 + i] += Z * v[i] * v[k];
      f[6 + i] += m * (Z * v[i] * v[k] + (i == k ? ws[4] : 0.0));
    }
  }
  double ptot = psum + 0.5 * (dot3(E, E) + dot3(B, B));
  for (int i = 0; i < 3; ++i) f[1 + i] += (i == k ? ptot : 0.0) - E[i] * E[k] - B[i] * B[k];
  f[4] = q[1 + k] - Dv;
  for (int i = 0; i < 3; ++i) {
    double sB = 0.0, sE = 0.0;
    for (int j = 0; j < 3; ++j) { sB -= lc(i, j, k) * E[j]; sE += lc(i, j, k) * B[j]; }
    f[10 + i] = sB + (i == k ? q[17] : 0.0);
    f[13 + i] = sE + (i == k ? q[16] : 0.0);
  }
  f[16] = E[k];
  f[17] = B[k];
}

// TF3, (A2) P:L445 with reading G2 (rho0 in the spatial friction term).
void t_source(const double* q, const double* w, const Par& P, double* s) {
  const double* B = w + 10; const double* E = w + 13;
  for (int i = 0; i < 18; ++i) s[i] = 0.0;
  TFaux a; t_aux(w, P, a);
  double uxB[3]; cross3(a.u, B, uxB);
  for (int i = 0; i < 3; ++i)
    s[6 + i] = a.wp2 * (a.Wbar * E[i] + uxB[i] - P.eta * (a.J[i] - a.rho0 * a.u[i]));
  s[9] = a.wp2 * (dot3(a.u, E) - P.eta * (a.rhoc - a.rho0 * a.Wbar));
  for (int i = 0; i < 3; ++i) s[13 + i] = -a.J[i];
  s[16] = a.rhoc - P.kappa * q[16];
  s[17] = -P.kappa * q[17];
}

// ---- model dispatch ---------------------------------------------------------------------
struct CellState {  // guesses carried between con2prim calls
  double Z[2];
};
int cons2prim(const double* q, const Par& P, const double* Zg, double* w, double* Zout, int& iters) {
  if (P.model == 0) return r_cons2prim(q, P, Zg ? Zg[0] : -1.0, w, Zout[0], iters);
  return t_cons2prim(q, P, Zg, w, Zout, iters);
}
void flux_vector(const double* q, const double* w, int k, const Par& P, double* f) {
  if (P.model == 0) r_flux(q, w, k, P.sigma, P.gam, f); else t_flux(q, w, k, P, f);
}
void source_vector(const double* q, const double* w, const Par& P, double* s) {
  if (P.model == 0) r_source(q, w, P.sigma, P.kappa, s); else t_source(q, w, P, s);
}
void guess_Z(const double* w, const Par& P, double* Zg) {
  int ns = P.model == 0 ? 1 : 2;
  for (int s = 0; s < ns; ++s) {
    const double* ws = w + 5 * s;
    Zg[s] = enthalpy_Z(ws[0], ws[4], lorentz(ws + 1), P.gam);
  }
}

// ---- dense linear algebra: LU with partial pivoting ---------------------------------------
bool lu_solve(int n, double* A /*n*n row-major, destroyed*/, double* b /*in: rhs, out: x*/) {
  for (int c = 0; c < n; ++c) {
    int piv = c; double best = std::fabs(A[c * n + c]);
    for (int r = c + 1; r < n; ++r) { double t = std::fabs(A[r * n + c]); if (t > best) { best = t; piv = r; } }
    if (!(best > 0.0) || !std::isfinite(best)) return false;
    if (piv != c) { for (int j = 0; j < n; ++j) std::swap(A[c * n + j], A[piv * n + j]); std::swap(b[c], b[piv]); }
    for (int r = c + 1; r < n; ++r) {
      double m = A[r * n + c] / A[c * n + c];
      if (m != 0.0) { for (int j = c; j < n; ++j) A[r * n + j] -= m * A[c * n + j]; b[r] -= m * b[c]; }
    }
  }
  for (int r = n - 1; r >= 0; --r) {
    double s = b[r];
    for (int j = r + 1; j < n; ++j) s -= A[r * n + j] * b[j];
    b[r] = s / A[r * n + r];
  }
  return true;
}

// ---- implicit stage (eq 10) ----------------------------------------------
// I.3: frozen-(v,W) guess for E*: the stage equation E - E_ex + a J(E) = 0 is
// linear in E when v, W are held: M E = b, M = (1+s) I - s v v^T, s = a W sigma,
// b = E_ex - a rhoc v - s (v x B).  Solved here by plain Gaussian elimination.
void r_stage_guess_E(const double* q_ex, const double* wg, double a, double sigma, double* Eg) {
  const double* v = wg + 1; const double* B = q_ex + 5;
  double W = lorentz(v);
  double s = a * W * sigma;
  double vxB[3]; cross3(v, B, vxB);
  double M[9], b[3];
  for (int i = 0; i < 3; ++i) {
    for (int j = 0; j < 3; ++j) M[3 * i + j] = (i == j ? 1.0 + s : 0.0) - s * v[i] * v[j];
    b[i] = q_ex[8 + i] - a * q_ex[11] * v[i] - s * vxB[i];
  }
  if (!lu_solve(3, M, b)) { for (int i = 0; i < 3; ++i) b[i] = q_ex[8 + i]; }
  for (int i = 0; i < 3; ++i) Eg[i] = b[i];
}

// residual of eq (10): R(q*) = q* - q_ex - a Psi(q*), Psi via con2prim(q*)
int stage_residual(const double* q, const double* q_ex, double a, const Par& P, const double* Zg,
                   double* R, double* w, double* Zout, int& c2p_it) {
  int n = ncons(P.model);
  int rc = cons2prim(q, P, Zg, w, Zout, c2p_it);
  if (rc) return rc;
  double s[MAXN];
  source_vector(q, w, P, s);
  for (int i = 0; i < n; ++i) R[i] = q[i] - q_ex[i] - a * s[i];
  return 0;
}

inline double norm2(int n, const double* x) { double s = 0.0; for (int i = 0; i < n; ++i) s += x[i] * x[i]; return std::sqrt(s); }
inline double norminf(int n, const double* x) { double s = 0.0; for (int i = 0; i < n; ++i) s = std::max(s, std::fabs(x[i])); return s; }

// I.4: N-dimensional root-find on all components of q* (the paper's formulation, P:L182:
// "a root-finding procedure of the same dimensionality as the conserved vector").  The
// paper uses CMINPACK hybrd (Powell hybrid with a finite-difference Jacobian); any
// convergent method reaches the same root, so this is Newton with a central-difference
// Jacobian (h_j = eps^(1/3) max(|q_j|,1); central so that mirror-image cells see
// mirror-image Jacobians bitwise), LU with partial pivoting and a backtracking line search
// on ||R||_2.  Stop (G6): Newton update ||dq||_inf <= tol_stage max(1, ||q||_inf); that
// update is still applied, so the root sits at round-off.  (A residual-norm test is not
// used: for stiff cells the E rows carry round-off of size eps*a*W*sigma*|E|.)
// returns 0 ok, >0 failure; iters = Newton iterations taken
int stage_solve(const double* q_ex, const double* wguess, double a, const Par& P,
                double* q, double* w, int& iters, int& c2p_max) {
  const int n = ncons(P.model);
  double Zg[2] = {-1.0, -1.0};
  guess_Z(wguess, P, Zg);
  for (int i = 0; i < n; ++i) q[i] = q_ex[i];
  if (P.model == 0) {
    double Eg[3]; r_stage_guess_E(q_ex, wguess, a, P.sigma, Eg);
    for (int i = 0; i < 3; ++i) q[8 + i] = Eg[i];
  }
  double R[MAXN], Zc[2], Rt[MAXN], wt[MAXP], Zt[2];
  int it_c2p;
  iters = 0; c2p_max = 0;
  int rc = stage_residual(q, q_ex, a, P, Zg, R, w, Zc, it_c2p);
  c2p_max = std::max(c2p_max, it_c2p);
  if (rc && P.model == 0) {  // frozen-v guess inadmissible: fall back to q_ex
    for (int i = 0; i < n; ++i) q[i] = q_ex[i];
    rc = stage_residual(q, q_ex, a, P, Zg, R, w, Zc, it_c2p);
  }
  if (rc) return 10 + rc;
  const double hrel = std::cbrt(std::numeric_limits<double>::epsilon());
  for (int it = 1; it <= P.maxit_stage; ++it) {
    iters = it;
    // central-difference Jacobian  J[i][j] = dR_i/dq_j
    double Jm[MAXN * MAXN], qp[MAXN], Rp[MAXN], Rm[MAXN], wtmp[MAXP], Ztmp[2];
    for (int j = 0; j < n; ++j) {
      double h = hrel * std::max(std::fabs(q[j]), 1.0);
      for (int i = 0; i < n; ++i) qp[i] = q[i];
      qp[j] = q[j] + h;
      int r1 = stage_residual(qp, q_ex, a, P, Zc, Rp, wtmp, Ztmp, it_c2p);
      qp[j] = q[j] - h;
      int r2 = stage_residual(qp, q_ex, a, P, Zc, Rm, wtmp, Ztmp, it_c2p);
      if (r1 || r2) return 20;
      for (int i = 0; i < n; ++i) Jm[i * n + j] = (Rp[i] - Rm[i]) / (2.0 * h);
    }
    double dq[MAXN];
    for (int i = 0; i < n; ++i) dq[i] = -R[i];
    if (!lu_solve(n, Jm, dq)) return 21;
    // G6: converged when the Newton update is below tol_stage (relative, inf-norm); the
    // update is still applied, so the returned root sits at round-off.
    const bool small = norminf(n, dq) <= P.tol_stage * std::max(1.0, norminf(n, q));
    // backtracking line search on ||R||_2 (a below-tolerance update is taken as is)
    const double r0 = norm2(n, R);
    double lam = 1.0; bool accepted = false;
    double qt[MAXN];
    for (int ls = 0; ls < 30; ++ls) {
      for (int i = 0; i < n; ++i) qt[i] = q[i] + lam * dq[i];
      int r = stage_residual(qt, q_ex, a, P, Zc, Rt, wt, Zt, it_c2p);
      if (!r) {
        c2p_max = std::max(c2p_max, it_c2p);
        if (small || norm2(n, Rt) <= r0) { accepted = true; break; }
      }
      if (small) break;
      lam *= 0.5;
    }
    if (!accepted) return 22;
    for (int i = 0; i < n; ++i) { q[i] = qt[i]; R[i] = Rt[i]; }
    for (int i = 0; i < nprim(P.model); ++i) w[i] = wt[i];
    Zc[0] = Zt[0]; Zc[1] = Zt[1];
    if (small) return 0;
  }
  return 23;
}

// ---- WENO3 (Shu 1997, r = 2; G7) -----------------------------------------------------------
// value at the face between b and c, biased toward a: stencils {b,c} and {a,b}
inline double weno3(double a, double b, double c) {
  const double eps = 1e-6;
  double beta0 = (c - b) * (c - b);
  double beta1 = (b - a) * (b - a);
  double a0 = (2.0 / 3.0) / ((eps + beta0) * (eps + beta0));
  double a1 = (1.0 / 3.0) / ((eps + beta1) * (eps + beta1));
  return (a0 * (0.5 * (b + c)) + a1 * (0.5 * (3.0 * b - a))) / (a0 + a1);
}

// ---- grid --------------------------------------------------------------------------------
struct Sim {
  Par P;
  int n[3];        // interior cells
  int ng;          // ghost layers on present axes
  int g[3];        // ghosts per axis (0 if axis absent)
  int N[3];        // total cells per axis
  double lo[3], hi[3], dx[3];
  int bc[3];
  double cfl, dt, t0;
  int integrator;
  long long nstep;
  size_t ntot;
  int nc, np;
  std::vector<double> q, w;            // [var][k][j][i]
  std::vector<double> q1, w1, L1, L2, Ps1, Ps2, qs;
  // stats
  std::vector<long long> hist_stage, hist_c2p;
  long long n_failed, first_failed;
  size_t idx(int i, int j, int k) const { return (size_t(k) * N[1] + j) * N[0] + i; }
};

// a6 / G11: outflow = copy nearest interior cell; periodic = wrap.  Axis by axis.
void fill_ghosts(const Sim& S, std::vector<double>& arr, int nvar) {
  for (int d = 0; d < 3; ++d) {
    if (S.g[d] == 0) continue;
    for (int var = 0; var < nvar; ++var) {
      double* a = arr.data() + size_t(var) * S.ntot;
      for (int k = 0; k < S.N[2]; ++k)
        for (int j = 0; j < S.N[1]; ++j)
          for (int i = 0; i < S.N[0]; ++i) {
            int c[3] = {i, j, k};
            int m = c[d] - S.g[d];
            if (m >= 0 && m < S.n[d]) continue;
            int src = m;
            if (S.bc[d] == 1) src = ((m % S.n[d]) + S.n[d]) % S.n[d];
            else src = m < 0 ? 0 : S.n[d] - 1;
            int s[3] = {i, j, k};
            s[d] = src + S.g[d];
            a[S.idx(i, j, k)] = a[S.idx(s[0], s[1], s[2])];
          }
    }
  }
}

// R4 (eq 12): L(q) = -sum_d dF^d/dx_d on interior cells, Lax-Friedrichs
// flux-vector splitting with alpha = 1 and WENO3 of f+ (left-biased) and f- (right-biased).
void eval_L(const Sim& S, const std::vector<double>& q, const std::vector<double>& w, std::vector<double>& L) {
  const int nc = S.nc, np = S.np;
  std::fill(L.begin(), L.end(), 0.0);
  for (int d = 0; d < 3; ++d) {
    if (S.g[d] == 0) continue;
    const int len = S.N[d];
    // lines along axis d
    int o1 = (d + 1) % 3, o2 = (d + 2) % 3;
    const int n1 = S.n[o1], n2 = S.n[o2];
#pragma omp parallel for collapse(2) schedule(static)
    for (int b2 = 0; b2 < n2; ++b2)
      for (int b1 = 0; b1 < n1; ++b1) {
        std::vector<double> fp(size_t(len) * nc), fm(size_t(len) * nc), F(size_t(len + 1) * nc);
        double qc[MAXN], wc[MAXP], f[MAXN];
        int c[3];
        c[o1] = b1 + S.g[o1]; c[o2] = b2 + S.g[o2];
        for (int m = 0; m < len; ++m) {
          c[d] = m;
          size_t id = S.idx(c[0], c[1], c[2]);
          for (int v = 0; v < nc; ++v) qc[v] = q[size_t(v) * S.ntot + id];
          for (int v = 0; v < np; ++v) wc[v] = w[size_t(v) * S.ntot + id];
          flux_vector(qc, wc, d, S.P, f);
          for (int v = 0; v < nc; ++v) {           // eq (12), alpha = 1
            fp[size_t(m) * nc + v] = 0.5 * (f[v] + qc[v]);
            fm[size_t(m) * nc + v] = 0.5 * (f[v] - qc[v]);
          }
        }
        // face m+1/2 for m = g-1 .. g+n-1
        for (int m = S.g[d] - 1; m < S.g[d] + S.n[d]; ++m)
          for (int v = 0; v < nc; ++v) {
            double fl = weno3(fp[size_t(m - 1) * nc + v], fp[size_t(m) * nc + v], fp[size_t(m + 1) * nc + v]);
            double fr = weno3(fm[size_t(m + 2) * nc + v], fm[size_t(m + 1) * nc + v], fm[size_t(m) * nc + v]);
            F[size_t(m + 1) * nc + v] = fl + fr;   // F_{m+1/2} stored at m+1
          }
        for (int m = S.g[d]; m < S.g[d] + S.n[d]; ++m) {
          c[d] = m;
          size_t id = S.idx(c[0], c[1], c[2]);
          for (int v = 0; v < nc; ++v)
            L[size_t(v) * S.ntot + id] -= (F[size_t(m + 1) * nc + v] - F[size_t(m) * nc + v]) / S.dx[d];
        }
      }
  }
}

void gather(const Sim& S, const std::vector<double>& a, int nvar, size_t id, double* out) {
  for (int v = 0; v < nvar; ++v) out[v] = a[size_t(v) * S.ntot + id];
}
void scatter(const Sim& S, std::vector<double>& a, int nvar, size_t id, const double* in) {
  for (int v = 0; v < nvar; ++v) a[size_t(v) * S.ntot + id] = in[v];
}

void record(Sim& S, std::vector<long long>& hist, int it) {
  int b = std::min<int>(it, int(hist.size()) - 1);
#pragma omp atomic
  hist[b]++;
}
void record_fail(Sim& S, long long cell) {
#pragma omp critical
  {
    S.n_failed++;
    if (S.first_failed < 0 || cell < S.first_failed) S.first_failed = cell;
  }
}

// T: one SSP2(222) step, Table 2, eq (10)-(11) P:L152-155 read as G1.
void step_once(Sim& S) {
  const double gam_rk = 1.0 - 1.0 / std::sqrt(2.0);
  const double dt = S.dt;
  const int nc = S.nc, np = S.np;
  const int nx = S.n[0], ny = S.n[1], nz = S.n[2];
  // --- S1: q1 = qn + gamma dt Psi(q1)
#pragma omp parallel for collapse(2) schedule(dynamic, 4)
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        size_t id = S.idx(i + S.g[0], j + S.g[1], k + S.g[2]);
        long long cell = (long long)(k) * ny * nx + (long long)(j) * nx + i;
        double qn[MAXN], wg[MAXP], qs[MAXN], ws[MAXP], ps[MAXN];
        gather(S, S.q, nc, id, qn); gather(S, S.w, np, id, wg);
        int it, c2;
        int rc = stage_solve(qn, wg, gam_rk * dt, S.P, qs, ws, it, c2);
        if (rc) record_fail(S, cell);
        record(S, S.hist_stage, it); record(S, S.hist_c2p, c2);
        source_vector(qs, ws, S.P, ps);
        scatter(S, S.q1, nc, id, qs); scatter(S, S.w1, np, id, ws); scatter(S, S.Ps1, nc, id, ps);
      }
  fill_ghosts(S, S.q1, nc); fill_ghosts(S, S.w1, np);
  // --- F1
  eval_L(S, S.q1, S.w1, S.L1);
  // --- S2: q2 = qn + dt L1 + (1-2 gamma) dt Psi(q1) + gamma dt Psi(q2)
#pragma omp parallel for collapse(2) schedule(dynamic, 4)
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        size_t id = S.idx(i + S.g[0], j + S.g[1], k + S.g[2]);
        long long cell = (long long)(k) * ny * nx + (long long)(j) * nx + i;
        double qn[MAXN], l1[MAXN], p1[MAXN], wg[MAXP], qe[MAXN], qs[MAXN], ws[MAXP], ps[MAXN];
        gather(S, S.q, nc, id, qn); gather(S, S.L1, nc, id, l1); gather(S, S.Ps1, nc, id, p1);
        gather(S, S.w1, np, id, wg);
        for (int v = 0; v < nc; ++v) qe[v] = qn[v] + dt * l1[v] + (1.0 - 2.0 * gam_rk) * dt * p1[v];
        int it, c2;
        int rc = stage_solve(qe, wg, gam_rk * dt, S.P, qs, ws, it, c2);
        if (rc) record_fail(S, cell);
        record(S, S.hist_stage, it); record(S, S.hist_c2p, c2);
        source_vector(qs, ws, S.P, ps);
        scatter(S, S.qs, nc, id, qs); scatter(S, S.w, np, id, ws); scatter(S, S.Ps2, nc, id, ps);
      }
  fill_ghosts(S, S.qs, nc); fill_ghosts(S, S.w, np);
  // --- F2
  eval_L(S, S.qs, S.w, S.L2);
  // --- C + P: q^{n+1} = qn + dt/2 (L1+L2) + dt/2 (Psi1+Psi2);  w^{n+1} = con2prim(q^{n+1})
#pragma omp parallel for collapse(2) schedule(dynamic, 4)
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        size_t id = S.idx(i + S.g[0], j + S.g[1], k + S.g[2]);
        long long cell = (long long)(k) * ny * nx + (long long)(j) * nx + i;
        double qn[MAXN], wg[MAXP], ws[MAXP], Zg[2], Zo[2];
        gather(S, S.q, nc, id, qn); gather(S, S.w, np, id, wg);
        for (int v = 0; v < nc; ++v) {
          size_t o = size_t(v) * S.ntot + id;
          qn[v] = qn[v] + 0.5 * dt * (S.L1[o] + S.L2[o]) + 0.5 * dt * (S.Ps1[o] + S.Ps2[o]);
        }
        guess_Z(wg, S.P, Zg);
        int it;
        int rc = cons2prim(qn, S.P, Zg, ws, Zo, it);
        if (rc) record_fail(S, cell);
        record(S, S.hist_c2p, it);
        scatter(S, S.q, nc, id, qn); scatter(S, S.w, np, id, ws);
      }
  fill_ghosts(S, S.q, nc); fill_ghosts(S, S.w, np);
  S.nstep++;
}

// T': one step of a general IMEX Runge-Kutta scheme written exactly as eq (10)-(11) P:L152-155 (read as G1):
//   q^(i)   = qn + dt sum_{j<i} at[i][j] L(q^(j)) + dt sum_{j<=i} a[i][j] Psi(q^(j)),   i = 1..nu
//   q^{n+1} = qn + dt sum_j wt[j] L(q^(j)) + dt sum_j w[j] Psi(q^(j))
// Stage i is the implicit solve q^(i) = q_ex + a[i][i] dt Psi(q^(i)) with q_ex the already known part.
// Used for SSP3(332), Table 3 P:L174-180 (G13: the row that lost its entries is c~ = 1, a~_21 = 1), and, as a
// cross-check of this routine against step_once, for SSP2(222), Table 2.
struct Tableau {
  int nu;
  double at[3][3], wt[3];   // explicit (tilde) part
  double a[3][3], w[3];     // implicit part
};

Tableau tableau_ssp2_222() {
  const double g = 1.0 - 1.0 / std::sqrt(2.0);
  Tableau T{};
  T.nu = 2;
  T.at[1][0] = 1.0; T.wt[0] = 0.5; T.wt[1] = 0.5;
  T.a[0][0] = g; T.a[1][0] = 1.0 - 2.0 * g; T.a[1][1] = g; T.w[0] = 0.5; T.w[1] = 0.5;
  return T;
}

Tableau tableau_ssp3_332() {
  const double g = 1.0 - 1.0 / std::sqrt(2.0);
  Tableau T{};
  T.nu = 3;
  T.at[1][0] = 1.0; T.at[2][0] = 0.25; T.at[2][1] = 0.25;
  T.wt[0] = 1.0 / 6.0; T.wt[1] = 1.0 / 6.0; T.wt[2] = 2.0 / 3.0;
  T.a[0][0] = g;
  T.a[1][0] = 1.0 - 2.0 * g; T.a[1][1] = g;
  T.a[2][0] = 0.5 - g; T.a[2][1] = 0.0; T.a[2][2] = g;
  T.w[0] = 1.0 / 6.0; T.w[1] = 1.0 / 6.0; T.w[2] = 2.0 / 3.0;
  return T;
}

void step_imex(Sim& S, const Tableau& T) {
  const double dt = S.dt;
  const int nc = S.nc, np = S.np;
  const int nx = S.n[0], ny = S.n[1], nz = S.n[2];
  const size_t a = S.ntot * nc;
  std::vector<std::vector<double>> Ls(T.nu, std::vector<double>(a, 0.0)), Ps(T.nu, std::vector<double>(a, 0.0));
  std::vector<double> wprev = S.w;           // Newton guess of stage i: primitives of stage i-1 (stage 1: w^n)
  for (int st = 0; st < T.nu; ++st) {
#pragma omp parallel for collapse(2) schedule(dynamic, 4)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          size_t id = S.idx(i + S.g[0], j + S.g[1], k + S.g[2]);
          long long cell = (long long)(k) * ny * nx + (long long)(j) * nx + i;
          double qe[MAXN], wg[MAXP], qs[MAXN], ws[MAXP], ps[MAXN];
          gather(S, S.q, nc, id, qe); gather(S, wprev, np, id, wg);
          for (int v = 0; v < nc; ++v) {
            size_t o = size_t(v) * S.ntot + id;
            for (int jj = 0; jj < st; ++jj) qe[v] = qe[v] + dt * T.at[st][jj] * Ls[jj][o] + dt * T.a[st][jj] * Ps[jj][o];
          }
          int it, c2;
          int rc = stage_solve(qe, wg, T.a[st][st] * dt, S.P, qs, ws, it, c2);
          if (rc) record_fail(S, cell);
          record(S, S.hist_stage, it); record(S, S.hist_c2p, c2);
          source_vector(qs, ws, S.P, ps);
          scatter(S, S.qs, nc, id, qs); scatter(S, S.w1, np, id, ws); scatter(S, Ps[st], nc, id, ps);
        }
    fill_ghosts(S, S.qs, nc); fill_ghosts(S, S.w1, np);
    eval_L(S, S.qs, S.w1, Ls[st]);
    wprev = S.w1;
  }
#pragma omp parallel for collapse(2) schedule(dynamic, 4)
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        size_t id = S.idx(i + S.g[0], j + S.g[1], k + S.g[2]);
        long long cell = (long long)(k) * ny * nx + (long long)(j) * nx + i;
        double qn[MAXN], wg[MAXP], ws[MAXP], Zg[2], Zo[2];
        gather(S, S.q, nc, id, qn); gather(S, wprev, np, id, wg);
        for (int v = 0; v < nc; ++v) {
          size_t o = size_t(v) * S.ntot + id;
          for (int jj = 0; jj < T.nu; ++jj) qn[v] = qn[v] + dt * T.wt[jj] * Ls[jj][o] + dt * T.w[jj] * Ps[jj][o];
        }
        guess_Z(wg, S.P, Zg);
        int it;
        int rc = cons2prim(qn, S.P, Zg, ws, Zo, it);
        if (rc) record_fail(S, cell);
        record(S, S.hist_c2p, it);
        scatter(S, S.q, nc, id, qn); scatter(S, S.w, np, id, ws);
      }
  fill_ghosts(S, S.q, nc); fill_ghosts(S, S.w, np);
  S.nstep++;
}

}  // namespace

// =====================================================================================
// C entry points (all arrays variable-major SoA: a[var][cell]; grids a[var][k][j][i])
// =====================================================================================
extern "C" {

typedef struct {
  int model;
  int nx, ny, nz;
  int ng;
  double xmin, xmax, ymin, ymax, zmin, zmax;
  int bc[3];
  double gamma, sigma, eta, mu_e, mu_p, kappa, cfl, tol_c2p, tol_stage;
  int max_iter_c2p, max_iter_stage;
  int integrator;   // 0: SSP2(222) (step_once), 1: SSP3(332) (step_imex), 2: SSP2(222) through step_imex (cross-check)
} oracle_params;

static Par to_par(const oracle_params* p) {
  Par P;
  P.model = p->model; P.gam = p->gamma; P.sigma = p->sigma; P.eta = p->eta;
  P.mu[0] = p->mu_e; P.mu[1] = p->mu_p; P.kappa = p->kappa;
  P.tol_c2p = p->tol_c2p > 0 ? p->tol_c2p : 1e-13;
  P.tol_stage = p->tol_stage > 0 ? p->tol_stage : 1e-12;
  P.maxit_c2p = p->max_iter_c2p > 0 ? p->max_iter_c2p : 100;
  P.maxit_stage = p->max_iter_stage > 0 ? p->max_iter_stage : 50;
  return P;
}

int oracle_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
  return omp_get_max_threads();
#else
  (void)n; return 1;
#endif
}

// ---- batched per-cell operations (n independent cells) ----------------------------------
int oracle_prim2cons_batch(const oracle_params* p, long long n, const double* prims, const double* rho_charge,
                           double* cons) {
  Par P = to_par(p); int nc = ncons(P.model), np = nprim(P.model);
#pragma omp parallel for schedule(static)
  for (long long c = 0; c < n; ++c) {
    double w[MAXP], q[MAXN];
    for (int v = 0; v < np; ++v) w[v] = prims[v * n + c];
    if (P.model == 0) r_prim2cons(w, rho_charge ? rho_charge[c] : 0.0, 0.0, 0.0, P.gam, q);
    else t_prim2cons(w, 0.0, 0.0, P, q);
    for (int v = 0; v < nc; ++v) cons[v * n + c] = q[v];
  }
  return 0;
}

int oracle_con2prim_batch(const oracle_params* p, long long n, const double* cons, const double* prim_guess,
                          double* prims, int* iters, int* fail) {
  Par P = to_par(p); int nc = ncons(P.model), np = nprim(P.model);
#pragma omp parallel for schedule(static)
  for (long long c = 0; c < n; ++c) {
    double w[MAXP], wg[MAXP], q[MAXN], Zg[2] = {-1.0, -1.0}, Zo[2];
    for (int v = 0; v < nc; ++v) q[v] = cons[v * n + c];
    if (prim_guess) { for (int v = 0; v < np; ++v) wg[v] = prim_guess[v * n + c]; guess_Z(wg, P, Zg); }
    int it;
    int rc = cons2prim(q, P, prim_guess ? Zg : nullptr, w, Zo, it);
    for (int v = 0; v < np; ++v) prims[v * n + c] = w[v];
    if (iters) iters[c] = it;
    if (fail) fail[c] = rc;
  }
  return 0;
}

int oracle_flux_vector_batch(const oracle_params* p, long long n, int dir, const double* cons,
                             const double* prims, const double* sigma_cell, double* f) {
  Par P0 = to_par(p); int nc = ncons(P0.model), np = nprim(P0.model);
#pragma omp parallel for schedule(static)
  for (long long c = 0; c < n; ++c) {
    Par P = P0; if (sigma_cell) P.sigma = sigma_cell[c];
    double w[MAXP], q[MAXN], ff[MAXN];
    for (int v = 0; v < nc; ++v) q[v] = cons[v * n + c];
    for (int v = 0; v < np; ++v) w[v] = prims[v * n + c];
    flux_vector(q, w, dir, P, ff);
    for (int v = 0; v < nc; ++v) f[v * n + c] = ff[v];
  }
  return 0;
}

int oracle_source_batch(const oracle_params* p, long long n, const double* cons, const double* prims,
                        const double* sigma_cell, double* src) {
  Par P0 = to_par(p); int nc = ncons(P0.model), np = nprim(P0.model);
#pragma omp parallel for schedule(static)
  for (long long c = 0; c < n; ++c) {
    Par P = P0; if (sigma_cell) P.sigma = sigma_cell[c];
    double w[MAXP], q[MAXN], s[MAXN];
    for (int v = 0; v < nc; ++v) q[v] = cons[v * n + c];
    for (int v = 0; v < np; ++v) w[v] = prims[v * n + c];
    source_vector(q, w, P, s);
    for (int v = 0; v < nc; ++v) src[v * n + c] = s[v];
  }
  return 0;
}

int oracle_species_split(double mu_e, double mu_p, long long n, const double* x, const double* xbar,
                         double* xe, double* xp) {
  if (mu_e == mu_p) return -1;
  double mu[2] = {mu_e, mu_p};
  for (long long c = 0; c < n; ++c) species_split(x[c], xbar[c], mu, &xe[c], &xp[c]);
  return 0;
}

int oracle_weno3(long long n, const double* a, const double* b, const double* c, double* out) {
  for (long long i = 0; i < n; ++i) out[i] = weno3(a[i], b[i], c[i]);
  return 0;
}

// frozen-v guess of the resistive stage (I.3); q_ex[14][n], prim_guess[11][n] -> E_guess[3][n]
int oracle_stage_guess_batch(const oracle_params* p, long long n, const double* q_ex, const double* prim_guess,
                             const double* sigma_cell, double a_dt, double* E_guess) {
  Par P = to_par(p);
  if (P.model != 0) return -1;
  for (long long c = 0; c < n; ++c) {
    double q[14], w[11], Eg[3];
    for (int v = 0; v < 14; ++v) q[v] = q_ex[v * n + c];
    for (int v = 0; v < 11; ++v) w[v] = prim_guess[v * n + c];
    r_stage_guess_E(q, w, a_dt, sigma_cell ? sigma_cell[c] : P.sigma, Eg);
    for (int i = 0; i < 3; ++i) E_guess[i * n + c] = Eg[i];
  }
  return 0;
}

// one implicit stage on n independent cells (config 2): q* - q_ex - a_dt Psi(q*) = 0
int oracle_stage_batch(const oracle_params* p, long long n, const double* q_ex, const double* prim_guess,
                       const double* sigma_cell, double a_dt, double* q_out, double* prims_out, int* iters,
                       int* fail) {
  Par P0 = to_par(p); int nc = ncons(P0.model), np = nprim(P0.model);
#pragma omp parallel for schedule(dynamic, 64)
  for (long long c = 0; c < n; ++c) {
    Par P = P0; if (sigma_cell) P.sigma = sigma_cell[c];
    double qe[MAXN], wg[MAXP], q[MAXN], w[MAXP];
    for (int v = 0; v < nc; ++v) qe[v] = q_ex[v * n + c];
    for (int v = 0; v < np; ++v) wg[v] = prim_guess[v * n + c];
    int it, c2;
    int rc = stage_solve(qe, wg, a_dt, P, q, w, it, c2);
    for (int v = 0; v < nc; ++v) q_out[v * n + c] = q[v];
    for (int v = 0; v < np; ++v) prims_out[v * n + c] = w[v];
    if (iters) iters[c] = it;
    if (fail) fail[c] = rc;
  }
  return 0;
}

// residual of eq (10) at given q (for the "stage residual" pin): R[nc][n]
int oracle_stage_residual_batch(const oracle_params* p, long long n, const double* q, const double* q_ex,
                                const double* sigma_cell, double a_dt, double* R, int* fail) {
  Par P0 = to_par(p); int nc = ncons(P0.model);
  for (long long c = 0; c < n; ++c) {
    Par P = P0; if (sigma_cell) P.sigma = sigma_cell[c];
    double qq[MAXN], qe[MAXN], r[MAXN], w[MAXP], Zo[2]; int it;
    for (int v = 0; v < nc; ++v) { qq[v] = q[v * n + c]; qe[v] = q_ex[v * n + c]; }
    int rc = stage_residual(qq, qe, a_dt, P, nullptr, r, w, Zo, it);
    for (int v = 0; v < nc; ++v) R[v * n + c] = rc ? std::numeric_limits<double>::quiet_NaN() : r[v];
    if (fail) fail[c] = rc;
  }
  return 0;
}

// ---- grid simulation -------------------------------------------------------------------
void* oracle_create(const oracle_params* p) {
  if (!p || (p->model != 0 && p->model != 1)) return nullptr;
  if (p->nx < 1 || p->ny < 1 || p->nz < 1 || p->ng < 2) return nullptr;
  if (p->model == 1 && p->mu_e == p->mu_p) return nullptr;
  Sim* S = new Sim();
  S->P = to_par(p);
  S->n[0] = p->nx; S->n[1] = p->ny; S->n[2] = p->nz;
  S->ng = p->ng;
  S->lo[0] = p->xmin; S->hi[0] = p->xmax; S->lo[1] = p->ymin; S->hi[1] = p->ymax; S->lo[2] = p->zmin; S->hi[2] = p->zmax;
  double inv = 0.0;
  S->ntot = 1;
  for (int d = 0; d < 3; ++d) {
    S->g[d] = S->n[d] > 1 ? p->ng : 0;
    S->N[d] = S->n[d] + 2 * S->g[d];
    S->dx[d] = (S->hi[d] - S->lo[d]) / S->n[d];
    S->bc[d] = p->bc[d];
    if (S->g[d]) inv += 1.0 / S->dx[d];
    S->ntot *= size_t(S->N[d]);
  }
  if (p->integrator < 0 || p->integrator > 2) { delete S; return nullptr; }
  S->integrator = p->integrator;
  S->cfl = p->cfl;
  S->dt = inv > 0 ? p->cfl / inv : p->cfl;   // G9: dt = CFL / sum_d 1/dx_d (alpha = 1)
  S->t0 = 0.0; S->nstep = 0;
  S->nc = ncons(S->P.model); S->np = nprim(S->P.model);
  size_t a = S->ntot * S->nc, b = S->ntot * S->np;
  S->q.assign(a, 0.0); S->q1.assign(a, 0.0); S->qs.assign(a, 0.0); S->L1.assign(a, 0.0); S->L2.assign(a, 0.0);
  S->Ps1.assign(a, 0.0); S->Ps2.assign(a, 0.0);
  S->w.assign(b, 0.0); S->w1.assign(b, 0.0);
  S->hist_stage.assign(64, 0); S->hist_c2p.assign(128, 0);
  S->n_failed = 0; S->first_failed = -1;
  return S;
}

// test hook: iterations of the first con2prim residual before the second takes over (default 20; 0 = second only)
int oracle_set_c2p_switch(int n) { int prev = g_c2p_switch; g_c2p_switch = n; return prev; }

void oracle_destroy(void* h) { delete static_cast<Sim*>(h); }
double oracle_dt(void* h) { return static_cast<Sim*>(h)->dt; }
double oracle_time(void* h) { Sim* S = static_cast<Sim*>(h); return S->t0 + double(S->nstep) * S->dt; }

// prims: interior cells only [np][nz][ny][nx]; rho_charge nullable ([nz][ny][nx]) =>
// Gauss's law with 2nd-order central differences on BC-filled ghosts (G10).
// psi = phi = 0.
int oracle_set_initial(void* h, const double* prims, const double* rho_charge) {
  Sim& S = *static_cast<Sim*>(h);
  const int nx = S.n[0], ny = S.n[1], nz = S.n[2];
  const size_t nin = size_t(nx) * ny * nz;
  for (int v = 0; v < S.np; ++v)
    for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i)
      S.w[size_t(v) * S.ntot + S.idx(i + S.g[0], j + S.g[1], k + S.g[2])] = prims[size_t(v) * nin + (size_t(k) * ny + j) * nx + i];
  fill_ghosts(S, S.w, S.np);
  const int eoff = S.P.model == 0 ? 8 : 13;
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    int c[3] = {i + S.g[0], j + S.g[1], k + S.g[2]};
    size_t id = S.idx(c[0], c[1], c[2]);
    double w[MAXP], q[MAXN];
    gather(S, S.w, S.np, id, w);
    if (S.P.model == 0) {
      double rc = 0.0;
      if (rho_charge) rc = rho_charge[(size_t(k) * ny + j) * nx + i];
      else {
        for (int d = 0; d < 3; ++d) {
          if (!S.g[d]) continue;
          int cp[3] = {c[0], c[1], c[2]}, cm[3] = {c[0], c[1], c[2]};
          cp[d] += 1; cm[d] -= 1;
          const double* Ed = S.w.data() + size_t(eoff + d) * S.ntot;
          rc += (Ed[S.idx(cp[0], cp[1], cp[2])] - Ed[S.idx(cm[0], cm[1], cm[2])]) / (2.0 * S.dx[d]);
        }
      }
      r_prim2cons(w, rc, 0.0, 0.0, S.P.gam, q);
    } else {
      t_prim2cons(w, 0.0, 0.0, S.P, q);
    }
    scatter(S, S.q, S.nc, id, q);
  }
  fill_ghosts(S, S.q, S.nc);
  S.nstep = 0; S.t0 = 0.0;
  std::fill(S.hist_stage.begin(), S.hist_stage.end(), 0);
  std::fill(S.hist_c2p.begin(), S.hist_c2p.end(), 0);
  S.n_failed = 0; S.first_failed = -1;
  return 0;
}

// overwrite the conserved state directly (interior) and recover primitives (for pins that
// need psi, phi != 0 or a specific conserved state).  prim_guess nullable.
int oracle_set_cons(void* h, const double* cons, const double* prim_guess) {
  Sim& S = *static_cast<Sim*>(h);
  const int nx = S.n[0], ny = S.n[1], nz = S.n[2];
  const size_t nin = size_t(nx) * ny * nz;
  int bad = 0;
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    size_t id = S.idx(i + S.g[0], j + S.g[1], k + S.g[2]);
    size_t ci = (size_t(k) * ny + j) * nx + i;
    double q[MAXN], w[MAXP], wg[MAXP], Zg[2] = {-1, -1}, Zo[2]; int it;
    for (int v = 0; v < S.nc; ++v) q[v] = cons[size_t(v) * nin + ci];
    if (prim_guess) { for (int v = 0; v < S.np; ++v) wg[v] = prim_guess[size_t(v) * nin + ci]; guess_Z(wg, S.P, Zg); }
    if (cons2prim(q, S.P, prim_guess ? Zg : nullptr, w, Zo, it)) bad++;
    scatter(S, S.q, S.nc, id, q); scatter(S, S.w, S.np, id, w);
  }
  fill_ghosts(S, S.q, S.nc); fill_ghosts(S, S.w, S.np);
  return bad;
}

int oracle_step(void* h, int nsteps) {
  Sim& S = *static_cast<Sim*>(h);
  for (int s = 0; s < nsteps; ++s) {
    if (S.integrator == 0) step_once(S);
    else step_imex(S, S.integrator == 1 ? tableau_ssp3_332() : tableau_ssp2_222());
  }
  return S.n_failed ? -3 : 0;
}

int oracle_get_state(void* h, double* cons, double* prims) {
  Sim& S = *static_cast<Sim*>(h);
  const int nx = S.n[0], ny = S.n[1], nz = S.n[2];
  const size_t nin = size_t(nx) * ny * nz;
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    size_t id = S.idx(i + S.g[0], j + S.g[1], k + S.g[2]);
    size_t ci = (size_t(k) * ny + j) * nx + i;
    if (cons) for (int v = 0; v < S.nc; ++v) cons[size_t(v) * nin + ci] = S.q[size_t(v) * S.ntot + id];
    if (prims) for (int v = 0; v < S.np; ++v) prims[size_t(v) * nin + ci] = S.w[size_t(v) * S.ntot + id];
  }
  return 0;
}

// L(q) of the current state on interior cells: Lout[nc][nz][ny][nx]
int oracle_eval_L(void* h, double* Lout) {
  Sim& S = *static_cast<Sim*>(h);
  eval_L(S, S.q, S.w, S.L1);
  const int nx = S.n[0], ny = S.n[1], nz = S.n[2];
  const size_t nin = size_t(nx) * ny * nz;
  for (int k = 0; k < nz; ++k) for (int j = 0; j < ny; ++j) for (int i = 0; i < nx; ++i) {
    size_t id = S.idx(i + S.g[0], j + S.g[1], k + S.g[2]);
    size_t ci = (size_t(k) * ny + j) * nx + i;
    for (int v = 0; v < S.nc; ++v) Lout[size_t(v) * nin + ci] = S.L1[size_t(v) * S.ntot + id];
  }
  return 0;
}

int oracle_get_stats(void* h, long long* hist_stage, long long* hist_c2p, int nbins, long long* n_failed,
                     long long* first_failed_cell) {
  Sim& S = *static_cast<Sim*>(h);
  for (int b = 0; b < nbins; ++b) {
    if (hist_stage) hist_stage[b] = b < int(S.hist_stage.size()) ? S.hist_stage[b] : 0;
    if (hist_c2p) hist_c2p[b] = b < int(S.hist_c2p.size()) ? S.hist_c2p[b] : 0;
  }
  if (n_failed) *n_failed = S.n_failed;
  if (first_failed_cell) *first_failed_cell = S.first_failed;
  return 0;
}

}  // extern "C"

// stage.cuh -- per-cell implicit-stage solvers (eq 10) kept in registers.
//
// The paper solves the stage with an N-dimensional hybrd root-find on all N conserved
// components (N = 14 / 18, work array N(3N+13) doubles in global memory).  Only the
// rows with a non-zero source are genuine unknowns (eq 1; A2 P:L445):
//   resistive : E (3)  [psi, phi are linear and closed-form];  all other rows equal q_ex
//   two-fluid : Sbar (3), taubar, E (3)
// and the primitive recovery nested inside every residual evaluation is removed by carrying
// Z = rho h W^2 (one per species) as an extra Newton unknown with its own residual
// f(Z) = Z - p - taut - D = 0.  Resistive: a 4x4 Newton system with closed-form Jacobian,
// reduced to 3x3 by eliminating Z (Schur complement), solved by Cramer's rule.
// The root is the one the oracle's full-N solve finds; parity tests check exactly that.
#pragma once
#include "physics.cuh"

namespace rmhd {

// ---------------------------------------------------------------------------------------
// Resistive stage:  E - E_ex + a J(E, v(E,Z), W(E,Z)) = 0,   Z - p(E,Z) - taut(E) - D = 0
// ---------------------------------------------------------------------------------------
struct RStage {
  // fixed data of the cell
  double D, Sx, Sy, Sz, tau, Bx, By, Bz, B2, Eex, Eey, Eez, rhoc;
  double a, sigma, scale;
  // unknowns
  double Ex, Ey, Ez, Z;
  int status;  // 0 iterating, 1 converged, <0 failed
  int iters;
};

RMHD_DEV bool r_admissible(const RStage& s, double Ex, double Ey, double Ez, double& S2, double& tD) {
  const double tx = s.Sx - (Ey * s.Bz - Ez * s.By);
  const double ty = s.Sy - (Ez * s.Bx - Ex * s.Bz);
  const double tz = s.Sz - (Ex * s.By - Ey * s.Bx);
  S2 = tx * tx + ty * ty + tz * tz;
  tD = s.tau - 0.5 * (Ex * Ex + Ey * Ey + Ez * Ez + s.B2) + s.D;
  return (tD > 0.0) && (tD * tD > S2);
}

// q_ex: the 14 explicit-part rows; (rho_g, vg, p_g): primitives near the solution (guess).
RMHD_DEV void r_stage_init(RStage& s, const double* qe, double rho_g, double vgx, double vgy, double vgz, double p_g,
                           double a, double sigma, const DevPar& P) {
  s.D = qe[0]; s.Sx = qe[1]; s.Sy = qe[2]; s.Sz = qe[3]; s.tau = qe[4];
  s.Bx = qe[5]; s.By = qe[6]; s.Bz = qe[7];
  s.Eex = qe[8]; s.Eey = qe[9]; s.Eez = qe[10]; s.rhoc = qe[11];
  s.B2 = s.Bx * s.Bx + s.By * s.By + s.Bz * s.Bz;
  s.a = a; s.sigma = sigma;
  s.status = 0; s.iters = 0;
  s.scale = fmax(fmax(1.0, fmax(fabs(s.D), fabs(s.tau))),
                 fmax(max3abs(s.Sx, s.Sy, s.Sz), fmax(max3abs(s.Bx, s.By, s.Bz), max3abs(s.Eex, s.Eey, s.Eez))));
  // frozen-(v,W) guess: (1+s) E - s v (v.E) = b,  b = E_ex - a rhoc v - s (v x B);  Sherman-Morrison inverse
  const double vg2 = vgx * vgx + vgy * vgy + vgz * vgz;
  const double Wg2 = 1.0 / (1.0 - vg2);
  const double Wg = sqrt(Wg2);
  const double sw = a * Wg * sigma;
  const double bx = s.Eex - a * s.rhoc * vgx - sw * (vgy * s.Bz - vgz * s.By);
  const double by = s.Eey - a * s.rhoc * vgy - sw * (vgz * s.Bx - vgx * s.Bz);
  const double bz = s.Eez - a * s.rhoc * vgz - sw * (vgx * s.By - vgy * s.Bx);
  const double c = sw * (vgx * bx + vgy * by + vgz * bz) / (1.0 + sw - sw * vg2);
  const double r = 1.0 / (1.0 + sw);
  s.Ex = (bx + c * vgx) * r; s.Ey = (by + c * vgy) * r; s.Ez = (bz + c * vgz) * r;
  s.Z = (rho_g + P.gi * p_g) * Wg2;
  double S2, tD;
  bool ok = isfinite(s.Ex + s.Ey + s.Ez) && r_admissible(s, s.Ex, s.Ey, s.Ez, S2, tD);
  if (!ok) {
    s.Ex = s.Eex; s.Ey = s.Eey; s.Ez = s.Eez;
    ok = r_admissible(s, s.Ex, s.Ey, s.Ez, S2, tD);
  }
  if (!ok || !(s.D > 0.0)) { s.status = -1; return; }
  if (!(s.Z * s.Z > S2) || !isfinite(s.Z)) s.Z = fmax(tD, sqrt(S2) * (1.0 + 1e-8) + 1e-300);
}

// one Newton iteration on (E, Z); sets status when converged / failed
RMHD_DEV void r_stage_iter(RStage& s, const DevPar& P) {
  const double Ex = s.Ex, Ey = s.Ey, Ez = s.Ez, Z = s.Z;
  const double ExBx = Ey * s.Bz - Ez * s.By, ExBy = Ez * s.Bx - Ex * s.Bz, ExBz = Ex * s.By - Ey * s.Bx;
  const double iZ = 1.0 / Z;
  const double vx = (s.Sx - ExBx) * iZ, vy = (s.Sy - ExBy) * iZ, vz = (s.Sz - ExBz) * iZ;
  const double v2 = vx * vx + vy * vy + vz * vz;
  const double om = 1.0 - v2;
  const double W = rsqrt(om);
  const double sq = om * W;
  const double E2 = Ex * Ex + Ey * Ey + Ez * Ez;
  // residuals
  const double F4 = Z - P.g * (Z * om - s.D * sq) - (s.tau - 0.5 * (E2 + s.B2)) - s.D;
  const double vxBx = vy * s.Bz - vz * s.By, vxBy = vz * s.Bx - vx * s.Bz, vxBz = vx * s.By - vy * s.Bx;
  const double vE = vx * Ex + vy * Ey + vz * Ez;
  const double Kx = Ex + vxBx - vE * vx, Ky = Ey + vxBy - vE * vy, Kz = Ez + vxBz - vE * vz;
  const double sW = s.sigma * W;
  const double F1 = Ex - s.Eex + s.a * (s.rhoc * vx + sW * Kx);
  const double F2 = Ey - s.Eey + s.a * (s.rhoc * vy + sW * Ky);
  const double F3 = Ez - s.Eez + s.a * (s.rhoc * vz + sW * Kz);
  // Jacobian: C = [B]x, dv/dE = C/Z, dv/dZ = -v/Z,
  // dv2/dE = 2 (v x B)/Z, dv2/dZ = -2 v2/Z, dW = W^3 dv2 / 2
  const double pv2 = P.g * (0.5 * s.D * W - Z);                 // dp/dv2
  const double A33 = 1.0 - P.g * om + 2.0 * pv2 * v2 * iZ;      // = f'(Z) of con2prim
  const double A30 = Ex - 2.0 * pv2 * iZ * vxBx;
  const double A31 = Ey - 2.0 * pv2 * iZ * vxBy;
  const double A32 = Ez - 2.0 * pv2 * iZ * vxBz;
  const double t1 = s.a * s.sigma * W * W * W * iZ;             // a d(sigma W)/dv2 * 2/Z
  const double aw = s.a * sW;
  const double awz = aw * iZ;
  const double arz = s.a * s.rhoc * iZ;
  // (Kv C)_ij = B2 delta_ij - B_i B_j - v_i (ExB)_j - vE C_ij ;  C_ij x_j = (B x x)_i
  // A_ij = delta_ij + arz C_ij + t1 K_i (vxB)_j + aw (delta_ij - v_i v_j) + awz (Kv C)_ij
  const double cc = arz - awz * vE;                             // coefficient of C_ij
  const double dg = 1.0 + aw + awz * s.B2;                      // coefficient of delta_ij
  double M00 = dg - aw * vx * vx - awz * (s.Bx * s.Bx + vx * ExBx) + t1 * Kx * vxBx;
  double M01 = -cc * s.Bz - aw * vx * vy - awz * (s.Bx * s.By + vx * ExBy) + t1 * Kx * vxBy;
  double M02 = cc * s.By - aw * vx * vz - awz * (s.Bx * s.Bz + vx * ExBz) + t1 * Kx * vxBz;
  double M10 = cc * s.Bz - aw * vy * vx - awz * (s.By * s.Bx + vy * ExBx) + t1 * Ky * vxBx;
  double M11 = dg - aw * vy * vy - awz * (s.By * s.By + vy * ExBy) + t1 * Ky * vxBy;
  double M12 = -cc * s.Bx - aw * vy * vz - awz * (s.By * s.Bz + vy * ExBz) + t1 * Ky * vxBz;
  double M20 = -cc * s.By - aw * vz * vx - awz * (s.Bz * s.Bx + vz * ExBx) + t1 * Kz * vxBx;
  double M21 = cc * s.Bx - aw * vz * vy - awz * (s.Bz * s.By + vz * ExBy) + t1 * Kz * vxBy;
  double M22 = dg - aw * vz * vz - awz * (s.Bz * s.Bz + vz * ExBz) + t1 * Kz * vxBz;
  // dF_i/dZ = a [ -rhoc v_i/Z - sigma W^3 v2/Z K_i - sigma W/Z ((v x B)_i - 2 vE v_i) ]
  const double t2 = t1 * v2;
  const double A03 = -(arz * vx + t2 * Kx + awz * (vxBx - 2.0 * vE * vx));
  const double A13 = -(arz * vy + t2 * Ky + awz * (vxBy - 2.0 * vE * vy));
  const double A23 = -(arz * vz + t2 * Kz + awz * (vxBz - 2.0 * vE * vz));
  // eliminate Z:  dZ = -(F4 + A3j dE_j)/A33
  const double r33 = 1.0 / A33;
  const double c0 = A03 * r33, c1 = A13 * r33, c2 = A23 * r33;
  M00 -= c0 * A30; M01 -= c0 * A31; M02 -= c0 * A32;
  M10 -= c1 * A30; M11 -= c1 * A31; M12 -= c1 * A32;
  M20 -= c2 * A30; M21 -= c2 * A31; M22 -= c2 * A32;
  const double b0 = -(F1 - c0 * F4), b1 = -(F2 - c1 * F4), b2 = -(F3 - c2 * F4);
  // Cramer
  const double k00 = M11 * M22 - M12 * M21, k01 = M10 * M22 - M12 * M20, k02 = M10 * M21 - M11 * M20;
  const double idet = 1.0 / (M00 * k00 - M01 * k01 + M02 * k02);
  double dEx = (b0 * k00 - M01 * (b1 * M22 - M12 * b2) + M02 * (b1 * M21 - M11 * b2)) * idet;
  double dEy = (M00 * (b1 * M22 - M12 * b2) - b0 * k01 + M02 * (M10 * b2 - b1 * M20)) * idet;
  double dEz = (M00 * (M11 * b2 - b1 * M21) - M01 * (M10 * b2 - b1 * M20) + b0 * k02) * idet;
  double dZ = -(F4 + A30 * dEx + A31 * dEy + A32 * dEz) * r33;
  s.iters++;
  if (!isfinite(dEx + dEy + dEz + dZ)) { s.status = -2; return; }
  // keep the iterate admissible (v^2 < 1, a root of f exists): halve the update if needed
  double lam = 1.0, S2, tD;
  bool ok = false;
  for (int h = 0; h < 12; ++h) {
    const double Zn = Z + lam * dZ;
    ok = r_admissible(s, Ex + lam * dEx, Ey + lam * dEy, Ez + lam * dEz, S2, tD) && (Zn > 0.0) && (Zn * Zn > S2 * (1.0 + 1e-14));
    if (ok) break;
    lam *= 0.5;
  }
  if (!ok) { s.status = -3; return; }
  dEx *= lam; dEy *= lam; dEz *= lam; dZ *= lam;
  s.Ex = Ex + dEx; s.Ey = Ey + dEy; s.Ez = Ez + dEz; s.Z = Z + dZ;
  // converged when the applied update is below tolerance (the root then sits at round-off)
  if (lam == 1.0 && max3abs(dEx, dEy, dEz) <= P.tol_stage * s.scale && fabs(dZ) <= P.tol_stage * fmax(s.scale, s.Z))
    s.status = 1;
}

// primitives, current and the closed-form linear rows at the converged (E, Z)
RMHD_DEV void r_stage_finish(const RStage& s, const DevPar& P, Hyd& h, double* J, double& psi, double& phi,
                             double qpsi_ex, double qphi_ex) {
  const double tx = s.Sx - (s.Ey * s.Bz - s.Ez * s.By);
  const double ty = s.Sy - (s.Ez * s.Bx - s.Ex * s.Bz);
  const double tz = s.Sz - (s.Ex * s.By - s.Ey * s.Bx);
  hyd_from_Z(s.D, tx, ty, tz, tx * tx + ty * ty + tz * tz, s.Z, P.g, h);
  const double vE = h.vx * s.Ex + h.vy * s.Ey + h.vz * s.Ez;
  const double ws = h.W * s.sigma;
  J[0] = s.rhoc * h.vx + ws * (s.Ex + (h.vy * s.Bz - h.vz * s.By) - vE * h.vx);
  J[1] = s.rhoc * h.vy + ws * (s.Ey + (h.vz * s.Bx - h.vx * s.Bz) - vE * h.vy);
  J[2] = s.rhoc * h.vz + ws * (s.Ez + (h.vx * s.By - h.vy * s.Bx) - vE * h.vz);
  // psi' = rhoc - kappa psi, phi' = -kappa phi with rhoc fixed in the stage: linear, closed form
  const double ik = 1.0 / (1.0 + s.a * P.kappa);
  psi = (qpsi_ex + s.a * s.rhoc) * ik;
  phi = qphi_ex * ik;
}

}  // namespace rmhd

namespace rmhd {

// ---------------------------------------------------------------------------------------
// Two-fluid stage (A2-A3 P:L445-451, eq 7-8; readings G2, G3).  Rows with a source:
// Sbar (3), taubar, E (3) [psi, phi closed form with rhoc = Dbar fixed]; D, S, tau, Dbar, B equal
// q_ex.  Unknowns x = (Sbar, taubar, E) and Z_e, Z_p (one per species, replacing the two nested
// con2prims):
//   F_Sbar = Sbar - Sbar_ex - a [Kq E + U x B - eta (wp2 J - rho0 U)]
//   F_tbar = tbar - tbar_ex - a [U.E - eta (wp2 rhoc - rho0 Kq)]
//   F_E    = E - E_ex + a J
//   G_s    = Z_s - p_s(Z_s, S_s) - tau_s - D_s,   S_s = c_s Sbar + d_s (S - E x B),
//            tau_s = c_s tbar + d_s (tau - (E^2+B^2)/2),   v_s = S_s / Z_s
// with m_s = mu_s D_s, m2_s = mu_s^2 D_s (constants of the stage), Kq = sum m2_s, rhoc = sum m_s,
// J = sum m_s v_s, U = sum m2_s v_s, wp2 = sum m2_s sqrt(1-v_s^2), rho0 = (Kq rhoc - J.U)/wp2.
// Jacobian by exact forward-mode tangents, one direction at a time (all in registers); Z_e, Z_p are
// eliminated in closed form inside the species tangent (G_s depends on one Z only and on x through
// v_s . dS_s and dtau_s; see t_stage_iter), leaving a 7x7 system solved by Gaussian elimination
// in the order (Sbar, tbar, E): the pivots are 1 + a eta wp2 k > 0 and 1 + a^2 k Kq/(..) > 0
// (k = sum m_s c_s / Z_s), so no pivoting is needed.
// ---------------------------------------------------------------------------------------
struct TKin { double iZ, vx, vy, vz, om, W, sq; };

struct TStage {
  double D[2], Sx, Sy, Sz, tau, Bx, By, Bz, B2;
  double Sbex[3], tbex, Eex[3];
  double m[2], m2[2], Kq, rhoc;
  double c[2], d[2];          // species split: x_s = c_s xbar + d_s x
  double a, eta, scale;
  double Sb[3], tb, E[3], Z[2];
  int status, iters;
};

// species momenta / energies at (Sb, tb, E); returns admissibility of both species for given Z
RMHD_DEV bool t_species(const TStage& s, const double* Sb, double tb, const double* E, const double* Z,
                        double Ss[2][3], double* ts) {
  const double tx = s.Sx - (E[1] * s.Bz - E[2] * s.By);
  const double ty = s.Sy - (E[2] * s.Bx - E[0] * s.Bz);
  const double tz = s.Sz - (E[0] * s.By - E[1] * s.Bx);
  const double taut = s.tau - 0.5 * (E[0] * E[0] + E[1] * E[1] + E[2] * E[2] + s.B2);
  bool ok = true;
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    Ss[k][0] = s.c[k] * Sb[0] + s.d[k] * tx;
    Ss[k][1] = s.c[k] * Sb[1] + s.d[k] * ty;
    Ss[k][2] = s.c[k] * Sb[2] + s.d[k] * tz;
    ts[k] = s.c[k] * tb + s.d[k] * taut;
    const double S2 = Ss[k][0] * Ss[k][0] + Ss[k][1] * Ss[k][1] + Ss[k][2] * Ss[k][2];
    const double tD = ts[k] + s.D[k];
    ok = ok && (tD > 0.0) && (tD * tD > S2) && (Z[k] > 0.0) && (Z[k] * Z[k] > S2 * (1.0 + 1e-14));
  }
  return ok;
}

// q_ex: the 18 explicit-part rows; wg: 10 hydro primitives near the solution
RMHD_DEV void t_stage_init(TStage& s, const double* qe, const double* wg, double a, const DevPar& P) {
  const Split sp(P);
  s.c[0] = sp.ce; s.d[0] = sp.de; s.c[1] = sp.cp; s.d[1] = sp.dp;
  s.D[0] = sp.ce * qe[5] + sp.de * qe[0];
  s.D[1] = sp.cp * qe[5] + sp.dp * qe[0];
  s.Sx = qe[1]; s.Sy = qe[2]; s.Sz = qe[3]; s.tau = qe[4];
  s.Bx = qe[10]; s.By = qe[11]; s.Bz = qe[12];
  s.B2 = s.Bx * s.Bx + s.By * s.By + s.Bz * s.Bz;
#pragma unroll
  for (int i = 0; i < 3; ++i) { s.Sbex[i] = qe[6 + i]; s.Eex[i] = qe[13 + i]; s.Sb[i] = qe[6 + i]; s.E[i] = qe[13 + i]; }
  s.tbex = qe[9]; s.tb = qe[9];
  s.m[0] = P.mu_e * s.D[0]; s.m[1] = P.mu_p * s.D[1];
  s.m2[0] = P.mu_e * s.m[0]; s.m2[1] = P.mu_p * s.m[1];
  s.Kq = s.m2[0] + s.m2[1]; s.rhoc = s.m[0] + s.m[1];
  s.a = a; s.eta = P.eta;
  s.status = 0; s.iters = 0;
  double sc = 1.0;
#pragma unroll
  for (int v = 0; v < 16; ++v) sc = fmax(sc, fabs(qe[v]));
  s.scale = sc;
#pragma unroll
  for (int k = 0; k < 2; ++k) s.Z[k] = Z_of_prims(wg[5 * k], wg[5 * k + 1], wg[5 * k + 2], wg[5 * k + 3], wg[5 * k + 4], P);
  if (!(s.D[0] > 0.0) || !(s.D[1] > 0.0) || !isfinite(sc)) { s.status = -1; return; }
  // the guess must be admissible for both species; repair Z_s if only that is off
  double Ss[2][3], ts[2];
  if (!t_species(s, s.Sb, s.tb, s.E, s.Z, Ss, ts)) {
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const double S2 = Ss[k][0] * Ss[k][0] + Ss[k][1] * Ss[k][1] + Ss[k][2] * Ss[k][2];
      if (!(s.Z[k] * s.Z[k] > S2 * (1.0 + 1e-14)) || !isfinite(s.Z[k])) s.Z[k] = fmax(ts[k] + s.D[k], sqrt(S2) * (1.0 + 1e-8) + 1e-300);
    }
    if (!t_species(s, s.Sb, s.tb, s.E, s.Z, Ss, ts)) s.status = -1;
  }
}

struct TAgg { double J[3], U[3], wp2, iw, rho0; };

// tangent of the seven F rows given the species tangents and the direct (dSb, dtb, dE) parts
RMHD_DEV void t_F_tan(const TStage& s, const TAgg& A, const double dv[2][3], const double* dsq,
                      const double* dSb, double dtb, const double* dE, double* dF) {
  double dJ[3], dU[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) { dJ[i] = s.m[0] * dv[0][i] + s.m[1] * dv[1][i]; dU[i] = s.m2[0] * dv[0][i] + s.m2[1] * dv[1][i]; }
  const double dwp2 = s.m2[0] * dsq[0] + s.m2[1] * dsq[1];
  const double dJU = dJ[0] * A.U[0] + dJ[1] * A.U[1] + dJ[2] * A.U[2] + A.J[0] * dU[0] + A.J[1] * dU[1] + A.J[2] * dU[2];
  const double drho0 = -(dJU + A.rho0 * dwp2) * A.iw;
  const double E0 = s.E[0], E1 = s.E[1], E2 = s.E[2];
  const double cx = dU[1] * s.Bz - dU[2] * s.By, cy = dU[2] * s.Bx - dU[0] * s.Bz, cz = dU[0] * s.By - dU[1] * s.Bx;
  const double ae = s.a * s.eta;
  dF[0] = dSb[0] - s.a * (s.Kq * dE[0] + cx) + ae * (dwp2 * A.J[0] + A.wp2 * dJ[0] - drho0 * A.U[0] - A.rho0 * dU[0]);
  dF[1] = dSb[1] - s.a * (s.Kq * dE[1] + cy) + ae * (dwp2 * A.J[1] + A.wp2 * dJ[1] - drho0 * A.U[1] - A.rho0 * dU[1]);
  dF[2] = dSb[2] - s.a * (s.Kq * dE[2] + cz) + ae * (dwp2 * A.J[2] + A.wp2 * dJ[2] - drho0 * A.U[2] - A.rho0 * dU[2]);
  dF[3] = dtb - s.a * (dU[0] * E0 + dU[1] * E1 + dU[2] * E2 + A.U[0] * dE[0] + A.U[1] * dE[1] + A.U[2] * dE[2])
          + ae * (dwp2 * s.rhoc - drho0 * s.Kq);
  dF[4] = dE[0] + s.a * dJ[0];
  dF[5] = dE[1] + s.a * dJ[1];
  dF[6] = dE[2] + s.a * dJ[2];
}

RMHD_DEV void t_stage_iter(TStage& s, const DevPar& P) {
  double Ss[2][3], ts[2];
  t_species(s, s.Sb, s.tb, s.E, s.Z, Ss, ts);
  TKin k[2];
  double G[2];
#pragma unroll
  for (int q = 0; q < 2; ++q) {
    k[q].iZ = 1.0 / s.Z[q];
    k[q].vx = Ss[q][0] * k[q].iZ; k[q].vy = Ss[q][1] * k[q].iZ; k[q].vz = Ss[q][2] * k[q].iZ;
    k[q].om = 1.0 - (k[q].vx * k[q].vx + k[q].vy * k[q].vy + k[q].vz * k[q].vz);
    k[q].W = rsqrt(k[q].om);
    k[q].sq = k[q].om * k[q].W;
    G[q] = s.Z[q] - P.g * (s.Z[q] * k[q].om - s.D[q] * k[q].sq) - ts[q] - s.D[q];
  }
  TAgg A;
  A.J[0] = s.m[0] * k[0].vx + s.m[1] * k[1].vx; A.J[1] = s.m[0] * k[0].vy + s.m[1] * k[1].vy; A.J[2] = s.m[0] * k[0].vz + s.m[1] * k[1].vz;
  A.U[0] = s.m2[0] * k[0].vx + s.m2[1] * k[1].vx; A.U[1] = s.m2[0] * k[0].vy + s.m2[1] * k[1].vy; A.U[2] = s.m2[0] * k[0].vz + s.m2[1] * k[1].vz;
  A.wp2 = s.m2[0] * k[0].sq + s.m2[1] * k[1].sq;
  A.iw = 1.0 / A.wp2;
  A.rho0 = (s.Kq * s.rhoc - (A.J[0] * A.U[0] + A.J[1] * A.U[1] + A.J[2] * A.U[2])) * A.iw;
  double F[7];
  {
    const double ae = s.a * s.eta;
    F[0] = s.Sb[0] - s.Sbex[0] - s.a * (s.Kq * s.E[0] + (A.U[1] * s.Bz - A.U[2] * s.By)) + ae * (A.wp2 * A.J[0] - A.rho0 * A.U[0]);
    F[1] = s.Sb[1] - s.Sbex[1] - s.a * (s.Kq * s.E[1] + (A.U[2] * s.Bx - A.U[0] * s.Bz)) + ae * (A.wp2 * A.J[1] - A.rho0 * A.U[1]);
    F[2] = s.Sb[2] - s.Sbex[2] - s.a * (s.Kq * s.E[2] + (A.U[0] * s.By - A.U[1] * s.Bx)) + ae * (A.wp2 * A.J[2] - A.rho0 * A.U[2]);
    F[3] = s.tb - s.tbex - s.a * (A.U[0] * s.E[0] + A.U[1] * s.E[1] + A.U[2] * s.E[2]) + ae * (A.wp2 * s.rhoc - A.rho0 * s.Kq);
    F[4] = s.E[0] - s.Eex[0] + s.a * A.J[0];
    F[5] = s.E[1] - s.Eex[1] + s.a * A.J[1];
    F[6] = s.E[2] - s.Eex[2] + s.a * A.J[2];
  }
  const double zero3[3] = {0.0, 0.0, 0.0};
  // ---- Z_s eliminated in closed form.  With dZ_s = 0:  dG_s = gam_s (v_s . dS_s) - dtau_s, gam_s = g (2 - D_s W_s / Z_s);
  // dG_s/dZ_s = f'(Z_s) = 1 - g (1 + v^2 - D W v^2 / Z) (con2prim's derivative).  The Newton condition G_s + dG_s = 0 gives
  //   dZ_s = -(G_s + gam_s v_s . dS_s - dtau_s) / f'_s,    dv_s = (dS_s - v_s dZ_s) / Z_s,    dsq_s = -W_s (v_s . dv_s),
  // i.e. dv_s is affine in (dS_s, dtau_s): the constant part (from G_s) goes to the right-hand side, the linear part
  // into the 7 x 7 matrix.  Same Newton step as a Schur complement on the 9 x 9 system, without its Z rows and columns.
  double gam[2], rfp[2];
#pragma unroll
  for (int q = 0; q < 2; ++q) {
    const double v2 = 1.0 - k[q].om;
    gam[q] = P.g * (2.0 - s.D[q] * k[q].W * k[q].iZ);
    rfp[q] = 1.0 / (1.0 - P.g * (1.0 + v2 - s.D[q] * k[q].W * v2 * k[q].iZ));
  }
  auto species_tan = [&](int q, double dSx, double dSy, double dSz, double dts, double G0, double* dv, double& dsq) {
    const double vdS = k[q].vx * dSx + k[q].vy * dSy + k[q].vz * dSz;
    const double mdZ = (G0 + gam[q] * vdS - dts) * rfp[q];          // = -dZ_s
    dv[0] = (dSx + k[q].vx * mdZ) * k[q].iZ;
    dv[1] = (dSy + k[q].vy * mdZ) * k[q].iZ;
    dv[2] = (dSz + k[q].vz * mdZ) * k[q].iZ;
    dsq = -(k[q].vx * dv[0] + k[q].vy * dv[1] + k[q].vz * dv[2]) * k[q].W;
  };
  double b[7];
  {   // right-hand side: -(F + dF/dv . dv0), dv0 = the change of v_s when Z_s alone takes its Newton correction
    double dv[2][3], dsq[2], dF[7];
#pragma unroll
    for (int q = 0; q < 2; ++q) species_tan(q, 0.0, 0.0, 0.0, 0.0, G[q], dv[q], dsq[q]);
    t_F_tan(s, A, dv, dsq, zero3, 0.0, zero3, dF);
#pragma unroll
    for (int i = 0; i < 7; ++i) b[i] = -(F[i] + dF[i]);
  }
  double M[7][7];
#pragma unroll
  for (int j = 0; j < 7; ++j) {
    double dSb[3] = {0, 0, 0}, dE[3] = {0, 0, 0}, dSt[3] = {0, 0, 0}, dtb = 0.0, dtaut = 0.0;
    if (j < 3) dSb[j] = 1.0;
    else if (j == 3) dtb = 1.0;
    else {
      const int e = j - 4;
      dE[e] = 1.0;
      // d(S - E x B)/dE_e = B x e_e
      if (e == 0) { dSt[1] = s.Bz; dSt[2] = -s.By; }
      if (e == 1) { dSt[0] = -s.Bz; dSt[2] = s.Bx; }
      if (e == 2) { dSt[0] = s.By; dSt[1] = -s.Bx; }
      dtaut = -s.E[e];
    }
    double dv[2][3], dsq[2], dF[7];
#pragma unroll
    for (int q = 0; q < 2; ++q)
      species_tan(q, s.c[q] * dSb[0] + s.d[q] * dSt[0], s.c[q] * dSb[1] + s.d[q] * dSt[1], s.c[q] * dSb[2] + s.d[q] * dSt[2],
                  s.c[q] * dtb + s.d[q] * dtaut, 0.0, dv[q], dsq[q]);
    t_F_tan(s, A, dv, dsq, dSb, dtb, dE, dF);
#pragma unroll
    for (int i = 0; i < 7; ++i) M[i][j] = dF[i];
  }
  // ---- Gaussian elimination, no pivoting (see header comment)
#pragma unroll
  for (int c = 0; c < 7; ++c) {
    const double r = 1.0 / M[c][c];
#pragma unroll
    for (int i = c + 1; i < 7; ++i) {
      const double f = M[i][c] * r;
#pragma unroll
      for (int j = c + 1; j < 7; ++j) M[i][j] -= f * M[c][j];
      b[i] -= f * b[c];
    }
  }
  double dx[7];
#pragma unroll
  for (int i = 6; i >= 0; --i) {
    double t = b[i];
#pragma unroll
    for (int j = i + 1; j < 7; ++j) t -= M[i][j] * dx[j];
    dx[i] = t / M[i][i];
  }
  double dZ[2];
  {
    // dS_s, dtau_s of the solved update:  dSt = B x dE,  dtaut = -E . dE
    const double tx = s.By * dx[6] - s.Bz * dx[5], ty = s.Bz * dx[4] - s.Bx * dx[6], tz = s.Bx * dx[5] - s.By * dx[4];
    const double dtaut = -(s.E[0] * dx[4] + s.E[1] * dx[5] + s.E[2] * dx[6]);
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const double vdS = k[q].vx * (s.c[q] * dx[0] + s.d[q] * tx) + k[q].vy * (s.c[q] * dx[1] + s.d[q] * ty) +
                         k[q].vz * (s.c[q] * dx[2] + s.d[q] * tz);
      dZ[q] = -(G[q] + gam[q] * vdS - (s.c[q] * dx[3] + s.d[q] * dtaut)) * rfp[q];
    }
  }
  s.iters++;
  double sum = dZ[0] + dZ[1];
#pragma unroll
  for (int j = 0; j < 7; ++j) sum += dx[j];
  if (!isfinite(sum)) { s.status = -2; return; }
  // keep both species admissible: halve the update if needed
  double lam = 1.0;
  bool ok = false;
  double Sbn[3], En[3], Zn[2], tbn = s.tb;
  for (int h = 0; h < 12; ++h) {
#pragma unroll
    for (int i = 0; i < 3; ++i) { Sbn[i] = s.Sb[i] + lam * dx[i]; En[i] = s.E[i] + lam * dx[4 + i]; }
    tbn = s.tb + lam * dx[3];
    Zn[0] = s.Z[0] + lam * dZ[0]; Zn[1] = s.Z[1] + lam * dZ[1];
    ok = t_species(s, Sbn, tbn, En, Zn, Ss, ts);
    if (ok) break;
    lam *= 0.5;
  }
  if (!ok) { s.status = -3; return; }
  double dmax = 0.0;
#pragma unroll
  for (int j = 0; j < 7; ++j) dmax = fmax(dmax, fabs(dx[j]));
#pragma unroll
  for (int i = 0; i < 3; ++i) { s.Sb[i] = Sbn[i]; s.E[i] = En[i]; }
  s.tb = tbn; s.Z[0] = Zn[0]; s.Z[1] = Zn[1];
  if (lam == 1.0 && dmax <= P.tol_stage * s.scale && fabs(dZ[0]) <= P.tol_stage * fmax(s.scale, s.Z[0]) &&
      fabs(dZ[1]) <= P.tol_stage * fmax(s.scale, s.Z[1]))
    s.status = 1;
}

// primitives and the source rows at the converged state.  src: Sbar(3), tbar, E(3), psi, phi rows
RMHD_DEV void t_stage_finish(const TStage& s, const DevPar& P, double* w /*10*/, double* src /*9*/, double& psi, double& phi,
                             double qpsi_ex, double qphi_ex) {
  double Ss[2][3], ts[2];
  t_species(s, s.Sb, s.tb, s.E, s.Z, Ss, ts);
  Hyd h[2];
#pragma unroll
  for (int q = 0; q < 2; ++q) {
    hyd_from_Z(s.D[q], Ss[q][0], Ss[q][1], Ss[q][2], Ss[q][0] * Ss[q][0] + Ss[q][1] * Ss[q][1] + Ss[q][2] * Ss[q][2], s.Z[q], P.g, h[q]);
    w[5 * q] = h[q].rho; w[5 * q + 1] = h[q].vx; w[5 * q + 2] = h[q].vy; w[5 * q + 3] = h[q].vz; w[5 * q + 4] = h[q].p;
  }
  const double B[3] = {s.Bx, s.By, s.Bz};
  t_source7(s.D, h, B, s.E, P, src);
  const double ik = 1.0 / (1.0 + s.a * P.kappa);
  psi = (qpsi_ex + s.a * s.rhoc) * ik;
  phi = qphi_ex * ik;
  src[7] = s.rhoc - P.kappa * psi;
  src[8] = -P.kappa * phi;
}

}  // namespace rmhd

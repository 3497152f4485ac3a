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

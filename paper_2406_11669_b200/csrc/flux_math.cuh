// flux_math.cuh -- per-face arithmetic of the marching flux kernel (flux_march.cuh):
// one side's conserved state, coordinate flux and characteristic speeds (R2, R3, R6 of
// DESIGN.md; eqs (13), (18), (20)-(22), (37) of PAPER.md:102-133, 266) and the HLLE / LxF
// combination (R7; eqs (29), (30) PAPER.md:196-203), written for a low FP64-pipe instruction
// count: everything a side needs is formed once, the speeds use one reciprocal and one
// square root per side, the face needs one reciprocal square root of det(gamma).
#pragma once
#include "phys.cuh"

namespace gk {

// 1/x to full double precision (<= 1 ulp, not correctly rounded): hardware seed
// (MUFU.RCP64H, ~2^-20) + two Newton steps.  x must be a normal, finite, non-zero number.
__device__ __forceinline__ double rcp_nr(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  return r;
}

// Rows of a face state: 0 D, 1-3 S_j, 4 tau, 5 and 6 the two transverse B components
// B^{(D+1)%3}, B^{(D+2)%3}.
template <int D>
__device__ __forceinline__ void side_rows(double rho, double vx, double vy, double vz, double p,
                                          double Bx, double By, double Bz, const Met& M,
                                          double gdd, const Eos& E, double U[7], double Gf[7],
                                          double& lm, double& lp) {
  // R5 (last part): floors and the velocity cap on the reconstructed state
  rho = rho < E.rho_atm ? E.rho_atm : rho;
  p = p < E.p_floor ? E.p_floor : p;
  double vlx, vly, vlz;
  lower(M, vx, vy, vz, vlx, vly, vlz);  // v_i = gamma_ij v^j
  double v2 = vlx * vx + vly * vy + vlz * vz;
  if (v2 > E.v2max) {  // rare
    const double f = sqrt(E.v2max / v2);
    vx *= f; vy *= f; vz *= f;
    lower(M, vx, vy, vz, vlx, vly, vlz);
    v2 = vlx * vx + vly * vy + vlz * vz;
  }
  double Blx, Bly, Blz;
  lower(M, Bx, By, Bz, Blx, Bly, Blz);  // B_i
  const double B2 = Blx * Bx + Bly * By + Blz * Bz;
  const double Bv = Bx * vlx + By * vly + Bz * vlz;
  const double iW2 = 1.0 - v2;
  const double W = rsqrt(iW2);          // W = (1 - v^2)^(-1/2)
  const double iW = iW2 * W;
  const double ab0 = W * Bv;            // alpha b^0, eq. (13)
  const double b2 = (B2 + ab0 * ab0) * iW2;
  const double blx = Blx * iW + ab0 * vlx;  // b_i, eq. (37)
  const double bly = Bly * iW + ab0 * vly;
  const double blz = Blz * iW + ab0 * vlz;
  const double rhoh = rho + E.GoGm1 * p;    // eq. (46) with h = 1 + eps + p/rho
  const double e = rhoh + b2;
  const double eW2 = e * W * W;
  const double ptot = p + 0.5 * b2;
  // eqs (20)-(22)
  U[0] = rho * W;
  U[1] = eW2 * vlx - ab0 * blx;
  U[2] = eW2 * vly - ab0 * bly;
  U[3] = eW2 * vlz - ab0 * blz;
  U[4] = eW2 - ptot - ab0 * ab0 - U[0];
  // coordinate flux G = alpha F^D of eq. (18) (reading G10); v~^i = alpha v^i - beta^i
  const double vtx = M.a * vx - M.bx, vty = M.a * vy - M.by, vtz = M.a * vz - M.bz;
  const double vtd = D == 0 ? vtx : (D == 1 ? vty : vtz);
  const double vd = D == 0 ? vx : (D == 1 ? vy : vz);
  const double Bd = D == 0 ? Bx : (D == 1 ? By : Bz);
  const double aBdW = M.a * Bd * iW;
  const double ap = M.a * ptot;
  Gf[0] = U[0] * vtd;
  Gf[1] = U[1] * vtd - blx * aBdW + (D == 0 ? ap : 0.0);
  Gf[2] = U[2] * vtd - bly * aBdW + (D == 1 ? ap : 0.0);
  Gf[3] = U[3] * vtd - blz * aBdW + (D == 2 ? ap : 0.0);
  Gf[4] = U[4] * vtd + ap * vd - ab0 * aBdW;
  const double B1 = D == 0 ? By : (D == 1 ? Bz : Bx);
  const double B2t = D == 0 ? Bz : (D == 1 ? Bx : By);
  const double vt1 = D == 0 ? vty : (D == 1 ? vtz : vtx);
  const double vt2 = D == 0 ? vtz : (D == 1 ? vtx : vty);
  U[5] = B1; U[6] = B2t;
  Gf[5] = B1 * vtd - Bd * vt1;
  Gf[6] = B2t * vtd - Bd * vt2;
  // R6 / G9 over one denominator: a^2 = N/Dn, N = Gamma p e + b^2 (rho h - Gamma p),
  // Dn = rho h e;  lambda_pm = alpha (v^d (Dn-N) +- sqrt(N (1-v^2) (g^dd (Dn - v^2 N)
  //                                  - (v^d)^2 (Dn-N)))) / (Dn - v^2 N) - beta^d
  const double Gp = E.Gamma * p;
  const double N = Gp * e + b2 * (rhoh - Gp);
  const double Dn = rhoh * e;
  const double DmN = Dn - N;
  const double den = Dn - v2 * N;
  double rad = N * iW2 * (gdd * den - vd * vd * DmN);
  rad = rad < 0.0 ? 0.0 : rad;
  const double root = sqrt(rad);
  const double aod = M.a * rcp_nr(den);
  const double mid = vd * DmN;
  const double bd = D == 0 ? M.bx : (D == 1 ? M.by : M.bz);
  lm = aod * (mid - root) - bd;
  lp = aod * (mid + root) - bd;
}

// R7: out[r] = sqrt(gamma_f) * F^[r] for the 7 stored rows.
__device__ __forceinline__ void hll_rows(const double UL[7], const double GL[7], double lmL,
                                         double lpL, const double UR[7], const double GR[7],
                                         double lmR, double lpR, double sgf, int riemann,
                                         double out[7]) {
  const double cmax = fmax(0.0, fmax(lpL, lpR));
  const double cmin = -fmin(0.0, fmin(lmL, lmR));
  if (riemann == 1) {  // eq. (30)
    const double cw = fmax(cmax, cmin);
    const double hs = 0.5 * sgf;
#pragma unroll
    for (int r = 0; r < 7; r++) out[r] = hs * (GR[r] + GL[r] - cw * (UR[r] - UL[r]));
  } else if (cmax + cmin < 1e-300) {
    const double hs = 0.5 * sgf;
#pragma unroll
    for (int r = 0; r < 7; r++) out[r] = hs * (GL[r] + GR[r]);
  } else {  // eq. (29)
    const double w = sgf * rcp_nr(cmax + cmin);
    const double cc = cmax * cmin;
#pragma unroll
    for (int r = 0; r < 7; r++)
      out[r] = (cmin * GR[r] + cmax * GL[r] - cc * (UR[r] - UL[r])) * w;
  }
}

}  // namespace gk

// phys.cuh -- per-point device arithmetic of the GRMHD substep (fp64, sm_100a).
//
// Everything here is a restatement, in register-friendly form, of formulas printed in the
// AsterX paper (arXiv 2406.11669; PAPER.md) or of the readings listed in DESIGN.md
// (R-rows = algorithm steps, G-rows = readings where the paper is silent).  No code is
// shared with oracle/ (the CPU checker); the two are compared by tests/ only.
//
// Conventions: prim = (rho, v^x, v^y, v^z, p, B^x, B^y, B^z) with Eulerian v^i, B^i
// (PAPER.md:98-105); metric = (alpha, beta^i, gamma_ij); cons = undensitised
// (D, S_j, tau, B^k) of eqs (20)-(22).
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace gk {

struct Met {
  double a, bx, by, bz, gxx, gxy, gxz, gyy, gyz, gzz;
};

struct Prim {
  double rho, vx, vy, vz, p, Bx, By, Bz;
};

// Constant options of a handle, passed by value to kernels.
struct Eos {
  double Gamma;     // ideal-fluid index, eq. (46)
  double GoGm1;     // Gamma/(Gamma-1):  rho h = rho + GoGm1 p  (h = 1+eps+p/rho)
  double gm1oG;     // (Gamma-1)/Gamma
  double rho_atm;
  double p_atm;     // max(K rho_atm^Gamma_p, p_floor), eqs (47)-(48) PAPER.md:340-342
  double p_floor;
  double v2max;     // 1 - 1/w_max^2 (G20)
  double c2p_tol;
  int c2p_maxit;
  int recon;        // 0 minmod, 1 PPM
  int flatten;
  int riemann;      // 0 HLLE eq. (29), 1 LxF eq. (30)
  int gauge;        // 0 algebraic gauge, 1 generalised Lorenz gauge (eqs 31-32)
  double lorenz_xi; // xi = lorenz_xi / dt
  int emf;          // 0 flux-CT (R10), 1 upwind CT (eqs 33-35)
  int c2p_backup;   // 1: 1-D scheme when the 2-D Newton iteration fails
};

__device__ __forceinline__ double sq(double x) { return x * x; }

// ---- special functions without special-case paths ----------------------------------------
// 1/x: hardware seed (2^-23) + two Newton steps; x normal, finite, non-zero.
__device__ __forceinline__ double ft_rcp(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  return r;
}
// x^(-1/2): hardware seed + two Newton steps (y <- y + y/2 (1 - x y^2)); x normal, > 0.
__device__ __forceinline__ double ft_rsqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double t = x * y;
  double e = fma(-t, y, 1.0);
  y = fma(0.5 * y, e, y);
  t = x * y;
  e = fma(-t, y, 1.0);
  y = fma(0.5 * y, e, y);
  return y;
}
// sqrt(x) for x >= 0 (0 below 1e-280): one Newton step on the seed (relative error e ~ 2^-43),
// s = x y, then one step with the residual x - s^2, which leaves e^2.
__device__ __forceinline__ double ft_sqrt(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double t = x * y;
  const double e = fma(-t, y, 1.0);
  y = fma(0.5 * y, e, y);
  double s = x * y;
  const double r = fma(-s, s, x);
  s = fma(0.5 * y, r, s);
  return x > 1e-280 ? s : 0.0;
}

// a and b have different signs (sign bits; a zero counts with its sign bit)
__device__ __forceinline__ bool ft_opposite(double a, double b) {
  return (__double2hiint(a) ^ __double2hiint(b)) < 0;
}


__device__ __forceinline__ double det_gamma(const Met& M) {
  return M.gxx * (M.gyy * M.gzz - M.gyz * M.gyz) - M.gxy * (M.gxy * M.gzz - M.gyz * M.gxz) +
         M.gxz * (M.gxy * M.gyz - M.gyy * M.gxz);
}

// upper metric gamma^{ij} (6 components), given 1/det
struct Sym3 {
  double xx, xy, xz, yy, yz, zz;
};
__device__ __forceinline__ Sym3 inv_gamma(const Met& M, double idet) {
  Sym3 u;
  u.xx = (M.gyy * M.gzz - M.gyz * M.gyz) * idet;
  u.xy = (M.gxz * M.gyz - M.gxy * M.gzz) * idet;
  u.xz = (M.gxy * M.gyz - M.gxz * M.gyy) * idet;
  u.yy = (M.gxx * M.gzz - M.gxz * M.gxz) * idet;
  u.yz = (M.gxz * M.gxy - M.gxx * M.gyz) * idet;
  u.zz = (M.gxx * M.gyy - M.gxy * M.gxy) * idet;
  return u;
}

// gamma^{dd} only (R4: the speeds along d need nothing else of the inverse)
template <int D>
__device__ __forceinline__ double inv_gamma_dd(const Met& M, double idet) {
  if (D == 0) return (M.gyy * M.gzz - M.gyz * M.gyz) * idet;
  if (D == 1) return (M.gxx * M.gzz - M.gxz * M.gxz) * idet;
  return (M.gxx * M.gyy - M.gxy * M.gxy) * idet;
}

__device__ __forceinline__ void lower(const Met& M, double x, double y, double z, double& lx,
                                      double& ly, double& lz) {
  lx = M.gxx * x + M.gxy * y + M.gxz * z;
  ly = M.gxy * x + M.gyy * y + M.gyz * z;
  lz = M.gxz * x + M.gyz * y + M.gzz * z;
}

// min / max as one compare + select (no NaN bookkeeping)
__device__ __forceinline__ double ft_min(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double ft_max(double a, double b) { return a > b ? a : b; }

// ---------------------------------------------------------------------------------------
// Point state shared by eqs (13), (20)-(22), (37): PAPER.md:102, 129-133, 266.
struct Pt {
  double W, iW, v2, vlx, vly, vlz, ab0, b2, blx, bly, blz, rhoh;
};

__device__ __forceinline__ Pt point_state(const Prim& P, const Met& M, const Eos& E) {
  Pt s;
  double Blx, Bly, Blz;
  lower(M, P.vx, P.vy, P.vz, s.vlx, s.vly, s.vlz);   // v_i = gamma_ij v^j
  lower(M, P.Bx, P.By, P.Bz, Blx, Bly, Blz);         // B_i
  s.v2 = s.vlx * P.vx + s.vly * P.vy + s.vlz * P.vz;
  const double B2 = Blx * P.Bx + Bly * P.By + Blz * P.Bz;
  const double Bv = P.Bx * s.vlx + P.By * s.vly + P.Bz * s.vlz;
  const double iW2 = 1.0 - s.v2;
  s.W = ft_rsqrt(iW2);               // W = (1 - v^2)^(-1/2)
  s.iW = iW2 * s.W;                  // 1/W
  s.ab0 = s.W * Bv;                  // alpha b^0 = W B^i v_i, eq. (13)
  s.b2 = (B2 + s.ab0 * s.ab0) * iW2; // b^2 = (B^2 + (alpha b^0)^2)/W^2, eq. (13)
  s.blx = Blx * s.iW + s.ab0 * s.vlx;  // b_i = B_i/W + alpha b^0 v_i, eq. (37)
  s.bly = Bly * s.iW + s.ab0 * s.vly;
  s.blz = Blz * s.iW + s.ab0 * s.vlz;
  s.rhoh = P.rho + E.GoGm1 * P.p;    // rho h for the ideal fluid, eq. (46)
  return s;
}

// R2: eqs (20)-(22); U = (D, S_x, S_y, S_z, tau), undensitised.
__device__ __forceinline__ void prim2con(const Prim& P, const Met& M, const Eos& E,
                                         double U[5]) {
  const Pt s = point_state(P, M, E);
  const double eW2 = (s.rhoh + s.b2) * s.W * s.W;
  U[0] = P.rho * s.W;
  U[1] = eW2 * s.vlx - s.ab0 * s.blx;
  U[2] = eW2 * s.vly - s.ab0 * s.bly;
  U[3] = eW2 * s.vlz - s.ab0 * s.blz;
  U[4] = eW2 - (P.p + 0.5 * s.b2) - s.ab0 * s.ab0 - U[0];
}

// R6 / G9: fast-magnetosonic bound of the characteristic speeds along direction D.
// a^2 = c_s^2 + v_A^2 - c_s^2 v_A^2 written over one denominator.
template <int D>
__device__ __forceinline__ void char_speeds(const Prim& P, const Pt& s, const Met& M, double gdd,
                                            const Eos& E, double& lm, double& lp) {
  const double e = s.rhoh + s.b2;
  const double Gp = E.Gamma * P.p;
  const double a2 = (Gp * e + s.b2 * (s.rhoh - Gp)) * ft_rcp(s.rhoh * e);
  const double vd = D == 0 ? P.vx : (D == 1 ? P.vy : P.vz);
  const double bd = D == 0 ? M.bx : (D == 1 ? M.by : M.bz);
  const double den = 1.0 - s.v2 * a2;
  double rad = a2 * (1.0 - s.v2) * (gdd * den - vd * vd * (1.0 - a2));
  rad = rad < 0.0 ? 0.0 : rad;
  const double root = ft_sqrt(rad);
  const double aoden = M.a * ft_rcp(den);
  const double mid = vd * (1.0 - a2);
  lm = aoden * (mid - root) - bd;
  lp = aoden * (mid + root) - bd;
}

}  // namespace gk

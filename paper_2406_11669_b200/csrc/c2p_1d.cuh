// c2p_1d.cuh -- row F4: the one-unknown conservative-to-primitive scheme the paper keeps as
// backup for the 2-D Newton iteration (eqs 42-45; backup policy PAPER.md:684).
//
// Written from the paper's steps (i)-(vii) alone, in a form that suits a register-only rare
// path; it shares no statement with the CPU checker in oracle/ (the two are compared by
// tests/ only).  What is computed:
//   (i)   q = tau/D, r = S^2/D^2, s = B^2/D, t^2 = (B.S)^2/D^3                     eq. (42)
//   (ii)  the root x = h W of f(x) = x - h^(x) W^(x) inside 1 + q - s < x < 2 + 2q - s   eq. (43)
//   (iii) 1/W^2 = 1 - [r x^2 + t^2 (2x + s)] / [x^2 (x + s)^2]                      eq. (44)
//   (v)   eps^ = -1 + x (1 - W^2)/W + W [1 + q - s + (t^2/x^2 + s/W^2)/2]           eq. (45)
//   (vii) v^i from eq. (41c) with z = D x
// Readings of DESIGN.md: G23 (eq. 45 prints t^2/x; dividing eq. 40b by D with z = D x gives
// t^2/x^2), G24 (v^2 = 1 - 1/W^2), G25 (lower bracket end raised to 1 since h W >= 1; 1/W^2
// kept in [1/w_max^2, 1]; eps^ >= 0 while iterating; the bracket is closed to a relative
// width of 1e-14 in at most 100 function evaluations; ideal fluid, h^ = 1 + Gamma eps^).
//
// The paper names Brent's technique for (ii).  Any bracketing solver that closes the bracket
// to the same width finds the same x; here it is the quadratic/bisection hybrid of
// Chandrupatla (three points, inverse quadratic interpolation where its two validity
// inequalities hold, bisection otherwise), which needs no step history: the whole solver
// state is three abscissae and three residuals.  Every trial point is kept at least half the
// target width away from both bracket ends, so that a trial landing next to the root steps
// across it and the bracket collapses to the target width instead of creeping.
#pragma once
#include "phys.cuh"

namespace gk {

// eq. (42) in the combinations eqs (44), (45) need (only t^2 occurs: no square root of D)
struct HwResidual {
  double e0;    // 1 + q - s
  double r, s, t2;
  double Gamma;
  double iw2lo; // 1/w_max^2

  // state at x: W^, 1/W^, eps^ (eqs 44, 45); returns f(x) of eq. (43)
  __device__ double at(double x, double& W, double& iW, double& eps) const {
    const double u = 1.0 / x;
    const double w = 1.0 / (x + s);
    const double t2u2 = t2 * u * u;                       // t^2 / x^2
    double iw2 = 1.0 - (r + t2u2 * (2.0 * x + s)) * (w * w);  // eq. (44), divided through by x^2
    iw2 = iw2 < iw2lo ? iw2lo : (iw2 > 1.0 ? 1.0 : iw2);
    iW = sqrt(iw2);
    W = 1.0 / iW;
    // eq. (45) collected by powers of W: x (1 - W^2)/W = x/W - x W
    eps = W * (e0 - x + 0.5 * t2u2) + iW * (x + 0.5 * s) - 1.0;
    eps = eps > 0.0 ? eps : 0.0;
    return x - (1.0 + Gamma * eps) * W;                   // h^ = 1 + Gamma eps^, eq. (46)
  }
};

// U = undensitised (D, S_j, tau).  Returns true and rho, v^i, eps on success; iters = number
// of trial points after the two bracket ends.
__device__ __noinline__ bool con2prim_1d(const double* U, double Bx, double By, double Bz,
                                         const Met& M, const Eos& E, double& rho, double& vx,
                                         double& vy, double& vz, double& eps, int& iters) {
  iters = 0;
  const double D = U[0], tau = U[4];
  // S^i = gamma^{ij} S_j, S^2, B^2 = gamma_ij B^i B^j, B.S
  const Sym3 gu = inv_gamma(M, 1.0 / det_gamma(M));
  const double Sux = gu.xx * U[1] + gu.xy * U[2] + gu.xz * U[3];
  const double Suy = gu.xy * U[1] + gu.yy * U[2] + gu.yz * U[3];
  const double Suz = gu.xz * U[1] + gu.yz * U[2] + gu.zz * U[3];
  const double S2 = Sux * U[1] + Suy * U[2] + Suz * U[3];
  double Blx, Bly, Blz;
  lower(M, Bx, By, Bz, Blx, Bly, Blz);
  const double B2 = Blx * Bx + Bly * By + Blz * Bz;
  const double BS = Bx * U[1] + By * U[2] + Bz * U[3];

  const double iD = 1.0 / D;
  HwResidual h;
  h.r = S2 * iD * iD;
  h.s = B2 * iD;
  h.t2 = BS * BS * iD * iD * iD;
  h.e0 = 1.0 + tau * iD - h.s;
  h.Gamma = E.Gamma;
  h.iw2lo = 1.0 - E.v2max;
  const double xlo = h.e0 > 1.0 ? h.e0 : 1.0;      // bracket of step (ii), lower end >= 1 (G25)
  const double xhi = h.e0 + (1.0 + tau * iD);      // 2 + 2q - s
  if (!(xhi > xlo)) return false;

  double W, iW, ee;
  const double flo = h.at(xlo, W, iW, ee), fhi = h.at(xhi, W, iW, ee);
  double x;
  bool closed = false;
  if (flo == 0.0) { x = xlo; closed = true; }
  else if (fhi == 0.0) { x = xhi; closed = true; }
  else if (!isfinite(flo) || !isfinite(fhi) || (flo < 0.0) == (fhi < 0.0)) return false;

  // a = newest trial point, b = the bracket end on the other side of the root,
  // c = the point the last trial replaced
  double a = xhi, fa = fhi, b = xlo, fb = flo, c = xlo, fc = flo;
  double th = 0.5;  // position of the next trial inside the bracket, from a towards b
  for (int n = 1; n <= 100 && !closed; n++) {
    iters = n;
    const double xt = a + th * (b - a);
    const double ft = h.at(xt, W, iW, ee);
    if (!isfinite(ft)) return false;
    if ((ft < 0.0) == (fa < 0.0)) { c = a; fc = fa; }         // root between xt and b
    else { c = b; fc = fb; b = a; fb = fa; }                  // root between a and xt
    a = xt; fa = ft;
    const bool a_best = fabs(fa) <= fabs(fb);
    x = a_best ? a : b;
    const double width = fabs(b - a);
    const double want = 1e-14 * fabs(x);                      // G25: relative bracket width
    if ((a_best ? fa : fb) == 0.0 || width <= want) { closed = true; break; }
    const double edge = 0.5 * want / width;                   // < 1/2 here
    // inverse quadratic interpolation through (a, b, c) where it is well conditioned
    const double xi = (a - b) / (c - b), ph = (fa - fb) / (fc - fb);
    th = 0.5;
    if (ph * ph < xi && (1.0 - ph) * (1.0 - ph) < 1.0 - xi)
      th = fa / (fb - fa) * (fc / (fb - fc)) + (c - a) / (b - a) * (fa / (fc - fa)) * (fb / (fc - fb));
    th = !(th > edge) ? edge : (th > 1.0 - edge ? 1.0 - edge : th);
  }
  if (!closed || !isfinite(x)) return false;

  h.at(x, W, iW, eps);                 // (iii), (v) at the root
  rho = D * iW;                        // (iv)
  const double z = D * x;              // (vii): z = rho W x
  const double k = 1.0 / (z + B2), m = BS / z;
  vx = (Sux + m * Bx) * k;             // eq. (41c)
  vy = (Suy + m * By) * k;
  vz = (Suz + m * Bz) * k;
  return isfinite(rho) && isfinite(eps) && isfinite(vx) && isfinite(vy) && isfinite(vz);
}

}  // namespace gk

// grmhd_ref.cpp -- the ORACLE: plain fp64 CPU implementation of the AsterX GRMHD substep.
//
// TEST INFRASTRUCTURE, NOT THE PRODUCT (see grmhd_ref.h).  Written from PAPER.md
// (arXiv 2406.11669) step by step, in the paper's notation; where the paper is silent the
// reading taken is the R/G row of DESIGN.md quoted beside the code.  No blocking, fusion
// or reordering: every face flux and every edge field is evaluated where it is defined.
// Compile with -O2 -ffp-contract=off (no FMA contraction).  The optional OpenMP pragmas
// sit on outer cell loops only; results are bit-identical for any thread count (cells are
// independent, the max reduction is exact, counters are integer sums).
//
// Pins (tests/, -m "not gpu"): P1 round trip, P2 uniform state on a constant metric,
// P3 conservation, P4 symmetry, P5 Alfven/entropy-wave convergence,
// P6 curl/div/flux-CT identities, P7 HLLE consistency, P8 reconstruction properties,
// P9 speeds closed forms, P10 con2prim closed forms, P11 sources vs brute-force 4-D
// Christoffels, P12 naive re-evaluation on 4^3 blocks, P13 constant-metric advection,
// P14 Rindler hydrostatic equilibrium, P15 the 1-D backup con2prim (eqs 42-45), P16 upwind CT
// (eqs 33-35), P17 the generalised Lorenz gauge (eqs 31-32); and by hand-worked numbers
// (tests/test_oracle_pins2.py): R16 max speed / dt / step_until clipping, R12 temporal order
// 2 / 3 / 4 of the RK tableaux, R15 linear continuation of A_i, R5 face floors and velocity cap,
// G16 static face field on a varying metric, G8(c) flattening between its ends, R7 HLLE,
// F2 Lax-Friedrichs (eq. 30).
// Parity UNPINNED by the paper: the PPM variant (G8) and the characteristic-speed bound (G9)
// are readings of citations that are not in PAPER.md; they are pinned only by the
// mathematical properties P8/P9.
#include "grmhd_ref.h"

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int G = 3;  // ghost zones

int g_threads = 1;

inline double sq(double x) { return x * x; }

// ----------------------------------------------------------------------------- metric
struct Metric {
  double alpha;
  double beta[3];
  double g[3][3];  // gamma_ij
};

Metric unpack_metric(const double m[10]) {
  Metric M;
  M.alpha = m[0];
  M.beta[0] = m[1]; M.beta[1] = m[2]; M.beta[2] = m[3];
  M.g[0][0] = m[4]; M.g[0][1] = M.g[1][0] = m[5]; M.g[0][2] = M.g[2][0] = m[6];
  M.g[1][1] = m[7]; M.g[1][2] = M.g[2][1] = m[8]; M.g[2][2] = m[9];
  return M;
}

double det3(const double g[3][3]) {
  return g[0][0] * (g[1][1] * g[2][2] - g[1][2] * g[2][1]) -
         g[0][1] * (g[1][0] * g[2][2] - g[1][2] * g[2][0]) +
         g[0][2] * (g[1][0] * g[2][1] - g[1][1] * g[2][0]);
}

void inv3(const double g[3][3], double det, double u[3][3]) {
  u[0][0] = (g[1][1] * g[2][2] - g[1][2] * g[2][1]) / det;
  u[0][1] = (g[0][2] * g[2][1] - g[0][1] * g[2][2]) / det;
  u[0][2] = (g[0][1] * g[1][2] - g[0][2] * g[1][1]) / det;
  u[1][1] = (g[0][0] * g[2][2] - g[0][2] * g[2][0]) / det;
  u[1][2] = (g[0][2] * g[1][0] - g[0][0] * g[1][2]) / det;
  u[2][2] = (g[0][0] * g[1][1] - g[0][1] * g[1][0]) / det;
  u[1][0] = u[0][1]; u[2][0] = u[0][2]; u[2][1] = u[1][2];
}

// ------------------------------------------------------------------------------- EOS
// R1: ideal fluid p = (Gamma-1) rho eps, eq. (46); h = 1 + eps + p/rho
// => rho h = rho + Gamma/(Gamma-1) p.
inline double rho_h(double rho, double p, double Gamma) {
  const double eps = p / ((Gamma - 1.0) * rho);
  return rho * (1.0 + eps) + p;
}

// ------------------------------------------------------------------------ prim -> cons
// Quantities shared by eqs (13),(20)-(22),(37): everything a point state defines.
struct PointState {
  double W, vlow[3], v2, Blow[3], B2, Bv, ab0, b2, blow[3], rhoh;
};

PointState point_state(const double P[8], const Metric& M, double Gamma) {
  PointState s;
  const double* v = P + 1;
  const double* B = P + 5;
  s.v2 = 0; s.B2 = 0; s.Bv = 0;
  for (int i = 0; i < 3; i++) {
    s.vlow[i] = 0; s.Blow[i] = 0;
    for (int j = 0; j < 3; j++) {
      s.vlow[i] += M.g[i][j] * v[j];  // v_i = gamma_ij v^j
      s.Blow[i] += M.g[i][j] * B[j];  // B_i
    }
  }
  for (int i = 0; i < 3; i++) {
    s.v2 += s.vlow[i] * v[i];
    s.B2 += s.Blow[i] * B[i];
    s.Bv += B[i] * s.vlow[i];
  }
  s.W = 1.0 / std::sqrt(1.0 - s.v2);       // W = (1 - v^i v_i)^(-1/2)
  s.ab0 = s.W * s.Bv;                       // alpha b^0 = W B^i v_i, eq. (13)
  s.b2 = (s.B2 + sq(s.ab0)) / sq(s.W);      // b^2 = (B^2 + (alpha b^0)^2)/W^2, eq. (13)
  for (int i = 0; i < 3; i++) s.blow[i] = s.Blow[i] / s.W + s.ab0 * s.vlow[i];  // eq. (37)
  s.rhoh = rho_h(P[0], P[4], Gamma);
  return s;
}

// R2: eqs (20)-(22); undensitised U = (D, S_j, tau, B^k).
void prim2con(const double P[8], const Metric& M, double Gamma, double U[8]) {
  const PointState s = point_state(P, M, Gamma);
  const double W2 = sq(s.W);
  U[0] = P[0] * s.W;                                                        // (20)
  for (int j = 0; j < 3; j++)
    U[1 + j] = (s.rhoh + s.b2) * W2 * s.vlow[j] - s.ab0 * s.blow[j];        // (21)
  U[4] = (s.rhoh + s.b2) * W2 - (P[4] + 0.5 * s.b2) - sq(s.ab0) - U[0];     // (22)
  U[5] = P[5]; U[6] = P[6]; U[7] = P[7];
}

// R3: flux vector F^d of eq. (18), exactly as printed (with its 1/alpha).
void flux18(int d, const double P[8], const Metric& M, double Gamma, double F[8]) {
  const PointState s = point_state(P, M, Gamma);
  double U[8];
  prim2con(P, M, Gamma, U);
  const double* v = P + 1;
  const double* B = P + 5;
  double vt[3];
  for (int i = 0; i < 3; i++) vt[i] = M.alpha * v[i] - M.beta[i];  // v~^i
  const double ptot = P[4] + 0.5 * s.b2;
  F[0] = U[0] * vt[d] / M.alpha;
  for (int j = 0; j < 3; j++)
    F[1 + j] = U[1 + j] * vt[d] / M.alpha + (j == d ? ptot : 0.0) - s.blow[j] * B[d] / s.W;
  F[4] = U[4] * vt[d] / M.alpha + ptot * v[d] - s.ab0 * B[d] / s.W;
  for (int k = 0; k < 3; k++) F[5 + k] = B[k] * vt[d] / M.alpha - B[d] * vt[k] / M.alpha;
}

// R6 / G9: closed-form fast-magnetosonic bound for the characteristic speeds along d.
// gdd = gamma^{dd}.  lam[0] = lambda_-, lam[1] = lambda_+.
void speeds(int d, const double P[8], const Metric& M, double gdd, double Gamma,
            double lam[2]) {
  const PointState s = point_state(P, M, Gamma);
  const double cs2 = Gamma * P[4] / s.rhoh;
  const double va2 = s.b2 / (s.rhoh + s.b2);
  const double a2 = cs2 + va2 - cs2 * va2;
  const double vd = P[1 + d];
  const double den = 1.0 - s.v2 * a2;
  double rad = a2 * (1.0 - s.v2) * (gdd * den - sq(vd) * (1.0 - a2));
  if (rad < 0.0) rad = 0.0;
  const double root = std::sqrt(rad);
  lam[0] = M.alpha * (vd * (1.0 - a2) - root) / den - M.beta[d];
  lam[1] = M.alpha * (vd * (1.0 - a2) + root) / den - M.beta[d];
}

// R5 (last part): floors and velocity cap applied to a reconstructed face state.
void face_floors(double P[8], const Metric& M, const ref_opts& o) {
  if (P[0] < o.rho_atm) P[0] = o.rho_atm;
  if (P[4] < o.p_floor) P[4] = o.p_floor;
  double v2 = 0;
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) v2 += M.g[i][j] * P[1 + i] * P[1 + j];
  const double v2max = 1.0 - 1.0 / sq(o.w_max);
  if (v2 > v2max) {
    const double f = std::sqrt(v2max / v2);
    for (int i = 0; i < 3; i++) P[1 + i] *= f;
  }
}

// R7: HLLE eq. (29) PAPER.md:196 (riemann = 0) or LxF eq. (30) PAPER.md:203 (riemann = 1).
// G10: the flux paired with the coordinate speeds is G = alpha_f F^d.  Returns F^ (not yet
// multiplied by sqrt(gamma_f)).
// `uct` (optional, 4 values): what the upwind constrained transport of PAPER.md:229-250 needs
// from this face -- a_+ and a_- of eq. (34) and the upwind transverse velocities of eq. (33),
// vbar^j = (a_+ v~^jL + a_- v~^jR)/(a_+ + a_-) for j = (d+1)%3, (d+2)%3 (their mean when
// a_+ + a_- vanishes), v~^j = alpha v^j - beta^j with the face metric.
void riemann(int d, const double PL_in[8], const double PR_in[8], const Metric& M,
             const ref_opts& o, double Fhat[8], double* uct = nullptr) {
  double PL[8], PR[8];
  std::memcpy(PL, PL_in, sizeof PL);
  std::memcpy(PR, PR_in, sizeof PR);
  face_floors(PL, M, o);
  face_floors(PR, M, o);
  double gu[3][3];
  inv3(M.g, det3(M.g), gu);
  double UL[8], UR[8], FL[8], FR[8], lamL[2], lamR[2];
  prim2con(PL, M, o.gamma_ad, UL);
  prim2con(PR, M, o.gamma_ad, UR);
  flux18(d, PL, M, o.gamma_ad, FL);
  flux18(d, PR, M, o.gamma_ad, FR);
  speeds(d, PL, M, gu[d][d], o.gamma_ad, lamL);
  speeds(d, PR, M, gu[d][d], o.gamma_ad, lamR);
  const double cmax = std::max(0.0, std::max(lamL[1], lamR[1]));
  const double cmin = -std::min(0.0, std::min(lamL[0], lamR[0]));
  for (int r = 0; r < 8; r++) {
    const double GL = M.alpha * FL[r], GR = M.alpha * FR[r];
    if (o.riemann == 1) {
      const double cw = std::max(cmax, cmin);
      Fhat[r] = 0.5 * (GR + GL - cw * (UR[r] - UL[r]));
    } else if (cmax + cmin < 1e-300) {
      Fhat[r] = 0.5 * (GL + GR);
    } else {
      Fhat[r] = (cmin * GR + cmax * GL - cmax * cmin * (UR[r] - UL[r])) / (cmax + cmin);
    }
  }
  Fhat[5 + d] = 0.0;  // the B^d row of eq. (18) vanishes identically
  if (uct) {
    uct[0] = cmax;  // eq. (34): a_+ = max{0, lambda_+(U^L), lambda_+(U^R)}
    uct[1] = cmin;  //           a_- = max{0, -lambda_-(U^L), -lambda_-(U^R)}
    for (int t = 0; t < 2; t++) {
      const int j = (d + 1 + t) % 3;
      const double vL = M.alpha * PL[1 + j] - M.beta[j], vR = M.alpha * PR[1 + j] - M.beta[j];
      uct[2 + t] = cmax + cmin < 1e-300 ? 0.5 * (vL + vR)
                                        : (cmax * vL + cmin * vR) / (cmax + cmin);  // eq. (33)
    }
  }
}

// eq. (35), one bracket: [a_+ v^L B^L + a_- v^R B^R - a_+ a_- (B^R - B^L)]/(a_+ + a_-)
inline double uct_bracket(double ap, double am, double vL, double vR, double BL, double BR) {
  if (ap + am < 1e-300) return 0.5 * (vL * BL + vR * BR);
  return (ap * vL * BL + am * vR * BR - ap * am * (BR - BL)) / (ap + am);
}

// ---------------------------------------------------------------------- reconstruction
// R5 / G7: minmod(a,b) = 0 if a*b <= 0 else sign(a) min(|a|,|b|).
inline double minmod(double a, double b) {
  if (a * b <= 0.0) return 0.0;
  const double m = std::min(std::fabs(a), std::fabs(b));
  return a > 0.0 ? m : -m;
}

// q[0..2] = q_{i-1}, q_i, q_{i+1}: qm = q^R_{i-1/2}, qp = q^L_{i+1/2}.
void minmod_cell(const double q[3], double& qm, double& qp) {
  const double s = minmod(q[1] - q[0], q[2] - q[1]);
  qp = q[1] + 0.5 * s;
  qm = q[1] - 0.5 * s;
}

// G8(a): monotonised central slope of cell i from q_{i-1}, q_i, q_{i+1}.
inline double ppm_dm(double qm1, double q0, double qp1) {
  const double dp = qp1 - q0, dm = q0 - qm1;
  if (dp * dm > 0.0) {
    const double d = 0.5 * (qp1 - qm1);
    const double lim = std::min(std::fabs(d), std::min(2.0 * std::fabs(dp), 2.0 * std::fabs(dm)));
    return d > 0.0 ? lim : -lim;
  }
  return 0.0;
}

// G8(c): flattening coefficient of cell i from p_{i-2..i+2} and v^d_{i-1}, v^d_{i+1}.
double ppm_flat(const double p[5], double vm1, double vp1) {
  const double dp1 = p[3] - p[1];
  const double dp2 = p[4] - p[0];
  if (std::fabs(dp1) > 0.33 * std::min(p[3], p[1]) && vm1 > vp1) {
    if (dp2 == 0.0) return 1.0;
    const double f = 10.0 * (dp1 / dp2 - 0.75);
    return std::min(1.0, std::max(0.0, f));
  }
  return 0.0;
}

// G8(a,b,c,d,e): PPM parabola of cell i from q[0..4] = q_{i-2..i+2}; f = flattening
// coefficient of cell i.  qm = q^-_i = q^R_{i-1/2}, qp = q^+_i = q^L_{i+1/2}.
void ppm_cell(const double q[5], double f, double& qm, double& qp) {
  const double dm_m = ppm_dm(q[0], q[1], q[2]);
  const double dm_0 = ppm_dm(q[1], q[2], q[3]);
  const double dm_p = ppm_dm(q[2], q[3], q[4]);
  qm = 0.5 * (q[1] + q[2]) - (dm_0 - dm_m) / 6.0;  // q_{i-1/2}
  qp = 0.5 * (q[2] + q[3]) - (dm_p - dm_0) / 6.0;  // q_{i+1/2}
  const double q0 = q[2];
  qp = f * q0 + (1.0 - f) * qp;
  qm = f * q0 + (1.0 - f) * qm;
  if ((qp - q0) * (q0 - qm) <= 0.0) {
    qp = q0; qm = q0;
  } else {
    const double D = qp - qm;
    const double m = q0 - 0.5 * (qp + qm);
    if (D * m > D * D / 6.0) qm = 3.0 * q0 - 2.0 * qp;
    else if (-D * D / 6.0 > D * m) qp = 3.0 * q0 - 2.0 * qm;
  }
}

// Reconstruct the L and R states at a face from the 6 cells around it: c[v][0..5] are cells
// f-3..f+2 of variable v (rho,vx,vy,vz,p,Bx,By,Bz).  L comes from cell f-1, R from cell f.
void recon_face(int d, const double c[8][6], const ref_opts& o, double PL[8], double PR[8]) {
  if (o.recon == 0) {
    for (int v = 0; v < 8; v++) {
      double qm, qp;
      minmod_cell(&c[v][1], qm, qp);  // cell f-1: cells f-2,f-1,f
      PL[v] = qp;
      minmod_cell(&c[v][2], qm, qp);  // cell f: cells f-1,f,f+1
      PR[v] = qm;
    }
  } else {
    double fL = 0.0, fR = 0.0;
    if (o.ppm_flatten) {
      fL = ppm_flat(&c[4][0], c[1 + d][1], c[1 + d][3]);  // cell f-1
      fR = ppm_flat(&c[4][1], c[1 + d][2], c[1 + d][4]);  // cell f
    }
    for (int v = 0; v < 8; v++) {
      double qm, qp;
      ppm_cell(&c[v][0], fL, qm, qp);
      PL[v] = qp;
      ppm_cell(&c[v][1], fR, qm, qp);
      PR[v] = qm;
    }
  }
}

// ------------------------------------------------------- con2prim, 1-D backup scheme (F4)
// Palenzuela et al. 1-D scheme: eqs (42)-(45), unknown x = h W, root of
// eq. (43) f(x) = x - h^ W^ bracketed by 1 + q - s < x < 2 + 2q - s and found with Brent's
// method (bracketing; no derivative).  Ideal fluid only (eq. 46), so Y_e of eq. (43) is unused.
// Readings (G23-G25): eq. (45) prints t^2/x where the reduction of eq. (40b) gives
// t^2/x^2 (z = D x); PAPER.md:315 prints "v^2 = 1 1/W^2" for v^2 = 1 - 1/W^2; 1/W^2 of eq. (44)
// is kept inside [1/w_max^2, 1] and eps^ is not allowed below 0 while iterating; the lower
// end of the bracket is raised to 1 when 1 + q - s < 1 (h W >= 1 always).
struct C2P1D {
  double q, r, s, t, D, Gamma, iw2min;
  // eq. (44): 1/W^2 from x
  double w2inv(double x) const {
    double v = 1.0 - (r * x * x + t * t * (2.0 * x + s)) / (x * x * sq(x + s));
    return std::min(std::max(v, iw2min), 1.0);
  }
  // eqs (44), (45): W^, eps^ from x
  void state(double x, double& W, double& eps) const {
    const double iw2 = w2inv(x);
    W = 1.0 / std::sqrt(iw2);
    eps = -1.0 + x / W * (1.0 - W * W) +
          W * (1.0 + q - s + 0.5 * (t * t / (x * x) + s * iw2));
    eps = std::max(eps, 0.0);
  }
  // eq. (43) with h^ = 1 + eps^ + p^/rho^ = 1 + Gamma eps^ (eq. 46)
  double f(double x) const {
    double W, eps;
    state(x, W, eps);
    return x - (1.0 + Gamma * eps) * W;
  }
};

// Brent's method on [a, b] with f(a) f(b) < 0: inverse quadratic interpolation / secant steps
// accepted only while they stay well inside the bracket and shrink fast enough, bisection
// otherwise.  Returns false if the root is not bracketed or maxit is exceeded.
template <class F>
bool brent(const F& f, double a, double b, double rtol, int maxit, double& root, int& iters) {
  double fa = f(a), fb = f(b);
  iters = 0;
  if (!(fa * fb < 0.0)) {
    if (fa == 0.0) { root = a; return true; }
    if (fb == 0.0) { root = b; return true; }
    return false;
  }
  double c = a, fc = fa, d = b - a, e = d;
  for (int it = 1; it <= maxit; it++) {
    iters = it;
    if ((fb > 0.0) == (fc > 0.0)) { c = a; fc = fa; d = b - a; e = d; }  // keep the root in [b, c]
    if (std::fabs(fc) < std::fabs(fb)) { a = b; b = c; c = a; fa = fb; fb = fc; fc = fa; }
    const double tol1 = 2.0 * 2.220446049250313e-16 * std::fabs(b) + 0.5 * rtol * std::fabs(b);
    const double xm = 0.5 * (c - b);
    if (std::fabs(xm) <= tol1 || fb == 0.0) { root = b; return true; }
    if (std::fabs(e) >= tol1 && std::fabs(fa) > std::fabs(fb)) {
      const double sv = fb / fa;
      double pp, qq;
      if (a == c) {  // secant
        pp = 2.0 * xm * sv;
        qq = 1.0 - sv;
      } else {  // inverse quadratic interpolation
        const double qa = fa / fc, rr = fb / fc;
        pp = sv * (2.0 * xm * qa * (qa - rr) - (b - a) * (rr - 1.0));
        qq = (qa - 1.0) * (rr - 1.0) * (sv - 1.0);
      }
      if (pp > 0.0) qq = -qq;
      pp = std::fabs(pp);
      if (2.0 * pp < std::min(3.0 * xm * qq - std::fabs(tol1 * qq), std::fabs(e * qq))) {
        e = d; d = pp / qq;
      } else {
        d = xm; e = d;
      }
    } else {
      d = xm; e = d;
    }
    a = b; fa = fb;
    b += std::fabs(d) > tol1 ? d : (xm > 0.0 ? tol1 : -tol1);
    fb = f(b);
  }
  return false;
}

// Steps (i)-(vii) of PAPER.md:299-320.  In: undensitised D, S_j, tau, B^i, metric.
// Out: rho, v^i, eps.  Returns false on failure (no bracket, no convergence, non-finite).
bool con2prim_1d(const double Uin[5], const double B[3], const Metric& M, const ref_opts& o,
                 double& rho, double v[3], double& eps, int* iters_out) {
  const double D = Uin[0], tau = Uin[4];
  const double* S = Uin + 1;
  double gu[3][3];
  inv3(M.g, det3(M.g), gu);
  double S2 = 0, B2 = 0, BS = 0;
  for (int i = 0; i < 3; i++) {
    for (int j = 0; j < 3; j++) {
      S2 += gu[i][j] * S[i] * S[j];
      B2 += M.g[i][j] * B[i] * B[j];
    }
    BS += B[i] * S[i];
  }
  C2P1D c;  // eq. (42)
  c.D = D; c.Gamma = o.gamma_ad; c.iw2min = 1.0 / sq(o.w_max);
  c.q = tau / D; c.r = S2 / (D * D); c.s = B2 / D; c.t = BS / (D * std::sqrt(D));
  const double lo = std::max(1.0 + c.q - c.s, 1.0), hi = 2.0 + 2.0 * c.q - c.s;
  int it = 0;
  double x = 0;
  const bool ok = hi > lo && brent([&](double xx) { return c.f(xx); }, lo, hi, 1e-14, 100, x, it);
  if (iters_out) *iters_out = it;
  if (!ok || !std::isfinite(x)) return false;
  double W;
  c.state(x, W, eps);          // (iii), (v)
  rho = D / W;                 // (iv)
  const double z = D * x;      // (vii): z = rho W x = rho h W^2
  for (int i = 0; i < 3; i++) {
    double Su = 0;
    for (int j = 0; j < 3; j++) Su += gu[i][j] * S[j];
    v[i] = Su / (z + B2) + BS * B[i] / (z * (z + B2));  // eq. (41c)
  }
  return std::isfinite(rho) && std::isfinite(eps) && std::isfinite(v[0]) &&
         std::isfinite(v[1]) && std::isfinite(v[2]);
}

// ------------------------------------------------------------------------- con2prim
// R14: Noble et al. 2-D Newton-Raphson on (z, v^2), eqs (36)-(41) PAPER.md:260-295, with
// the atmosphere of PAPER.md:326 and the failure policy G17-G20.
// In: undensitised D,S_j,tau; B^i; metric.  Out: P5 = rho,v^i,p; U5 = D,S_j,tau (rewritten
// when a floor or cap was applied).  Returns status bits.
// `backup`: on a failure of the 2-D scheme try the 1-D scheme above before giving up
// (PAPER.md:684); status bit 16 marks a state recovered that way.
int con2prim(const double Uin[5], const double B[3], const Metric& M, const ref_opts& o,
             bool masked, double P5[5], double U5[5], int* iters_out, bool backup = false) {
  const double Gamma = o.gamma_ad;
  const double p_atm = std::max(o.poly_k * std::pow(o.rho_atm, o.poly_gamma), o.p_floor);
  const double v2max = 1.0 - 1.0 / sq(o.w_max);
  const double v2clamp = 1.0 - 1e-12;  // G18: iteration stays subluminal; the W cap acts after
  int iters = 0;
  auto atmosphere = [&](int bits) {
    // rho = rho_atm, p (and eps) from the polytrope, v = 0, B kept, cons reset.
    double P[8] = {o.rho_atm, 0, 0, 0, p_atm, B[0], B[1], B[2]};
    double U[8];
    prim2con(P, M, Gamma, U);
    for (int r = 0; r < 5; r++) { P5[r] = P[r]; U5[r] = U[r]; }
    if (iters_out) *iters_out = iters;
    return bits;
  };
  for (int r = 0; r < 5; r++) U5[r] = Uin[r];
  const double D = Uin[0], tau = Uin[4];
  const double* S = Uin + 1;
  if (masked || !(D > o.rho_atm)) return atmosphere(1);

  double gu[3][3];
  inv3(M.g, det3(M.g), gu);
  double S2 = 0, B2 = 0, BS = 0;
  for (int i = 0; i < 3; i++) {
    for (int j = 0; j < 3; j++) {
      S2 += gu[i][j] * S[i] * S[j];
      B2 += M.g[i][j] * B[i] * B[j];
    }
    BS += B[i] * S[i];
  }
  const double BS2 = sq(BS);
  const double gm1g = (Gamma - 1.0) / Gamma;

  // G17: stateless initial guess z0 = tau + D, v2 = 0.
  double z = tau + D, v2 = 0.0;
  bool converged = false;
  for (int it = 1; it <= o.c2p_maxit; it++) {
    iters = it;
    const double sw = std::sqrt(1.0 - v2);  // 1/W
    const double p = gm1g * (z * (1.0 - v2) - D * sw);
    const double z2 = z * z, z3 = z2 * z;
    // eqs (40a), (40b)
    const double f1 = v2 * sq(B2 + z) - BS2 * (B2 + 2.0 * z) / z2 - S2;
    const double f2 = tau + D - 0.5 * B2 * (1.0 + v2) + BS2 / (2.0 * z2) - z + p;
    const double J11 = 2.0 * (B2 + z) * (v2 + BS2 / z3);
    const double J12 = sq(B2 + z);
    const double J21 = -BS2 / z3 - 1.0 + gm1g * (1.0 - v2);
    const double J22 = -0.5 * B2 + gm1g * (-z + D / (2.0 * sw));
    const double det = J11 * J22 - J12 * J21;
    const double dz = (f2 * J12 - f1 * J22) / det;
    const double dv = (f1 * J21 - f2 * J11) / det;
    const double zn = std::fabs(z + dz);
    const double vn = std::min(std::max(v2 + dv, 0.0), v2clamp);
    const double err = std::fabs(dz) / zn + std::fabs(dv);  // G18
    z = zn; v2 = vn;
    if (!std::isfinite(err)) break;
    if (err < o.c2p_tol) { converged = true; break; }
  }
  bool have = converged && std::isfinite(z) && std::isfinite(v2);
  double rho = 0, v[3] = {0, 0, 0}, eps = 0, p = 0;
  if (have) {
    // eqs (41a)-(41d); G19: the 1/gamma of (41d) is 1/Gamma.
    const double W = 1.0 / std::sqrt(1.0 - v2);
    rho = D / W;
    for (int i = 0; i < 3; i++) {
      double Su = 0;
      for (int j = 0; j < 3; j++) Su += gu[i][j] * S[j];
      v[i] = Su / (z + B2) + BS * B[i] / (z * (z + B2));
    }
    eps = (z / (rho * W * W) - 1.0) / Gamma;
    p = (Gamma - 1.0) * rho * eps;
    have = std::isfinite(rho) && std::isfinite(p) && std::isfinite(v[0]) &&
           std::isfinite(v[1]) && std::isfinite(v[2]) && !(rho < o.rho_atm);
  }
  int bits = 0;
  if (!have) {
    int it1 = 0;
    if (backup && con2prim_1d(Uin, B, M, o, rho, v, eps, &it1) && !(rho < o.rho_atm)) {
      p = (Gamma - 1.0) * rho * eps;
      bits |= 16;
    } else {
      return atmosphere(2);
    }
  }

  bool rewrite = false;
  if (eps < 0.0 || p < o.p_floor) {  // G20 (ii): pressure fix, keep rho and v
    p = o.p_floor;
    bits |= 4;
    rewrite = true;
  }
  double vv = 0;
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) vv += M.g[i][j] * v[i] * v[j];
  if (vv > v2max) {  // R14 (8): Lorentz-factor cap
    const double f = std::sqrt(v2max / vv);
    for (int i = 0; i < 3; i++) v[i] *= f;
    bits |= 8;
    rewrite = true;
  }
  P5[0] = rho; P5[1] = v[0]; P5[2] = v[1]; P5[3] = v[2]; P5[4] = p;
  if (rewrite) {
    double P[8] = {rho, v[0], v[1], v[2], p, B[0], B[1], B[2]};
    double U[8];
    prim2con(P, M, Gamma, U);
    if (bits & 8) U5[0] = U[0];  // the pressure fix alone leaves D untouched
    for (int r = 1; r < 5; r++) U5[r] = U[r];
  }
  if (iters_out) *iters_out = iters;
  return bits;
}

// ---------------------------------------------------------------------------- sources
// R9 / G11: eq. (19) PAPER.md:125 in its exact 3+1 reduction.  dbeta[j][i] = d_j beta^i,
// dg[j][k][l] = d_j gamma_kl.
void sources(const double P[8], const Metric& M, const double K[3][3], const double dalpha[3],
             const double dbeta[3][3], const double dg[3][3][3], double Gamma, double S[5]) {
  const PointState s = point_state(P, M, Gamma);
  const double* v = P + 1;
  const double* B = P + 5;
  const double a = M.alpha;
  double gu[3][3];
  inv3(M.g, det3(M.g), gu);
  // four-velocity and comoving field, eq. (13)
  const double u0 = s.W / a;
  double u[3], b[3];
  const double b0 = s.ab0 / a;
  for (int i = 0; i < 3; i++) u[i] = s.W * (v[i] - M.beta[i] / a);
  for (int i = 0; i < 3; i++) b[i] = (B[i] + s.ab0 * u[i]) / s.W;
  // inverse 4-metric
  const double g00 = -1.0 / (a * a);
  double g0i[3], gij[3][3];
  for (int i = 0; i < 3; i++) g0i[i] = M.beta[i] / (a * a);
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) gij[i][j] = gu[i][j] - M.beta[i] * M.beta[j] / (a * a);
  // T^{mu nu}, eq. (16)
  const double e = s.rhoh + s.b2, pt = P[4] + 0.5 * s.b2;
  const double T00 = e * u0 * u0 + pt * g00 - b0 * b0;
  double T0i[3], Tij[3][3];
  for (int i = 0; i < 3; i++) T0i[i] = e * u0 * u[i] + pt * g0i[i] - b0 * b[i];
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) Tij[i][j] = e * u[i] * u[j] + pt * gij[i][j] - b[i] * b[j];
  double betal[3], T0low[3];
  for (int i = 0; i < 3; i++) {
    betal[i] = 0;
    for (int k = 0; k < 3; k++) betal[i] += M.g[i][k] * M.beta[k];
  }
  for (int i = 0; i < 3; i++) {
    T0low[i] = T00 * betal[i];
    for (int k = 0; k < 3; k++) T0low[i] += T0i[k] * M.g[k][i];
  }
  S[0] = 0.0;
  for (int j = 0; j < 3; j++) {
    double bbdg = 0, t0bdg = 0, t0db = 0, tdg = 0;
    for (int k = 0; k < 3; k++)
      for (int l = 0; l < 3; l++) bbdg += M.beta[k] * M.beta[l] * dg[j][k][l];
    for (int i = 0; i < 3; i++)
      for (int k = 0; k < 3; k++) t0bdg += T0i[i] * M.beta[k] * dg[j][i][k];
    for (int i = 0; i < 3; i++) t0db += T0low[i] * dbeta[j][i];
    for (int i = 0; i < 3; i++)
      for (int k = 0; k < 3; k++) tdg += Tij[i][k] * dg[j][i][k];
    S[1 + j] = T00 * (0.5 * bbdg - a * dalpha[j]) + t0bdg + t0db + 0.5 * tdg;
  }
  double bbK = 0, bda = 0, t0 = 0, tK = 0;
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) bbK += M.beta[i] * M.beta[j] * K[i][j];
  for (int i = 0; i < 3; i++) bda += M.beta[i] * dalpha[i];
  for (int i = 0; i < 3; i++) {
    double bK = 0;
    for (int j = 0; j < 3; j++) bK += M.beta[j] * K[i][j];
    t0 += T0i[i] * (2.0 * bK - dalpha[i]);
  }
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) tK += Tij[i][j] * K[i][j];
  S[4] = T00 * (bbK - bda) + t0 + tK;
}

}  // namespace

// =================================================================================
// The block driver
// =================================================================================
struct ref_grmhd {
  int nx, ny, nz;
  int n[3];
  double dx[3];
  ref_opts o;
  int PX, PY, PZ;  // staggered-shape extents n+2G+1
  size_t NP;
  std::vector<double> met[16];
  std::vector<double> P[5];    // rho, v^i, p (cell centres)
  std::vector<double> Bc[3];   // Eulerian B^i at cell centres
  std::vector<double> Bf[3];   // densitised B~^d on d-faces (total)
  std::vector<double> B0[3];   // static part B~0 (G16)
  std::vector<double> U[5];    // densitised D~, S~_j, tau~
  std::vector<double> A[3];    // vector potential on edges
  std::vector<double> Psi;     // Psi_mhd = sqrt(gamma) Phi on vertices (generalised Lorenz gauge)
  int gauge = 0;               // option "gauge": 0 algebraic, 1 generalised Lorenz
  double lorenz_xi = 1.5;      // option "lorenz_xi": xi = lorenz_xi / dt
  double cur_dt = 0;           // dt of the step being taken (for xi)
  std::vector<double> F[3][8]; // stored fluxes
  std::vector<double> W[3][4]; // UCT face data per direction: a_+, a_-, vbar^{(d+1)%3}, vbar^{(d+2)%3}
  int emf = 0;                 // option "emf": 0 flux-CT (R10), 1 upwind CT
  std::vector<uint8_t> mask;
  bool have_metric = false, have_prims = false, have_mask = false;
  double t = 0, dt = 0, fixed_dt = 0, maxspeed[3] = {0, 0, 0};
  long long steps = 0, c2p_fail = 0, p_fix = 0, atmo = 0, w_cap = 0, c2p_maxiter = 0;
  long long c2p_backup_used = 0;
  int c2p_backup = 0;  // option: 1-D scheme on a failure of the 2-D one
  bool bad_dt = false;

  size_t idx(int i, int j, int k) const {
    return ((size_t)(k + G) * PY + (size_t)(j + G)) * PX + (size_t)(i + G);
  }
  Metric cell_metric(size_t c) const {
    double m[10];
    for (int f = 0; f < 10; f++) m[f] = met[f][c];
    return unpack_metric(m);
  }
  double sqrtg_cell(size_t c) const {
    const Metric M = cell_metric(c);
    return std::sqrt(det3(M.g));
  }
  // R4: 4-point Lagrange interpolation of alpha, beta^k, gamma_kl to face `f-1/2` along d
  // (adapted per G3).  (i,j,k) = index of the UPPER cell of the face.
  Metric face_metric(int d, int i, int j, int k) const {
    const int e[3] = {d == 0, d == 1, d == 2};
    const size_t c0 = idx(i - 2 * e[0], j - 2 * e[1], k - 2 * e[2]);
    const size_t c1 = idx(i - e[0], j - e[1], k - e[2]);
    const size_t c2 = idx(i, j, k);
    const size_t c3 = idx(i + e[0], j + e[1], k + e[2]);
    double m[10];
    for (int f = 0; f < 10; f++)
      m[f] = (-met[f][c0] + 9.0 * met[f][c1] + 9.0 * met[f][c2] - met[f][c3]) / 16.0;
    return unpack_metric(m);
  }

  // ------------------------------------------------------------------ ghost fill (R15)
  // stag[a] = 1 if the field is staggered along axis a.  kind: 0 copy (Neumann/outflow for
  // prims and B~0), 1 linear extrapolation (A_i).  Periodic axes wrap.  x, then y, then z,
  // each pass spanning the full (already filled) extent of the previous axes.
  void fill_ghosts(std::vector<double>& q, const int stag[3], int kind) const {
    int lo[3], hi[3];  // currently valid index range per axis, inclusive
    for (int a = 0; a < 3; a++) { lo[a] = 0; hi[a] = n[a] - 1 + stag[a]; }
    for (int a = 0; a < 3; a++) {
      const bool periodic = (o.bc[a] == 0);
      const int glo = -G, ghi = n[a] + G - 1 + stag[a];
      const int b0 = (a + 1) % 3, b1 = (a + 2) % 3;
      auto do_layer = [&](int g) {
        int src, src2 = 0;
        if (periodic) {
          src = ((g % n[a]) + n[a]) % n[a];  // period n[a]; staggered index n[a] = image of 0
        } else if (g < 0) {
          src = (kind == 0) ? 0 : g + 1;
          src2 = g + 2;
        } else {
          src = (kind == 0) ? hi[a] : g - 1;
          src2 = g - 2;
        }
        for (int q1 = lo[b1]; q1 <= hi[b1]; q1++)
          for (int q0 = lo[b0]; q0 <= hi[b0]; q0++) {
            int I[3], J[3], K2[3];
            I[a] = g; I[b0] = q0; I[b1] = q1;
            J[a] = src; J[b0] = q0; J[b1] = q1;
            K2[a] = src2; K2[b0] = q0; K2[b1] = q1;
            if (!periodic && kind == 1)  // A_g = 2 A_{g-+1} - A_{g-+2}, layer by layer
              q[idx(I[0], I[1], I[2])] =
                  2.0 * q[idx(J[0], J[1], J[2])] - q[idx(K2[0], K2[1], K2[2])];
            else
              q[idx(I[0], I[1], I[2])] = q[idx(J[0], J[1], J[2])];
          }
      };
      for (int g = -1; g >= glo; g--) do_layer(g);
      for (int g = (periodic ? n[a] : hi[a] + 1); g <= ghi; g++) do_layer(g);
      lo[a] = glo; hi[a] = ghi;
    }
  }

  // ---------------------------------------------------------------- B from A (R13)
  void field_from_potential() {
    const int sAx[3] = {0, 1, 1}, sAy[3] = {1, 0, 1}, sAz[3] = {1, 1, 0};
    fill_ghosts(A[0], sAx, 1);
    fill_ghosts(A[1], sAy, 1);
    fill_ghosts(A[2], sAz, 1);
    // B~^i = B~0^i + [ijk] d_j A_k on faces, eq. (24) PAPER.md:149 with
    // epsilon^{ijk} = [ijk]/sqrt(gamma).  All faces whose edges exist.
#pragma omp parallel for num_threads(g_threads)
    for (int k = -G; k < nz + G; k++)
      for (int j = -G; j < ny + G; j++)
        for (int i = -G; i < nx + G; i++) {
          const size_t c = idx(i, j, k);
          Bf[0][c] = B0[0][c] + (A[2][idx(i, j + 1, k)] - A[2][c]) / dx[1] -
                     (A[1][idx(i, j, k + 1)] - A[1][c]) / dx[2];
          Bf[1][c] = B0[1][c] + (A[0][idx(i, j, k + 1)] - A[0][c]) / dx[2] -
                     (A[2][idx(i + 1, j, k)] - A[2][c]) / dx[0];
          Bf[2][c] = B0[2][c] + (A[1][idx(i + 1, j, k)] - A[1][c]) / dx[0] -
                     (A[0][idx(i, j + 1, k)] - A[0][c]) / dx[1];
        }
    // upper boundary faces (index n+G along the face normal) keep the static value:
    for (int k = -G; k <= nz + G; k++)
      for (int j = -G; j <= ny + G; j++)
        for (int i = -G; i <= nx + G; i++) {
          if (i < nx + G && j < ny + G && k < nz + G) continue;
          const size_t c = idx(i, j, k);
          for (int d = 0; d < 3; d++) Bf[d][c] = B0[d][c];
        }
    // the x-faces at i = nx+G with j,k inside DO have all their edges: evaluate them too.
    for (int k = -G; k < nz + G; k++)
      for (int j = -G; j < ny + G; j++) {
        const int i = nx + G;
        const size_t c = idx(i, j, k);
        Bf[0][c] = B0[0][c] + (A[2][idx(i, j + 1, k)] - A[2][c]) / dx[1] -
                   (A[1][idx(i, j, k + 1)] - A[1][c]) / dx[2];
      }
    for (int k = -G; k < nz + G; k++)
      for (int i = -G; i < nx + G; i++) {
        const int j = ny + G;
        const size_t c = idx(i, j, k);
        Bf[1][c] = B0[1][c] + (A[0][idx(i, j, k + 1)] - A[0][c]) / dx[2] -
                   (A[2][idx(i + 1, j, k)] - A[2][c]) / dx[0];
      }
    for (int j = -G; j < ny + G; j++)
      for (int i = -G; i < nx + G; i++) {
        const int k = nz + G;
        const size_t c = idx(i, j, k);
        Bf[2][c] = B0[2][c] + (A[1][idx(i + 1, j, k)] - A[1][c]) / dx[0] -
                   (A[0][idx(i, j + 1, k)] - A[0][c]) / dx[1];
      }
    // cell centres: mean of the two faces, undensitised
#pragma omp parallel for num_threads(g_threads)
    for (int k = -G; k < nz + G; k++)
      for (int j = -G; j < ny + G; j++)
        for (int i = -G; i < nx + G; i++) {
          const size_t c = idx(i, j, k);
          const double sg = sqrtg_cell(c);
          Bc[0][c] = 0.5 * (Bf[0][c] + Bf[0][idx(i + 1, j, k)]) / sg;
          Bc[1][c] = 0.5 * (Bf[1][c] + Bf[1][idx(i, j + 1, k)]) / sg;
          Bc[2][c] = 0.5 * (Bf[2][c] + Bf[2][idx(i, j, k + 1)]) / sg;
        }
  }

  // ------------------------------------------------- con2prim over the interior (R14)
  void recover_primitives() {
    long long nf = 0, np = 0, na = 0, nw = 0, nb = 0, mi = 0;
#pragma omp parallel for num_threads(g_threads) reduction(+ : nf, np, na, nw, nb) reduction(max : mi)
    for (int k = 0; k < nz; k++)
      for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) {
          const size_t c = idx(i, j, k);
          const Metric M = cell_metric(c);
          const double sg = std::sqrt(det3(M.g));
          double Uin[5], B[3], P5[5], U5[5];
          for (int r = 0; r < 5; r++) Uin[r] = U[r][c] / sg;  // undensitise, eq. (17)
          for (int d = 0; d < 3; d++) B[d] = Bc[d][c];
          int it = 0;
          const int bits = con2prim(Uin, B, M, o, have_mask && mask[c], P5, U5, &it,
                                    c2p_backup != 0);
          for (int r = 0; r < 5; r++) P[r][c] = P5[r];
          if (bits & (1 | 2 | 4 | 8)) {
            if (bits & (1 | 2 | 8)) U[0][c] = sg * U5[0];
            for (int r = 1; r < 5; r++) U[r][c] = sg * U5[r];
          }
          nf += (bits & 2) != 0; np += (bits & 4) != 0; na += (bits & 1) != 0;
          nw += (bits & 8) != 0; nb += (bits & 16) != 0;
          if (it > mi) mi = it;
        }
    c2p_fail += nf; p_fix += np; atmo += na; w_cap += nw; c2p_backup_used += nb;
    c2p_maxiter = std::max(c2p_maxiter, mi);
  }

  void fill_prim_ghosts() {
    const int cc[3] = {0, 0, 0};
    for (int r = 0; r < 5; r++) fill_ghosts(P[r], cc, 0);
  }

  // everything that follows a change of (U, A): R13, R14, R15
  void after_stage() {
    if (gauge == 1) {
      const int sV[3] = {1, 1, 1};
      fill_ghosts(Psi, sV, 0);  // periodic wrap / copy
    }
    field_from_potential();
    recover_primitives();
    fill_prim_ghosts();
  }

  void prims_to_cons_interior() {
#pragma omp parallel for num_threads(g_threads)
    for (int k = 0; k < nz; k++)
      for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) {
          const size_t c = idx(i, j, k);
          const Metric M = cell_metric(c);
          const double sg = std::sqrt(det3(M.g));
          double Pp[8] = {P[0][c], P[1][c], P[2][c], P[3][c], P[4][c],
                          Bc[0][c], Bc[1][c], Bc[2][c]};
          double Uu[8];
          prim2con(Pp, M, o.gamma_ad, Uu);
          for (int r = 0; r < 5; r++) U[r][c] = sg * Uu[r];
        }
  }

  // ---------------------------------------------------------------- fluxes (R4-R7)
  void compute_fluxes() {
    for (int d = 0; d < 3; d++) {
      const int e[3] = {d == 0, d == 1, d == 2};
      for (int r = 0; r < 8; r++) std::fill(F[d][r].begin(), F[d][r].end(), 0.0);
      // faces f = 0..n_d along d; transverse cells with a 1-cell apron (R10), or with the 3
      // cells the face -> edge PPM stencils of the upwind CT reach (G26)
      const int ap = emf == 1 ? 3 : 1;
      if (emf == 1)
        for (int r = 0; r < 4; r++) W[d][r].assign(NP, 0.0);
      const int lo[3] = {e[0] ? 0 : -ap, e[1] ? 0 : -ap, e[2] ? 0 : -ap};
      const int hi[3] = {e[0] ? nx : nx + ap - 1, e[1] ? ny : ny + ap - 1,
                         e[2] ? nz : nz + ap - 1};  // inclusive
#pragma omp parallel for num_threads(g_threads)
      for (int k = lo[2]; k <= hi[2]; k++)
        for (int j = lo[1]; j <= hi[1]; j++)
          for (int i = lo[0]; i <= hi[0]; i++) {
            const Metric Mf = face_metric(d, i, j, k);
            const double sgf = std::sqrt(det3(Mf.g));
            double c[8][6];
            for (int s = 0; s < 6; s++) {
              const size_t cc = idx(i + (s - 3) * e[0], j + (s - 3) * e[1], k + (s - 3) * e[2]);
              for (int v = 0; v < 5; v++) c[v][s] = P[v][cc];
              for (int v = 0; v < 3; v++) c[5 + v][s] = Bc[v][cc];
            }
            double PL[8], PR[8], Fh[8];
            recon_face(d, c, o, PL, PR);
            // G6: the normal component is the single-valued staggered field
            PL[5 + d] = PR[5 + d] = Bf[d][idx(i, j, k)] / sgf;
            double uct[4];
            riemann(d, PL, PR, Mf, o, Fh, emf == 1 ? uct : nullptr);
            for (int r = 0; r < 8; r++) F[d][r][idx(i, j, k)] = sgf * Fh[r];
            if (emf == 1)
              for (int r = 0; r < 4; r++) W[d][r][idx(i, j, k)] = uct[r];
          }
    }
  }

  // 4th-order centred derivative along axis a (R9 / G12); exactly 0 on constants.
  double deriv(const std::vector<double>& q, int a, int i, int j, int k) const {
    const int e[3] = {a == 0, a == 1, a == 2};
    const double p1 = q[idx(i + e[0], j + e[1], k + e[2])];
    const double m1 = q[idx(i - e[0], j - e[1], k - e[2])];
    const double p2 = q[idx(i + 2 * e[0], j + 2 * e[1], k + 2 * e[2])];
    const double m2 = q[idx(i - 2 * e[0], j - 2 * e[1], k - 2 * e[2])];
    return (8.0 * (p1 - m1) - (p2 - m2)) / (12.0 * dx[a]);
  }

  // ---------------------------------------------------------- L(Y) (R8, R10, R11)
  void rhs(std::vector<double> kU[5], std::vector<double> kA[3],
           std::vector<double>* kPsi = nullptr) {
    compute_fluxes();
    for (int r = 0; r < 5; r++) kU[r].assign(NP, 0.0);
    for (int d = 0; d < 3; d++) kA[d].assign(NP, 0.0);
#pragma omp parallel for num_threads(g_threads)
    for (int k = 0; k < nz; k++)
      for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) {
          const size_t c = idx(i, j, k);
          const Metric M = cell_metric(c);
          const double sg = std::sqrt(det3(M.g));
          double Kc[3][3];
          Kc[0][0] = met[10][c]; Kc[0][1] = Kc[1][0] = met[11][c];
          Kc[0][2] = Kc[2][0] = met[12][c]; Kc[1][1] = met[13][c];
          Kc[1][2] = Kc[2][1] = met[14][c]; Kc[2][2] = met[15][c];
          double da[3], db[3][3], dg[3][3][3];
          for (int a = 0; a < 3; a++) {
            da[a] = deriv(met[0], a, i, j, k);
            for (int b = 0; b < 3; b++) db[a][b] = deriv(met[1 + b], a, i, j, k);
            dg[a][0][0] = deriv(met[4], a, i, j, k);
            dg[a][0][1] = dg[a][1][0] = deriv(met[5], a, i, j, k);
            dg[a][0][2] = dg[a][2][0] = deriv(met[6], a, i, j, k);
            dg[a][1][1] = deriv(met[7], a, i, j, k);
            dg[a][1][2] = dg[a][2][1] = deriv(met[8], a, i, j, k);
            dg[a][2][2] = deriv(met[9], a, i, j, k);
          }
          double Pp[8] = {P[0][c], P[1][c], P[2][c], P[3][c], P[4][c],
                          Bc[0][c], Bc[1][c], Bc[2][c]};
          double S[5];
          sources(Pp, M, Kc, da, db, dg, o.gamma_ad, S);
          for (int r = 0; r < 5; r++) {
            // eq. (17): d_t(sqrt(gamma) F^0) = -d_i(sqrt(-g) F^i) + sqrt(-g) S
            double div = 0;
            div += (F[0][r][idx(i + 1, j, k)] - F[0][r][c]) / dx[0];
            div += (F[1][r][idx(i, j + 1, k)] - F[1][r][c]) / dx[1];
            div += (F[2][r][idx(i, j, k + 1)] - F[2][r][c]) / dx[2];
            kU[r][c] = -div + M.alpha * sg * S[r];
          }
        }
    if (kPsi) kPsi->assign(NP, 0.0);
    if (emf == 1) {
      uct_rhs(kA);
      if (gauge == 1 && kPsi) lorenz_terms(kA, *kPsi);
      return;
    }
    // R10: flux-CT electric field on edges; R11: d_t A_i = -E_i (algebraic gauge)
    const std::vector<double>&FxBy = F[0][6], &FxBz = F[0][7], &FyBx = F[1][5],
                             &FyBz = F[1][7], &FzBx = F[2][5], &FzBy = F[2][6];
    for (int k = 0; k <= nz; k++)
      for (int j = 0; j <= ny; j++)
        for (int i = 0; i <= nx; i++) {
          const size_t c = idx(i, j, k);
          if (i < nx) {  // E_x at (i, j-1/2, k-1/2)
            const double Ex = 0.25 * (-FyBz[idx(i, j, k - 1)] - FyBz[c] +
                                      FzBy[idx(i, j - 1, k)] + FzBy[c]);
            kA[0][c] = -Ex;
          }
          if (j < ny) {  // E_y at (i-1/2, j, k-1/2)
            const double Ey = 0.25 * (-FzBx[idx(i - 1, j, k)] - FzBx[c] +
                                      FxBz[idx(i, j, k - 1)] + FxBz[c]);
            kA[1][c] = -Ey;
          }
          if (k < nz) {  // E_z at (i-1/2, j-1/2, k)
            const double Ez = 0.25 * (-FxBy[idx(i, j - 1, k)] - FxBy[c] +
                                      FyBx[idx(i - 1, j, k)] + FyBx[c]);
            kA[2][c] = -Ez;
          }
        }
    if (gauge == 1 && kPsi) lorenz_terms(kA, *kPsi);
  }

  // ---------------------------------------- generalised Lorenz gauge (row F3, G29-G32)
  // eqs (31), (32).  Everything is evaluated at the vertices
  // (i-1/2, j-1/2, k-1/2) where Psi_mhd lives: the metric there is the mean of the 8 cells
  // around the vertex (G29: the metric is cell-centred input, G3), A_j the mean of the two
  // edges of its own axis that end at the vertex (G30).
  struct VertexData {
    double alpha, beta[3], sg, gu[3][3], Av[3], psi;
  };
  VertexData vertex(int i, int j, int k) const {
    VertexData v;
    Metric M;
    double acc[10] = {0};
    for (int c = 0; c < 8; c++) {
      const size_t q = idx(i - (c & 1), j - ((c >> 1) & 1), k - ((c >> 2) & 1));
      for (int f = 0; f < 10; f++) acc[f] += met[f][q];
    }
    for (int f = 0; f < 10; f++) acc[f] *= 0.125;
    M = unpack_metric(acc);
    v.alpha = M.alpha;
    for (int a = 0; a < 3; a++) v.beta[a] = M.beta[a];
    const double det = det3(M.g);
    v.sg = std::sqrt(det);
    inv3(M.g, det, v.gu);
    v.Av[0] = 0.5 * (A[0][idx(i - 1, j, k)] + A[0][idx(i, j, k)]);
    v.Av[1] = 0.5 * (A[1][idx(i, j - 1, k)] + A[1][idx(i, j, k)]);
    v.Av[2] = 0.5 * (A[2][idx(i, j, k - 1)] + A[2][idx(i, j, k)]);
    v.psi = Psi[idx(i, j, k)];
    return v;
  }
  // G_A = alpha Psi/sqrt(gamma) - beta^j A_j, eq. (31) (eq. (25) prints beta^j A_i: read A_j)
  double gauge_GA(int i, int j, int k) const {
    const VertexData v = vertex(i, j, k);
    return v.alpha * v.psi / v.sg - (v.beta[0] * v.Av[0] + v.beta[1] * v.Av[1] + v.beta[2] * v.Av[2]);
  }
  // F_Psi^d = alpha sqrt(gamma) A^d - beta^d Psi, eq. (32), A^d = gamma^{dl} A_l
  double gauge_FPsi(int d, int i, int j, int k) const {
    const VertexData v = vertex(i, j, k);
    const double Au = v.gu[d][0] * v.Av[0] + v.gu[d][1] * v.Av[1] + v.gu[d][2] * v.Av[2];
    return v.alpha * v.sg * Au - v.beta[d] * v.psi;
  }
  // adds -d_i G_A to d_t A_i (2-point difference of the two vertices bounding the edge, G31:
  // a discrete gradient, so that B = curl A is untouched) and forms
  // d_t Psi = -d_j F_Psi^j - xi alpha Psi at the vertices (2nd-order centred differences, G32)
  void lorenz_terms(std::vector<double> kA[3], std::vector<double>& kPsi) const {
    const double xi = cur_dt > 0 ? lorenz_xi / cur_dt : 0.0;
    for (int k = 0; k <= nz; k++)
      for (int j = 0; j <= ny; j++)
        for (int i = 0; i <= nx; i++) {
          const size_t c = idx(i, j, k);
          const double G0 = gauge_GA(i, j, k);
          if (i < nx) kA[0][c] -= (gauge_GA(i + 1, j, k) - G0) / dx[0];
          if (j < ny) kA[1][c] -= (gauge_GA(i, j + 1, k) - G0) / dx[1];
          if (k < nz) kA[2][c] -= (gauge_GA(i, j, k + 1) - G0) / dx[2];
          double div = 0;
          div += (gauge_FPsi(0, i + 1, j, k) - gauge_FPsi(0, i - 1, j, k)) / (2.0 * dx[0]);
          div += (gauge_FPsi(1, i, j + 1, k) - gauge_FPsi(1, i, j - 1, k)) / (2.0 * dx[1]);
          div += (gauge_FPsi(2, i, j, k + 1) - gauge_FPsi(2, i, j, k - 1)) / (2.0 * dx[2]);
          kPsi[c] = -div - xi * vertex(i, j, k).alpha * Psi[c];
        }
  }

  // ------------------------------------- upwind constrained transport (row F1, G26-G28)
  // PAPER.md:229-250, eqs (33)-(35).  For the edge component E_c with (a, b, c) cyclic:
  //   E_c = - [a-bracket of vbar^a B~^b] + [b-bracket of vbar^b B~^a]
  // The a-bracket takes vbar^a (eq. 33, stored on the b-faces) and the staggered B~^b (on the
  // b-faces), both reconstructed ALONG a to the edge with the PPM of G8 (no flattening): L
  // from the lower, R from the upper side; its a_+-, a_-^a are the larger of the values on the
  // two a-faces that share the edge.  Lower convention: edge (i,j,k) of E_z = (i-1/2, j-1/2, k).
  double edge_bracket(int a, int b, int i, int j, int k) const {
    const int ea[3] = {a == 0, a == 1, a == 2}, eb[3] = {b == 0, b == 1, b == 2};
    // vbar^a on b-faces: slot 2 if a == (b+1)%3 else slot 3
    const std::vector<double>& vb = W[b][a == (b + 1) % 3 ? 2 : 3];
    double sv[6], sB[6];
    for (int m = 0; m < 6; m++) {
      const size_t c = idx(i + (m - 3) * ea[0], j + (m - 3) * ea[1], k + (m - 3) * ea[2]);
      sv[m] = vb[c];
      sB[m] = Bf[b][c];
    }
    double vL, vR, BL, BR, dum;
    ppm_cell(sv, 0.0, dum, vL);      // q^+ of the lower cell
    ppm_cell(sv + 1, 0.0, vR, dum);  // q^- of the upper cell
    ppm_cell(sB, 0.0, dum, BL);
    ppm_cell(sB + 1, 0.0, BR, dum);
    const size_t c0 = idx(i, j, k), cm = idx(i - eb[0], j - eb[1], k - eb[2]);
    const double ap = std::max(W[a][0][c0], W[a][0][cm]);
    const double am = std::max(W[a][1][c0], W[a][1][cm]);
    return uct_bracket(ap, am, vL, vR, BL, BR);
  }

  void uct_rhs(std::vector<double> kA[3]) {
    for (int k = 0; k <= nz; k++)
      for (int j = 0; j <= ny; j++)
        for (int i = 0; i <= nx; i++) {
          const size_t c = idx(i, j, k);
          // R11: d_t A_i = -E_i
          if (i < nx) kA[0][c] = -(-edge_bracket(1, 2, i, j, k) + edge_bracket(2, 1, i, j, k));
          if (j < ny) kA[1][c] = -(-edge_bracket(2, 0, i, j, k) + edge_bracket(0, 2, i, j, k));
          if (k < nz) kA[2][c] = -(-edge_bracket(0, 1, i, j, k) + edge_bracket(1, 0, i, j, k));
        }
  }

  // ------------------------------------------------------------------- dt (R16)
  void compute_maxspeed() {
    double m[3] = {0, 0, 0};
    for (int d = 0; d < 3; d++) {
      double md = 0;
#pragma omp parallel for num_threads(g_threads) reduction(max : md)
      for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++)
          for (int i = 0; i < nx; i++) {
            const size_t c = idx(i, j, k);
            const Metric M = cell_metric(c);
            double gu[3][3];
            inv3(M.g, det3(M.g), gu);
            double Pp[8] = {P[0][c], P[1][c], P[2][c], P[3][c], P[4][c],
                            Bc[0][c], Bc[1][c], Bc[2][c]};
            double lam[2];
            speeds(d, Pp, M, gu[d][d], o.gamma_ad, lam);
            const double s = std::max(std::fabs(lam[0]), std::fabs(lam[1]));
            if (s > md) md = s;
          }
      m[d] = md;
    }
    for (int d = 0; d < 3; d++) maxspeed[d] = m[d];
  }

  double cfl_dt(double cfl) const {
    if (fixed_dt > 0) return fixed_dt;
    double dtm = INFINITY;
    for (int d = 0; d < 3; d++) dtm = std::min(dtm, dx[d] / maxspeed[d]);
    return cfl * dtm;
  }

  // ---------------------------------------------------------------- one RK step (R12)
  void axpby(double a, const std::vector<double>& x, double b, const std::vector<double>& y,
             std::vector<double>& out) const {
    for (size_t q = 0; q < NP; q++) out[q] = a * x[q] + b * y[q];
  }

  void one_step(double h) {
    cur_dt = h;
    std::vector<double> Y0[9], k1[9], k2[9], k3[9], k4[9];  // D~, S~_j, tau~, A_i, Psi_mhd
    auto Y = [&](int r) -> std::vector<double>& { return r < 5 ? U[r] : (r < 8 ? A[r - 5] : Psi); };
    for (int r = 0; r < 9; r++) Y0[r] = Y(r);
    auto L = [&](std::vector<double> k[9]) { rhs(k, k + 5, &k[8]); };
    if (o.rk == 2) {
      // SSP-RK2 (Heun): Y1 = Y0 + dt L(Y0); Y^{n+1} = 1/2 Y0 + 1/2 (Y1 + dt L(Y1))
      L(k1);
      for (int r = 0; r < 9; r++) axpby(1.0, Y0[r], h, k1[r], Y(r));
      after_stage();
      L(k2);
      for (int r = 0; r < 9; r++) {
        std::vector<double>& y = Y(r);
        for (size_t q = 0; q < NP; q++) y[q] = 0.5 * Y0[r][q] + 0.5 * (y[q] + h * k2[r][q]);
      }
      after_stage();
    } else if (o.rk == 3) {
      // SSP-RK3 (Shu-Osher)
      L(k1);
      for (int r = 0; r < 9; r++) axpby(1.0, Y0[r], h, k1[r], Y(r));
      after_stage();
      L(k2);
      for (int r = 0; r < 9; r++) {
        std::vector<double>& y = Y(r);
        for (size_t q = 0; q < NP; q++) y[q] = 0.75 * Y0[r][q] + 0.25 * (y[q] + h * k2[r][q]);
      }
      after_stage();
      L(k3);
      for (int r = 0; r < 9; r++) {
        std::vector<double>& y = Y(r);
        for (size_t q = 0; q < NP; q++)
          y[q] = (1.0 / 3.0) * Y0[r][q] + (2.0 / 3.0) * (y[q] + h * k3[r][q]);
      }
      after_stage();
    } else {
      // classic RK4
      L(k1);
      for (int r = 0; r < 9; r++) axpby(1.0, Y0[r], 0.5 * h, k1[r], Y(r));
      after_stage();
      L(k2);
      for (int r = 0; r < 9; r++) axpby(1.0, Y0[r], 0.5 * h, k2[r], Y(r));
      after_stage();
      L(k3);
      for (int r = 0; r < 9; r++) axpby(1.0, Y0[r], h, k3[r], Y(r));
      after_stage();
      L(k4);
      for (int r = 0; r < 9; r++) {
        std::vector<double>& y = Y(r);
        for (size_t q = 0; q < NP; q++)
          y[q] = Y0[r][q] +
                 (h / 6.0) * (k1[r][q] + 2.0 * k2[r][q] + 2.0 * k3[r][q] + k4[r][q]);
      }
      after_stage();
    }
    t += h;
    dt = h;
    steps++;
    compute_maxspeed();
  }
};

// =================================================================================
// C ABI
// =================================================================================
extern "C" {

void ref_set_num_threads(int n) { g_threads = n < 1 ? 1 : n; }
int ref_get_num_threads(void) { return g_threads; }

int ref_create(int nx, int ny, int nz, int ghosts, const double dx[3], const ref_opts* o,
               ref_grmhd** out) {
  if (!o || !dx || !out || ghosts != G || nx < 1 || ny < 1 || nz < 1) return -1;
  const int n[3] = {nx, ny, nz};
  for (int a = 0; a < 3; a++) {
    if (!(dx[a] > 0)) return -1;
    if (o->bc[a] != 0 && o->bc[a] != 1) return -1;
    if (o->bc[a] == 1 && n[a] < 2) return -1;
  }
  if (o->rk < 2 || o->rk > 4 || o->recon < 0 || o->recon > 1 || !(o->gamma_ad > 1.0) ||
      !(o->p_floor > 0) || !(o->rho_atm > 0) || !(o->w_max > 1.0) || o->c2p_maxit < 1 ||
      o->riemann < 0 || o->riemann > 1)
    return -1;
  ref_grmhd* h = new ref_grmhd;
  h->nx = nx; h->ny = ny; h->nz = nz;
  for (int a = 0; a < 3; a++) { h->n[a] = n[a]; h->dx[a] = dx[a]; }
  h->o = *o;
  h->PX = nx + 2 * G + 1; h->PY = ny + 2 * G + 1; h->PZ = nz + 2 * G + 1;
  h->NP = (size_t)h->PX * h->PY * h->PZ;
  for (auto& v : h->met) v.assign(h->NP, 0.0);
  for (auto& v : h->P) v.assign(h->NP, 0.0);
  for (int d = 0; d < 3; d++) {
    h->Bc[d].assign(h->NP, 0.0); h->Bf[d].assign(h->NP, 0.0); h->B0[d].assign(h->NP, 0.0);
    h->A[d].assign(h->NP, 0.0);
    for (int r = 0; r < 8; r++) h->F[d][r].assign(h->NP, 0.0);
  }
  h->Psi.assign(h->NP, 0.0);
  for (auto& v : h->U) v.assign(h->NP, 0.0);
  h->mask.assign(h->NP, 0);
  *out = h;
  return 0;
}

int ref_destroy(ref_grmhd* h) { delete h; return 0; }

static void copy_in_cc(ref_grmhd* h, const double* src, std::vector<double>& dst) {
  const int sx = h->nx + 2 * G, sy = h->ny + 2 * G;
  for (int k = -G; k < h->nz + G; k++)
    for (int j = -G; j < h->ny + G; j++)
      for (int i = -G; i < h->nx + G; i++)
        dst[h->idx(i, j, k)] = src[((size_t)(k + G) * sy + (j + G)) * sx + (i + G)];
}
static void copy_out_cc(ref_grmhd* h, const std::vector<double>& src, double* dst) {
  const int sx = h->nx + 2 * G, sy = h->ny + 2 * G;
  for (int k = -G; k < h->nz + G; k++)
    for (int j = -G; j < h->ny + G; j++)
      for (int i = -G; i < h->nx + G; i++)
        dst[((size_t)(k + G) * sy + (j + G)) * sx + (i + G)] = src[h->idx(i, j, k)];
}

int ref_set_metric(ref_grmhd* h, const double* const field[16]) {
  if (!h || !field) return -1;
  for (int f = 0; f < 16; f++) {
    if (!field[f]) return -1;
    copy_in_cc(h, field[f], h->met[f]);
  }
  h->have_metric = true;
  return 0;
}

static void init_state_from_prims(ref_grmhd* h) {
  h->field_from_potential();
  h->prims_to_cons_interior();
  h->compute_maxspeed();
}

int ref_set_prims(ref_grmhd* h, const double* const field[8]) {
  if (!h || !field) return -1;
  if (!h->have_metric) return -3;
  for (int r = 0; r < 5; r++)
    if (!field[r]) return -1;
  const bool haveB = field[5] && field[6] && field[7];
  if (!haveB && (field[5] || field[6] || field[7])) return -1;
  const int cc[3] = {0, 0, 0};
  for (int r = 0; r < 5; r++) { copy_in_cc(h, field[r], h->P[r]); }
  h->fill_prim_ghosts();
  for (int d = 0; d < 3; d++) {
    std::fill(h->A[d].begin(), h->A[d].end(), 0.0);
    std::fill(h->B0[d].begin(), h->B0[d].end(), 0.0);
  }
  std::fill(h->Psi.begin(), h->Psi.end(), 0.0);
  if (haveB) {
    // G16: static face field B~0 = 2-point mean along the component's own axis of
    // sqrt(gamma_c) B^i_c, on faces 0..n_d, then ghost faces by wrap / copy.
    for (int d = 0; d < 3; d++) {
      std::vector<double> Bin(h->NP, 0.0);
      copy_in_cc(h, field[5 + d], Bin);
      h->fill_ghosts(Bin, cc, 0);
      const int e[3] = {d == 0, d == 1, d == 2};
      for (int k = 0; k < h->nz + e[2]; k++)
        for (int j = 0; j < h->ny + e[1]; j++)
          for (int i = 0; i < h->nx + e[0]; i++) {
            const size_t c = h->idx(i, j, k), cm = h->idx(i - e[0], j - e[1], k - e[2]);
            h->B0[d][c] = 0.5 * (h->sqrtg_cell(cm) * Bin[cm] + h->sqrtg_cell(c) * Bin[c]);
          }
      h->fill_ghosts(h->B0[d], e, 0);
    }
  }
  h->have_prims = true;
  h->t = 0; h->steps = 0; h->dt = 0;
  h->c2p_fail = h->p_fix = h->atmo = h->w_cap = h->c2p_maxiter = h->c2p_backup_used = 0;
  h->bad_dt = false;
  init_state_from_prims(h);
  return 0;
}

int ref_set_vecpot(ref_grmhd* h, const double* const field[3]) {
  if (!h || !field) return -1;
  if (!h->have_prims) return -3;
  for (int d = 0; d < 3; d++) {
    if (!field[d]) return -1;
    std::memcpy(h->A[d].data(), field[d], h->NP * sizeof(double));
  }
  init_state_from_prims(h);
  return 0;
}

int ref_set_mask(ref_grmhd* h, const unsigned char* mask) {
  if (!h) return -1;
  if (!mask) { h->have_mask = false; return 0; }
  const int sx = h->nx + 2 * G, sy = h->ny + 2 * G;
  for (int k = -G; k < h->nz + G; k++)
    for (int j = -G; j < h->ny + G; j++)
      for (int i = -G; i < h->nx + G; i++)
        h->mask[h->idx(i, j, k)] = mask[((size_t)(k + G) * sy + (j + G)) * sx + (i + G)];
  h->have_mask = true;
  return 0;
}

int ref_step(ref_grmhd* h, int n, double cfl) {
  if (!h || n < 0) return -1;
  if (!h->have_metric || !h->have_prims) return -3;
  for (int s = 0; s < n; s++) {
    const double dt = h->cfl_dt(cfl);
    if (!(dt > 0) || !std::isfinite(dt)) { h->bad_dt = true; return -5; }
    h->one_step(dt);
  }
  return 0;
}

int ref_step_until(ref_grmhd* h, double t_end, double cfl, int* nsteps_done) {
  if (!h) return -1;
  if (!h->have_metric || !h->have_prims) return -3;
  int n = 0;
  while (t_end - h->t > 1e-12 * std::max(1.0, std::fabs(t_end))) {
    double dt = h->cfl_dt(cfl);
    if (!(dt > 0) || !std::isfinite(dt)) { h->bad_dt = true; return -5; }
    if (dt > t_end - h->t) dt = t_end - h->t;
    h->one_step(dt);
    n++;
  }
  if (nsteps_done) *nsteps_done = n;
  return 0;
}

int ref_get_prims(ref_grmhd* h, double* const field[8]) {
  if (!h || !field) return -1;
  for (int r = 0; r < 5; r++) copy_out_cc(h, h->P[r], field[r]);
  for (int d = 0; d < 3; d++) copy_out_cc(h, h->Bc[d], field[5 + d]);
  return 0;
}

int ref_get_cons(ref_grmhd* h, double* const field[8]) {
  if (!h || !field) return -1;
  std::vector<double> tmp(h->NP);
  for (int r = 0; r < 8; r++) {
    std::fill(tmp.begin(), tmp.end(), 0.0);
    for (int k = 0; k < h->nz; k++)
      for (int j = 0; j < h->ny; j++)
        for (int i = 0; i < h->nx; i++) {
          const size_t c = h->idx(i, j, k);
          tmp[c] = r < 5 ? h->U[r][c] / h->sqrtg_cell(c) : h->Bc[r - 5][c];
        }
    copy_out_cc(h, tmp, field[r]);
  }
  return 0;
}

int ref_get_vecpot(ref_grmhd* h, double* const field[3]) {
  if (!h || !field) return -1;
  for (int d = 0; d < 3; d++) std::memcpy(field[d], h->A[d].data(), h->NP * sizeof(double));
  return 0;
}

int ref_get_psi(ref_grmhd* h, double* field) {
  if (!h || !field) return -1;
  std::memcpy(field, h->Psi.data(), h->NP * sizeof(double));
  return 0;
}

int ref_get_bface(ref_grmhd* h, double* const field[3]) {
  if (!h || !field) return -1;
  for (int d = 0; d < 3; d++) std::memcpy(field[d], h->Bf[d].data(), h->NP * sizeof(double));
  return 0;
}

int ref_set_option(ref_grmhd* h, const char* key, double value) {
  if (!h || !key) return -1;
  if (std::strcmp(key, "fixed_dt") == 0) { h->fixed_dt = value; return 0; }
  if (std::strcmp(key, "c2p_backup") == 0) { h->c2p_backup = value != 0.0; return 0; }
  if (std::strcmp(key, "emf") == 0) { h->emf = value != 0.0; return 0; }
  if (std::strcmp(key, "gauge") == 0) { h->gauge = value != 0.0; return 0; }
  if (std::strcmp(key, "lorenz_xi") == 0) { h->lorenz_xi = value; return 0; }
  return -1;
}

int ref_get_stats(ref_grmhd* h, ref_stats* out) {
  if (!h || !out) return -1;
  out->t = h->t; out->dt = h->dt;
  for (int d = 0; d < 3; d++) out->maxspeed[d] = h->maxspeed[d];
  out->steps = h->steps; out->c2p_fail = h->c2p_fail; out->p_fix = h->p_fix;
  out->atmo = h->atmo; out->w_cap = h->w_cap; out->c2p_maxiter = h->c2p_maxiter;
  out->c2p_backup = h->c2p_backup_used;
  return h->bad_dt ? -5 : 0;
}

int ref_rhs(ref_grmhd* h, double* const dU[5], double* const dA[3]) {
  if (!h || !dU || !dA) return -1;
  if (!h->have_metric || !h->have_prims) return -3;
  std::vector<double> k[8];
  h->rhs(k, k + 5);
  for (int r = 0; r < 5; r++) copy_out_cc(h, k[r], dU[r]);
  for (int d = 0; d < 3; d++) std::memcpy(dA[d], k[5 + d].data(), h->NP * sizeof(double));
  return 0;
}

int ref_rhs_gauge(ref_grmhd* h, double* const dA[3], double* dPsi) {
  if (!h || !dA || !dPsi) return -1;
  if (!h->have_metric || !h->have_prims) return -3;
  std::vector<double> k[8], kp;
  h->rhs(k, k + 5, &kp);
  for (int d = 0; d < 3; d++) std::memcpy(dA[d], k[5 + d].data(), h->NP * sizeof(double));
  std::memcpy(dPsi, kp.data(), h->NP * sizeof(double));
  return 0;
}

int ref_fluxes(ref_grmhd* h, double* const flux[24]) {
  if (!h || !flux) return -1;
  if (!h->have_metric || !h->have_prims) return -3;
  h->compute_fluxes();
  for (int d = 0; d < 3; d++)
    for (int r = 0; r < 8; r++)
      std::memcpy(flux[d * 8 + r], h->F[d][r].data(), h->NP * sizeof(double));
  return 0;
}

void ref_prim2con_pt(const double prim[8], const double metric[10], double gamma_ad,
                     double cons[8]) {
  prim2con(prim, unpack_metric(metric), gamma_ad, cons);
}

int ref_con2prim_pt(const double cons[8], const double metric[10], const ref_opts* o,
                    int masked, double prim_out[5], double cons_out[5], int* iters) {
  return con2prim(cons, cons + 5, unpack_metric(metric), *o, masked != 0, prim_out, cons_out,
                  iters);
}

int ref_con2prim_backup_pt(const double cons[8], const double metric[10], const ref_opts* o,
                           double prim_out[5], double cons_out[5], int* iters) {
  return con2prim(cons, cons + 5, unpack_metric(metric), *o, false, prim_out, cons_out, iters,
                  true);
}

int ref_con2prim1d_pt(const double cons[8], const double metric[10], const ref_opts* o,
                      double prim_out[5], int* iters) {
  double rho, v[3], eps;
  const bool ok = con2prim_1d(cons, cons + 5, unpack_metric(metric), *o, rho, v, eps, iters);
  prim_out[0] = rho; prim_out[1] = v[0]; prim_out[2] = v[1]; prim_out[3] = v[2];
  prim_out[4] = (o->gamma_ad - 1.0) * rho * eps;
  return ok ? 0 : 2;
}

void ref_c2p1d_relations_pt(const double cons[8], const double metric[10], const ref_opts* o,
                            double x, double out[3]) {
  // eq. (44) -> W^, eq. (45) -> eps^, eq. (43) -> f at a given x: pins of the restatement
  const Metric M = unpack_metric(metric);
  double gu[3][3];
  inv3(M.g, det3(M.g), gu);
  const double* S = cons + 1;
  const double* B = cons + 5;
  double S2 = 0, B2 = 0, BS = 0;
  for (int i = 0; i < 3; i++) {
    for (int j = 0; j < 3; j++) { S2 += gu[i][j] * S[i] * S[j]; B2 += M.g[i][j] * B[i] * B[j]; }
    BS += B[i] * S[i];
  }
  const double D = cons[0];
  C2P1D c;
  c.D = D; c.Gamma = o->gamma_ad; c.iw2min = 1.0 / sq(o->w_max);
  c.q = cons[4] / D; c.r = S2 / (D * D); c.s = B2 / D; c.t = BS / (D * std::sqrt(D));
  c.state(x, out[0], out[1]);
  out[2] = c.f(x);
}

void ref_flux_pt(int d, const double prim[8], const double metric[10], double gamma_ad,
                 double F[8]) {
  flux18(d, prim, unpack_metric(metric), gamma_ad, F);
}

void ref_speeds_pt(int d, const double prim[8], const double metric[10], double gamma_ad,
                   double lam[2]) {
  const Metric M = unpack_metric(metric);
  double gu[3][3];
  inv3(M.g, det3(M.g), gu);
  speeds(d, prim, M, gu[d][d], gamma_ad, lam);
}

void ref_riemann_pt(int d, const double primL[8], const double primR[8],
                    const double metric_face[10], const ref_opts* o, double Fhat[8]) {
  riemann(d, primL, primR, unpack_metric(metric_face), *o, Fhat);
}

void ref_source_pt(const double prim[8], const double metric[10], const double K[6],
                   const double dalpha[3], const double dbeta[9], const double dgam[18],
                   double gamma_ad, double S[5]) {
  double Kc[3][3], db[3][3], dg[3][3][3];
  Kc[0][0] = K[0]; Kc[0][1] = Kc[1][0] = K[1]; Kc[0][2] = Kc[2][0] = K[2];
  Kc[1][1] = K[3]; Kc[1][2] = Kc[2][1] = K[4]; Kc[2][2] = K[5];
  for (int j = 0; j < 3; j++) {
    for (int i = 0; i < 3; i++) db[j][i] = dbeta[3 * j + i];
    const double* q = dgam + 6 * j;
    dg[j][0][0] = q[0]; dg[j][0][1] = dg[j][1][0] = q[1]; dg[j][0][2] = dg[j][2][0] = q[2];
    dg[j][1][1] = q[3]; dg[j][1][2] = dg[j][2][1] = q[4]; dg[j][2][2] = q[5];
  }
  sources(prim, unpack_metric(metric), Kc, dalpha, db, dg, gamma_ad, S);
}

void ref_recon_line(int method, int flatten, int n, const double* q, const double* press,
                    const double* vnorm, double* qL, double* qR) {
  for (int f = 3; f <= n - 3; f++) {
    if (method == 0) {
      double qm, qp;
      minmod_cell(q + f - 2, qm, qp); qL[f] = qp;
      minmod_cell(q + f - 1, qm, qp); qR[f] = qm;
    } else {
      double fL = 0, fR = 0, qm, qp;
      if (flatten) {
        fL = ppm_flat(press + f - 3, vnorm[f - 2], vnorm[f]);
        fR = ppm_flat(press + f - 2, vnorm[f - 1], vnorm[f + 1]);
      }
      ppm_cell(q + f - 3, fL, qm, qp); qL[f] = qp;
      ppm_cell(q + f - 2, fR, qm, qp); qR[f] = qm;
    }
  }
}

}  // extern "C"

// flux_face.cuh -- the per-face and per-cell arithmetic both flux kernels share (A3 + A4):
// branch-free reconstruction steps (R5 / G7 / G8), one side of a face (R2, R3, R6: eqs (13),
// (18), (20)-(22), (37) of PAPER.md:102-133, 266), the HLLE / LxF combination (R7: eqs (29),
// (30)) and the upwind-CT face rows (eqs (33), (34)).
//
// The face metric is STATIC (the ADM variables are input, held fixed): the
// 4-point Lagrange values of R4 and sqrt(gamma_f) are field family F_FM, written once by
// k_face_metric (kernels_aux.cuh) when the metric is set; a face costs 11 loads instead of a
// 40-value stencil, 40 interpolation FMAs, a determinant and a reciprocal square root.
#pragma once
#include "kernels_aux.cuh"

namespace gk {

constexpr int FX_NV = 7;  // reconstructed variables: rho, v^x, v^y, v^z, p and the two
                          // transverse B (the normal B is the staggered face value, G6)

__device__ __forceinline__ int flux_var_field(int D, int slot) {
  // slots 0..4 = rho, v^x, v^y, v^z, p; 5, 6 = B^{(D+1)%3}, B^{(D+2)%3} at cell centres
  return slot < 5 ? F_P + slot : F_BC + (D + 1 + (slot - 5)) % 3;
}
__host__ __device__ constexpr int flux_field(int D) { return D == 0 ? F_FX : (D == 1 ? F_FY : F_FZ); }

// ---- branch-free reconstruction ------------------------------------------------------------
// select that stays a select (the compiler turns ?: chains of the limiter into branches)
__device__ __forceinline__ double ft_sel(bool c, double a, double b) {
  double r;
  asm("{\n.reg .pred p;\nsetp.ne.s32 p, %3, 0;\nselp.f64 %0, %1, %2, p;\n}"
      : "=d"(r) : "d"(a), "d"(b), "r"((int)c));
  return r;
}

// G8(a): TWICE the monotonised-central slope from the two one-sided differences (the factor 2
// is an exact scaling: it saves the halving of the central difference and is undone by the 1/12
// of ft_iface).  For same-signed dm, dp the candidates dp+dm and 4 min(|dp|,|dm|) carry the sign
// of the slope already; if one of them is zero so is the candidate chosen, so "dp dm > 0"
// reduces to a sign-bit test.
__device__ __forceinline__ double ft_slope2(double dm, double dp) {
  const double s = dp + dm;
  const double m = fabs(dp) < fabs(dm) ? dp : dm;
  const double m4 = 4.0 * m;
  const double r = fabs(s) < fabs(m4) ? s : m4;
  return ft_opposite(dp, dm) ? 0.0 : r;
}
// G8(b): 4th-order interface value between cells (qa | qb) from their doubled slopes:
// (qa + qb)/2 - (dm_b - dm_a)/6
__device__ __forceinline__ double ft_iface(double qa, double qb, double s2a, double s2b) {
  return 0.5 * (qa + qb) - (s2b - s2a) * (1.0 / 12.0);
}

// G8(c, d) on the two interface values of a cell: flatten (f = 0 leaves the values untouched
// exactly; anyf = some lane of the warp has f != 0), then monotonise with a = q^+ - q,
// b = q - q^-: a b <= 0 -> flat; |b| > 2|a| -> q^- = q - 2a; |a| > 2|b| -> q^+ = q + 2b (the
// Colella-Woodward conditions in the form that needs no product of differences).
template <bool FLATTEN>
__device__ __forceinline__ void ft_parabola(double q, double f, bool anyf, double& qm, double& qp) {
  if (FLATTEN && anyf) {
    const double qpf = f * q + (1.0 - f) * qp;
    const double qmf = f * q + (1.0 - f) * qm;
    qp = f != 0.0 ? qpf : qp;
    qm = f != 0.0 ? qmf : qm;
  }
  const double a = qp - q, b = q - qm;
  const double aa = fabs(a), ab = fabs(b);
  // a b <= 0: with a = 0 or b = 0 the two fixes below give q as well, so the sign bits decide
  const bool flat = ft_opposite(a, b);
  const bool fixm = ab > 2.0 * aa;
  const bool fixp = aa > 2.0 * ab;
  const double qm2 = fma(-2.0, a, q);
  const double qp2 = fma(2.0, b, q);
  qm = ft_sel(flat, q, ft_sel(fixm, qm2, qm));
  qp = ft_sel(flat, q, ft_sel(fixp, qp2, qp));
}

// Reconstruction state of one variable on one pencil, carried from cell to cell: every
// limited slope, interface value and parabola is formed exactly once.
// RECON: 0 minmod, 1 PPM without flattening, 2 PPM with flattening.
template <int RECON>
struct FtMarch {
  double qa, qb;  // q_c, q_{c+1}
  double dl;      // q_c - q_{c-1}
  double s0;      // PPM: twice the limited slope of cell c
  double il;      // PPM: interface value at c - 1/2
  double qpp;     // q^+ of the previous cell (left state of the next face to be stored)
  // q0..q3 = cells c-2, c-1, c, c+1 where c is the first cell to be processed
  __device__ __forceinline__ void init(double q0, double q1, double q2, double q3) {
    qa = q2; qb = q3; qpp = 0.0;
    dl = q2 - q1;
    if (RECON == 0) {
      s0 = 0.0; il = 0.0;
    } else {
      const double d01 = q1 - q0;
      const double dmA = ft_slope2(d01, dl);
      s0 = ft_slope2(dl, q3 - q2);
      il = ft_iface(q1, q2, dmA, s0);
    }
  }
  // process cell c given qn = q_{c+2} and the flattening coefficient f of cell c
  __device__ __forceinline__ void step(double qn, double f, bool anyf, double& qm, double& qp) {
    const double dr = qb - qa;
    if (RECON == 0) {
      // G7
      const double m = fabs(dl) < fabs(dr) ? dl : dr;
      const double s = dl * dr > 0.0 ? m : 0.0;
      qm = fma(-0.5, s, qa);
      qp = fma(0.5, s, qa);
    } else {
      const double dmn = ft_slope2(dr, qn - qb);       // (doubled) slope of cell c+1
      const double ir = ft_iface(qa, qb, s0, dmn);      // interface c + 1/2, G8(b)
      qm = il; qp = ir;
      ft_parabola<RECON == 2>(qa, f, anyf, qm, qp);
      s0 = dmn; il = ir;
    }
    dl = dr; qa = qb; qb = qn;
  }
};

// G8(c): flattening coefficient of a cell from p_{c-2}, p_{c-1}, p_{c+1}, p_{c+2} and the
// normal velocities v_{c-1}, v_{c+1}
// Called by whole warps: where no lane sees the shock switch the coefficient is 0 without the
// division.
__device__ __forceinline__ double ft_flatten(double pm2, double pm1, double pp1, double pp2,
                                             double vm1, double vp1) {
  const double dp1 = pp1 - pm1;
  const bool on = fabs(dp1) > 0.33 * ft_min(pp1, pm1) && vm1 > vp1;
  if (!__any_sync(0xffffffffu, on)) return 0.0;
  const double dp2 = pp2 - pm2;
  const bool z = dp2 == 0.0;
  const double r = ft_rcp(z ? 1.0 : dp2);
  double f = 10.0 * fma(dp1, r, -0.75);
  f = ft_min(1.0, ft_max(0.0, f));
  f = z ? 1.0 : f;
  return on ? f : 0.0;
}

// ---- static face metric ----------------------------------------------------------------------
struct FaceMet {
  Met M;
  double sg;   // sqrt(gamma_f)
  double isg;  // 1/sqrt(gamma_f)
  double gdd;  // gamma^{DD}_f (R4: the speeds along D need nothing else of the inverse)
};
// v[0..10] = the F_FM values of the face (alpha, beta^i, gamma_ij, sqrt(gamma))
template <int D>
__device__ __forceinline__ FaceMet face_met(const double v[NFM]) {
  FaceMet f;
  f.M.a = v[0]; f.M.bx = v[1]; f.M.by = v[2]; f.M.bz = v[3];
  f.M.gxx = v[4]; f.M.gxy = v[5]; f.M.gxz = v[6]; f.M.gyy = v[7]; f.M.gyz = v[8]; f.M.gzz = v[9];
  f.sg = v[10];
  f.isg = ft_rcp(f.sg);
  f.gdd = inv_gamma_dd<D>(f.M, f.isg * f.isg);
  return f;
}

// ---- one side of a face ----------------------------------------------------------------------
// R5 (floors, velocity cap) on the reconstructed state, then U = (D, S_j, tau, B^t1, B^t2) of
// eqs (20)-(22), the coordinate flux G = alpha F^D of eq. (18) (the alpha: reading G10) and the
// speeds of R6 / G9.  Written for a low FP64 instruction count (the kernels run against the
// power cap: every instruction counts):
//   * S_j in the form of eq. (38), S_j = (z + B^2) v_j - (B^i v_i) B_j with z = rho h W^2
//     (PAPER.md:268), which needs neither b_j nor alpha b^0; likewise
//     tau = (z + B^2) - (p + b^2/2) - D   since (rho h + b^2) W^2 - (alpha b^0)^2 = z + B^2;
//   * b_j alpha B^d / W = alpha B^d (B_j / W^2 + (B^i v_i) v_j)  and  alpha b^0 alpha B^d / W =
//     alpha B^d (B^i v_i)  (eq. 37 with alpha b^0 = W B^i v_i, eq. 13);
//   * B_j = gamma_jk B^k with the normal-field part gamma_jD B^D formed once per face (gBn: the
//     staggered normal field is the same on both sides, G6);
//   * the speeds over one denominator:
//       a^2 = N/Dn, N = Gamma p e + b^2 (rho h - Gamma p), Dn = rho h e, e = rho h + b^2
//       lambda_pm = alpha (v^d (Dn-N) +- sqrt(N (1-v^2) (g^dd (Dn - v^2 N) - (v^d)^2 (Dn-N))))
//                   / (Dn - v^2 N) - beta^d
// Rows: 0 D, 1-3 S_j, 4 tau, 5 and 6 the transverse B^{(D+1)%3}, B^{(D+2)%3}.
// Bt1, Bt2 = those transverse components, Bn = B^D; vt (optional): v~^{(D+1)%3}, v~^{(D+2)%3}
// for eq. (33).
template <int D>
__device__ __forceinline__ void ft_side(double rho, double vx, double vy, double vz, double p,
                                        double Bt1, double Bt2, double Bn, const double gBn[3],
                                        const Met& M, double gdd, const Eos& E, double U[7],
                                        double Gf[7], double& lm, double& lp,
                                        double* vt = nullptr) {
  rho = rho < E.rho_atm ? E.rho_atm : rho;
  p = p < E.p_floor ? E.p_floor : p;
  double vlx, vly, vlz;
  lower(M, vx, vy, vz, vlx, vly, vlz);
  double v2 = vlx * vx + vly * vy + vlz * vz;
  if (v2 > E.v2max) {  // rare (R5: velocity cap on the reconstructed state)
    const double f = sqrt(E.v2max / v2);
    vx *= f; vy *= f; vz *= f;
    lower(M, vx, vy, vz, vlx, vly, vlz);
    v2 = vlx * vx + vly * vy + vlz * vz;
  }
  // B_j: transverse part here, normal part from gBn
  const double Bx = D == 0 ? Bn : (D == 1 ? Bt2 : Bt1);
  const double By = D == 1 ? Bn : (D == 2 ? Bt2 : Bt1);
  const double Bz = D == 2 ? Bn : (D == 0 ? Bt2 : Bt1);
  double Blx, Bly, Blz;
  if (D == 0) {
    Blx = fma(M.gxz, Bz, fma(M.gxy, By, gBn[0]));
    Bly = fma(M.gyz, Bz, fma(M.gyy, By, gBn[1]));
    Blz = fma(M.gzz, Bz, fma(M.gyz, By, gBn[2]));
  } else if (D == 1) {
    Blx = fma(M.gxz, Bz, fma(M.gxx, Bx, gBn[0]));
    Bly = fma(M.gyz, Bz, fma(M.gxy, Bx, gBn[1]));
    Blz = fma(M.gzz, Bz, fma(M.gxz, Bx, gBn[2]));
  } else {
    Blx = fma(M.gxy, By, fma(M.gxx, Bx, gBn[0]));
    Bly = fma(M.gyy, By, fma(M.gxy, Bx, gBn[1]));
    Blz = fma(M.gyz, By, fma(M.gxz, Bx, gBn[2]));
  }
  const double B2 = Blx * Bx + Bly * By + Blz * Bz;
  const double Bv = Bx * vlx + By * vly + Bz * vlz;   // B^i v_i
  const double iW2 = 1.0 - v2;
  const double W = ft_rsqrt(iW2);
  const double rhoh = rho + E.GoGm1 * p;        // eq. (46) with h = 1 + eps + p/rho
  const double z = rhoh * (W * W);              // eq. (36)
  const double b2 = fma(B2, iW2, Bv * Bv);      // eq. (13): b^2 = B^2/W^2 + (B^i v_i)^2
  const double X = z + B2;
  const double ptot = fma(0.5, b2, p);
  U[0] = rho * W;
  U[1] = X * vlx - Bv * Blx;                    // eq. (38)
  U[2] = X * vly - Bv * Bly;
  U[3] = X * vlz - Bv * Blz;
  U[4] = X - ptot - U[0];
  const double vtx = M.a * vx - M.bx, vty = M.a * vy - M.by, vtz = M.a * vz - M.bz;
  const double vtd = D == 0 ? vtx : (D == 1 ? vty : vtz);
  const double vd = D == 0 ? vx : (D == 1 ? vy : vz);
  const double aBd = M.a * Bn;
  const double c1 = aBd * iW2, c2 = aBd * Bv;
  const double ap = M.a * ptot;
  Gf[0] = U[0] * vtd;
  Gf[1] = U[1] * vtd - fma(c2, vlx, c1 * Blx) + (D == 0 ? ap : 0.0);
  Gf[2] = U[2] * vtd - fma(c2, vly, c1 * Bly) + (D == 1 ? ap : 0.0);
  Gf[3] = U[3] * vtd - fma(c2, vlz, c1 * Blz) + (D == 2 ? ap : 0.0);
  Gf[4] = fma(U[4], vtd, fma(ap, vd, -c2));
  const double vt1 = D == 0 ? vty : (D == 1 ? vtz : vtx);
  const double vt2 = D == 0 ? vtz : (D == 1 ? vtx : vty);
  if (vt) { vt[0] = vt1; vt[1] = vt2; }
  U[5] = Bt1; U[6] = Bt2;
  Gf[5] = Bt1 * vtd - Bn * vt1;
  Gf[6] = Bt2 * vtd - Bn * vt2;
  const double e = rhoh + b2;
  const double Gp = E.Gamma * p;
  const double N = Gp * e + b2 * (rhoh - Gp);
  const double Dn = rhoh * e;
  const double DmN = Dn - N;
  const double den = Dn - v2 * N;
  double rad = N * iW2 * (gdd * den - vd * vd * DmN);
  rad = rad < 0.0 ? 0.0 : rad;
  const double root = ft_sqrt(rad);
  const double aod = M.a * ft_rcp(den);
  const double mid = vd * DmN;
  const double bd = D == 0 ? M.bx : (D == 1 ? M.by : M.bz);
  lm = aod * (mid - root) - bd;
  lp = aod * (mid + root) - bd;
}

// R7 (eq. 29 / eq. 30): out[r] = sqrt(gamma_f) * F^[r]; apm (optional) = a_+, a_- of eq. (34)
__device__ __forceinline__ void ft_hll(const double UL[7], const double GL[7], double lmL,
                                       double lpL, const double UR[7], const double GR[7],
                                       double lmR, double lpR, double sgf, int riemann,
                                       double out[7], double* apm = nullptr) {
  const double cmax = ft_max(0.0, ft_max(lpL, lpR));
  const double cmin = -ft_min(0.0, ft_min(lmL, lmR));
  if (apm) { apm[0] = cmax; apm[1] = cmin; }
  const double cs = cmax + cmin;
  if (riemann == 1) {  // eq. (30)
    const double cw = ft_max(cmax, cmin);
    const double hs = 0.5 * sgf;
#pragma unroll
    for (int r = 0; r < 7; r++) out[r] = hs * (GR[r] + GL[r] - cw * (UR[r] - UL[r]));
  } else {  // eq. (29); c_max + c_min < 1e-300: plain average
    const bool deg = cs < 1e-300;
    const double w = sgf * ft_rcp(deg ? 1.0 : cs);
    const double a = deg ? 0.5 * sgf : cmin * w;
    const double b = deg ? 0.5 * sgf : cmax * w;
    const double cc = deg ? 0.0 : cmax * cmin * w;
#pragma unroll
    for (int r = 0; r < 7; r++) out[r] = a * GR[r] + b * GL[r] - cc * (UR[r] - UL[r]);
  }
}

// Riemann problem of one face from the two reconstructed states (slots as flux_var_field) and
// the staggered normal field bf = B~^D of the face.  out = the 7 stored flux rows; with UCT also
// the upwind-CT face data w[4] = a_+, a_-, vbar^{(D+1)%3}, vbar^{(D+2)%3} (eqs 33, 34; the mean
// of the two sides when a_+ + a_- vanishes).
template <int D, bool UCT>
__device__ __forceinline__ void ft_face(const double qL[FX_NV], const double qR[FX_NV], double bf,
                                        const FaceMet& fm, const Eos& E, double out[7],
                                        double w[4]) {
  const double Bn = bf * fm.isg;  // G6
  // gamma_jD B^D, common to both sides
  const Met& M = fm.M;
  const double gBn[3] = {(D == 0 ? M.gxx : (D == 1 ? M.gxy : M.gxz)) * Bn,
                         (D == 0 ? M.gxy : (D == 1 ? M.gyy : M.gyz)) * Bn,
                         (D == 0 ? M.gxz : (D == 1 ? M.gyz : M.gzz)) * Bn};
  double UL[7], GL[7], UR[7], GR[7], lmL, lpL, lmR, lpR;
  double vtL[2], vtR[2], apm[2];
  ft_side<D>(qL[0], qL[1], qL[2], qL[3], qL[4], qL[5], qL[6], Bn, gBn, M, fm.gdd, E, UL, GL, lmL,
             lpL, UCT ? vtL : nullptr);
  ft_side<D>(qR[0], qR[1], qR[2], qR[3], qR[4], qR[5], qR[6], Bn, gBn, M, fm.gdd, E, UR, GR, lmR,
             lpR, UCT ? vtR : nullptr);
  ft_hll(UL, GL, lmL, lpL, UR, GR, lmR, lpR, fm.sg, E.riemann, out, UCT ? apm : nullptr);
  if (UCT) {
    const double cs = apm[0] + apm[1];
    const bool deg = cs < 1e-300;
    const double r = ft_rcp(deg ? 1.0 : cs);
    const double a = deg ? 0.5 : apm[0] * r, b = deg ? 0.5 : apm[1] * r;
    w[0] = apm[0];
    w[1] = apm[1];
    w[2] = a * vtL[0] + b * vtR[0];
    w[3] = a * vtL[1] + b * vtR[1];
  }
}

}  // namespace gk

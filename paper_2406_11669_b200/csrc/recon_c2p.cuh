// recon_c2p.cuh -- reconstruction (R5/G7/G8), con2prim (R14) and source terms (R9/G11).
// Device-only restatements of PAPER.md:190-192 (reconstruction), PAPER.md:256-295 +
// PAPER.md:326 (con2prim + atmosphere) and eq. (19) PAPER.md:125 (sources).
#pragma once
#include "phys.cuh"

namespace gk {

// ------------------------------------------------------------------------ reconstruction
// G7: minmod(a,b) = 0 if a*b <= 0 else sign(a) min(|a|,|b|)
__device__ __forceinline__ double minmod(double a, double b) {
  if (a * b <= 0.0) return 0.0;
  const double m = fmin(fabs(a), fabs(b));
  return a > 0.0 ? m : -m;
}

// G8(a): monotonised central slope of a cell from its two neighbours.
__device__ __forceinline__ double ppm_slope(double qm1, double q0, double qp1) {
  const double dp = qp1 - q0, dm = q0 - qm1;
  if (dp * dm > 0.0) {
    const double d = 0.5 * (qp1 - qm1);
    const double lim = fmin(fabs(d), fmin(2.0 * fabs(dp), 2.0 * fabs(dm)));
    return d > 0.0 ? lim : -lim;
  }
  return 0.0;
}

// G8(c): flattening coefficient of a cell from p_{i-2..i+2} and v^d_{i-1}, v^d_{i+1}.
__device__ __forceinline__ double ppm_flatten(double pm2, double pm1, double pp1, double pp2,
                                              double vm1, double vp1) {
  const double dp1 = pp1 - pm1;
  const double dp2 = pp2 - pm2;
  if (fabs(dp1) > 0.33 * fmin(pp1, pm1) && vm1 > vp1) {
    if (dp2 == 0.0) return 1.0;
    const double f = 10.0 * (dp1 / dp2 - 0.75);
    return fmin(1.0, fmax(0.0, f));
  }
  return 0.0;
}

// G8(b): 4th-order interface value between cells (q0 | q1) from the two limited slopes.
__device__ __forceinline__ double ppm_iface(double q0, double q1, double dm0, double dm1) {
  return 0.5 * (q0 + q1) - (dm1 - dm0) * (1.0 / 6.0);
}

// G8(c,d): flatten + monotonise the parabola of one cell; qm = q^-_i, qp = q^+_i.
__device__ __forceinline__ void ppm_limit(double q0, double f, double& qm, double& qp) {
  qp = f * q0 + (1.0 - f) * qp;
  qm = f * q0 + (1.0 - f) * qm;
  if ((qp - q0) * (q0 - qm) <= 0.0) {
    qp = q0; qm = q0;
  } else {
    const double Dq = qp - qm;
    const double m = q0 - 0.5 * (qp + qm);
    const double D26 = Dq * Dq * (1.0 / 6.0);
    if (Dq * m > D26) qm = 3.0 * q0 - 2.0 * qp;
    else if (-D26 > Dq * m) qp = 3.0 * q0 - 2.0 * qm;
  }
}

// Face states of one variable from the 6 cells c[0..5] = f-3..f+2 around face f:
// qL from cell f-1, qR from cell f.  fL/fR are the flattening coefficients of those cells.
__device__ __forceinline__ void recon_pair(int recon, const double c[6], double fL, double fR,
                                           double& qL, double& qR) {
  if (recon == 0) {
    qL = c[2] + 0.5 * minmod(c[2] - c[1], c[3] - c[2]);
    qR = c[3] - 0.5 * minmod(c[3] - c[2], c[4] - c[3]);
  } else {
    const double d1 = ppm_slope(c[0], c[1], c[2]);
    const double d2 = ppm_slope(c[1], c[2], c[3]);
    const double d3 = ppm_slope(c[2], c[3], c[4]);
    const double d4 = ppm_slope(c[3], c[4], c[5]);
    const double i12 = ppm_iface(c[1], c[2], d1, d2);  // interface f-3/2
    const double i23 = ppm_iface(c[2], c[3], d2, d3);  // interface f-1/2 (this face)
    const double i34 = ppm_iface(c[3], c[4], d3, d4);  // interface f+1/2
    double qm = i12, qp = i23;
    ppm_limit(c[2], fL, qm, qp);
    qL = qp;
    qm = i23; qp = i34;
    ppm_limit(c[3], fR, qm, qp);
    qR = qm;
  }
}

// --------------------------------------------------------- con2prim, 1-D backup scheme
// Row F4: the scheme of PAPER.md:297-320 (eqs 42-45) the paper falls back to when the 2-D
// Newton iteration fails.  One unknown x = h W, bracketed by
// max(1 + q - s, 1) < x < 2 + 2q - s, root of eq. (43) by Brent's method.  Readings G23-G25 of
// DESIGN.md (t^2/x^2 in eq. (45); 1/W^2 kept in [1/w_max^2, 1]; eps^ >= 0 while iterating).
// Rare path: plain IEEE division and square root, not inlined.
struct C2p1d {
  double q, r, s, t, Gamma, iw2min;
  __device__ void state(double x, double& W, double& eps) const {
    double iw2 = 1.0 - (r * x * x + t * t * (2.0 * x + s)) / (x * x * (x + s) * (x + s));  // (44)
    iw2 = fmin(fmax(iw2, iw2min), 1.0);
    W = 1.0 / sqrt(iw2);
    eps = -1.0 + x / W * (1.0 - W * W) +
          W * (1.0 + q - s + 0.5 * (t * t / (x * x) + s * iw2));  // (45)
    eps = fmax(eps, 0.0);
  }
  __device__ double f(double x) const {  // (43), h^ = 1 + Gamma eps^ for the ideal fluid
    double W, eps;
    state(x, W, eps);
    return x - (1.0 + Gamma * eps) * W;
  }
};

// U = undensitised (D, S_j, tau).  Returns true and rho, v^i, eps on success.
__device__ __noinline__ bool con2prim_1d(const double* U, double Bx, double By, double Bz,
                                         const Met& M, const Eos& E, double& rho, double& vx,
                                         double& vy, double& vz, double& eps, int& iters) {
  const double D = U[0], Sx = U[1], Sy = U[2], Sz = U[3], tau = U[4];
  const double idet = 1.0 / det_gamma(M);
  const Sym3 gu = inv_gamma(M, idet);
  const double Sux = gu.xx * Sx + gu.xy * Sy + gu.xz * Sz;
  const double Suy = gu.xy * Sx + gu.yy * Sy + gu.yz * Sz;
  const double Suz = gu.xz * Sx + gu.yz * Sy + gu.zz * Sz;
  const double S2 = Sux * Sx + Suy * Sy + Suz * Sz;
  double Blx, Bly, Blz;
  lower(M, Bx, By, Bz, Blx, Bly, Blz);
  const double B2 = Blx * Bx + Bly * By + Blz * Bz;
  const double BS = Bx * Sx + By * Sy + Bz * Sz;
  C2p1d c;  // eq. (42)
  c.Gamma = E.Gamma; c.iw2min = 1.0 - E.v2max;
  c.q = tau / D; c.r = S2 / (D * D); c.s = B2 / D; c.t = BS / (D * sqrt(D));
  double a = fmax(1.0 + c.q - c.s, 1.0), b = 2.0 + 2.0 * c.q - c.s;
  iters = 0;
  if (!(b > a)) return false;
  // Brent: bracket [b, cc] with |f(b)| <= |f(cc)|, a = previous iterate
  double fa = c.f(a), fb = c.f(b);
  bool found = false;
  double x = 0.0;
  if (fa == 0.0) { x = a; found = true; }
  else if (fb == 0.0) { x = b; found = true; }
  else if (!(fa * fb < 0.0)) return false;
  double cc = a, fc = fa, d = b - a, e = d;
  for (int it = 1; it <= 100 && !found; it++) {
    iters = it;
    if ((fb > 0.0) == (fc > 0.0)) { cc = a; fc = fa; d = b - a; e = d; }
    if (fabs(fc) < fabs(fb)) { a = b; b = cc; cc = a; fa = fb; fb = fc; fc = fa; }
    const double tol1 = 2.0 * 2.220446049250313e-16 * fabs(b) + 0.5 * 1e-14 * fabs(b);
    const double xm = 0.5 * (cc - b);
    if (fabs(xm) <= tol1 || fb == 0.0) { x = b; found = true; break; }
    if (fabs(e) >= tol1 && fabs(fa) > fabs(fb)) {
      const double sv = fb / fa;
      double pp, qq;
      if (a == cc) {
        pp = 2.0 * xm * sv;
        qq = 1.0 - sv;
      } else {
        const double qa = fa / fc, rr = fb / fc;
        pp = sv * (2.0 * xm * qa * (qa - rr) - (b - a) * (rr - 1.0));
        qq = (qa - 1.0) * (rr - 1.0) * (sv - 1.0);
      }
      if (pp > 0.0) qq = -qq;
      pp = fabs(pp);
      if (2.0 * pp < fmin(3.0 * xm * qq - fabs(tol1 * qq), fabs(e * qq))) { e = d; d = pp / qq; }
      else { d = xm; e = d; }
    } else {
      d = xm; e = d;
    }
    a = b; fa = fb;
    b += fabs(d) > tol1 ? d : (xm > 0.0 ? tol1 : -tol1);
    fb = c.f(b);
  }
  if (!found || !isfinite(x)) return false;
  double W;
  c.state(x, W, eps);
  rho = D / W;
  const double z = D * x;  // (vii): z = rho W x
  const double izB = 1.0 / (z + B2), BSz = BS / z;
  vx = (Sux + BSz * Bx) * izB;  // eq. (41c)
  vy = (Suy + BSz * By) * izB;
  vz = (Suz + BSz * Bz) * izB;
  return isfinite(rho) && isfinite(eps) && isfinite(vx) && isfinite(vy) && isfinite(vz);
}

// ---------------------------------------------------------------------------- con2prim
// R14: Noble 2-D Newton-Raphson on (z, v^2), eqs (36)-(41) PAPER.md:260-295; atmosphere
// PAPER.md:326; failure policy G17-G20.  U = undensitised (D,S_j,tau) in/out, B^i, metric.
// Returns status bits: 1 atmosphere, 2 failed solve, 4 pressure fix, 8 W cap.
// `rewrite` mask tells which of U changed: bit0 -> D, bit1 -> S_j and tau.
// BACKUP (compile time, so that the default kernel carries no call frame): on a failure of
// the Newton iteration try con2prim_1d before giving up; status bit 16 = recovered that way.
template <bool BACKUP = false>
__device__ __forceinline__ int con2prim(double U[5], double Bx, double By, double Bz,
                                        const Met& M, const Eos& E, bool masked, double P5[5],
                                        int& iters, int& rewrite) {
  iters = 0;
  rewrite = 0;
  int bits = 0;
  const double D = U[0], tau = U[4];
  bool atmo = masked || !(D > E.rho_atm);
  if (atmo) bits = 1;
  double rho = 0, vx = 0, vy = 0, vz = 0, p = 0;
  if (!atmo) {
    const double idet = ft_rcp(det_gamma(M));
    const Sym3 gu = inv_gamma(M, idet);
    const double Sx = U[1], Sy = U[2], Sz = U[3];
    const double Sux = gu.xx * Sx + gu.xy * Sy + gu.xz * Sz;  // S^i
    const double Suy = gu.xy * Sx + gu.yy * Sy + gu.yz * Sz;
    const double Suz = gu.xz * Sx + gu.yz * Sy + gu.zz * Sz;
    const double S2 = Sux * Sx + Suy * Sy + Suz * Sz;
    double Blx, Bly, Blz;
    lower(M, Bx, By, Bz, Blx, Bly, Blz);
    const double B2 = Blx * Bx + Bly * By + Blz * Bz;
    const double BS = Bx * Sx + By * Sy + Bz * Sz;
    const double BS2 = BS * BS;
    const double g1 = E.gm1oG;
    double z = tau + D, v2 = 0.0;  // G17: stateless initial guess
    double iz = ft_rcp(z);         // 1/z, carried from the convergence test of the last iterate
    bool conv = false;
    for (int it = 1; it <= E.c2p_maxit; it++) {
      iters = it;
      const double omv = 1.0 - v2;
      const double W = ft_rsqrt(omv);
      const double sw = omv * W;  // 1/W
      const double pz = g1 * (z * omv - D * sw);
      const double iz2 = iz * iz, BS2iz3 = BS2 * iz2 * iz;
      const double B2z = B2 + z;
      // eqs (40a), (40b) and their Jacobian
      const double f1 = v2 * B2z * B2z - BS2 * (B2 + 2.0 * z) * iz2 - S2;
      const double f2 = tau + D - 0.5 * B2 * (1.0 + v2) + 0.5 * BS2 * iz2 - z + pz;
      const double J11 = 2.0 * B2z * (v2 + BS2iz3);
      const double J12 = B2z * B2z;
      const double J21 = -BS2iz3 - 1.0 + g1 * omv;
      const double J22 = -0.5 * B2 + g1 * (0.5 * D * W - z);
      const double idetJ = ft_rcp(J11 * J22 - J12 * J21);
      const double dz = (f2 * J12 - f1 * J22) * idetJ;
      const double dv = (f1 * J21 - f2 * J11) * idetJ;
      const double zn = fabs(z + dz);
      const double vs = v2 + dv;
      const double vn = ft_min(ft_max(vs, 0.0), 1.0 - 1e-12);  // G18
      const double izn = ft_rcp(zn);
      const double err = fabs(dz) * izn + fabs(dv);
      z = zn; v2 = vn; iz = izn;
      if (!isfinite(err)) break;
      if (err < E.c2p_tol) { conv = true; break; }
    }
    bool have = conv && isfinite(z) && isfinite(v2);
    double eps = 0.0;
    if (have) {
      // eqs (41a)-(41d); G19: the 1/gamma of (41d) is 1/Gamma
      const double iW2 = 1.0 - v2;
      const double iW = iW2 * ft_rsqrt(iW2);
      rho = D * iW;
      const double izB = ft_rcp(z + B2);
      const double BSz = BS * iz;
      vx = (Sux + BSz * Bx) * izB;
      vy = (Suy + BSz * By) * izB;
      vz = (Suz + BSz * Bz) * izB;
      // z (1 - v^2)/rho = z/(D W)
      eps = (z * iW * ft_rcp(D) - 1.0) * (1.0 - E.gm1oG);
      p = (E.Gamma - 1.0) * rho * eps;
      have = isfinite(rho) && isfinite(p) && isfinite(vx) && isfinite(vy) && isfinite(vz) &&
             !(rho < E.rho_atm);
    }
    if (BACKUP && !have) {  // the 1-D scheme as backup (row F4)
      int it1;
      if (con2prim_1d(U, Bx, By, Bz, M, E, rho, vx, vy, vz, eps, it1) && !(rho < E.rho_atm)) {
        p = (E.Gamma - 1.0) * rho * eps;
        bits |= 16;
        have = true;
      }
    }
    if (!have) {
      atmo = true; bits = 2;
    } else {
      if (eps < 0.0 || p < E.p_floor) {  // G20 (ii): pressure fix, keep rho and v
        p = E.p_floor;
        bits |= 4;
      }
      double lx, ly, lz;
      lower(M, vx, vy, vz, lx, ly, lz);
      const double vv = lx * vx + ly * vy + lz * vz;
      if (vv > E.v2max) {  // R14 (8): Lorentz-factor cap
        const double f = sqrt(E.v2max / vv);
        vx *= f; vy *= f; vz *= f;
        bits |= 8;
      }
    }
  }
  if (atmo) {  // rho_atm, polytropic p, v = 0, B kept, cons recomputed
    rho = E.rho_atm; vx = vy = vz = 0.0; p = E.p_atm;
  }
  P5[0] = rho; P5[1] = vx; P5[2] = vy; P5[3] = vz; P5[4] = p;
  if (bits & (1 | 2 | 4 | 8)) {
    Prim P = {rho, vx, vy, vz, p, Bx, By, Bz};
    double Un[5];
    prim2con(P, M, E, Un);
    if (bits & (1 | 2 | 8)) { U[0] = Un[0]; rewrite |= 1; }  // pressure fix alone keeps D
    U[1] = Un[1]; U[2] = Un[2]; U[3] = Un[3]; U[4] = Un[4];
    rewrite |= 2;
  }
  return bits;
}

// ----------------------------------------------------------------------------- sources
// R9 / G11: S of eq. (19) PAPER.md:125 in its exact 3+1 reduction, split in two parts so
// that derivatives can be consumed one axis at a time:
//   S_j   = C^{ik} d_j gamma_ik - T^{00} alpha d_j alpha + T^0_i d_j beta^i
//   S_tau = 2 C^{ik} K_ik - (T^{00} beta^i + T^{0i}) d_i alpha
// with C^{ik} = 1/2 (T^{00} beta^i beta^k + T^{0i} beta^k + T^{0k} beta^i + T^{ik}).
struct SrcCoef {
  Sym3 C;                 // C^{ik}
  double T00a;            // T^{00} alpha
  double T0lx, T0ly, T0lz;  // T^0_i = T^{00} beta_i + T^{0k} gamma_ki
  double ax, ay, az;      // T^{00} beta^i + T^{0i}
};

__device__ __forceinline__ SrcCoef source_coef(const Prim& P, const Met& M, const Eos& E) {
  const Pt s = point_state(P, M, E);
  const double ia = ft_rcp(M.a), ia2 = ia * ia;
  const double idet = ft_rcp(det_gamma(M));
  const Sym3 gu = inv_gamma(M, idet);
  // four-velocity and comoving field, eq. (13)
  const double u0 = s.W * ia;
  const double ux = s.W * (P.vx - M.bx * ia), uy = s.W * (P.vy - M.by * ia),
               uz = s.W * (P.vz - M.bz * ia);
  const double b0 = s.ab0 * ia;
  const double bx = (P.Bx + s.ab0 * ux) * s.iW, by = (P.By + s.ab0 * uy) * s.iW,
               bz = (P.Bz + s.ab0 * uz) * s.iW;
  const double e = s.rhoh + s.b2, pt = P.p + 0.5 * s.b2;
  // T^{mu nu}, eq. (16), with g^{00} = -1/alpha^2, g^{0i} = beta^i/alpha^2,
  // g^{ij} = gamma^{ij} - beta^i beta^j/alpha^2
  const double T00 = e * u0 * u0 - pt * ia2 - b0 * b0;
  const double T0x = e * u0 * ux + pt * M.bx * ia2 - b0 * bx;
  const double T0y = e * u0 * uy + pt * M.by * ia2 - b0 * by;
  const double T0z = e * u0 * uz + pt * M.bz * ia2 - b0 * bz;
  const double pia2 = pt * ia2;
  const double Txx = e * ux * ux + pt * gu.xx - pia2 * M.bx * M.bx - bx * bx;
  const double Txy = e * ux * uy + pt * gu.xy - pia2 * M.bx * M.by - bx * by;
  const double Txz = e * ux * uz + pt * gu.xz - pia2 * M.bx * M.bz - bx * bz;
  const double Tyy = e * uy * uy + pt * gu.yy - pia2 * M.by * M.by - by * by;
  const double Tyz = e * uy * uz + pt * gu.yz - pia2 * M.by * M.bz - by * bz;
  const double Tzz = e * uz * uz + pt * gu.zz - pia2 * M.bz * M.bz - bz * bz;
  SrcCoef c;
  c.ax = T00 * M.bx + T0x; c.ay = T00 * M.by + T0y; c.az = T00 * M.bz + T0z;
  // C^{ik} = 1/2 (beta^i a^k + T^{0k} beta^i ... ) written symmetrically:
  // T00 b^i b^k + T0i b^k + T0k b^i = a^i b^k + T0k b^i
  c.C.xx = 0.5 * (c.ax * M.bx + T0x * M.bx + Txx);
  c.C.xy = 0.5 * (c.ax * M.by + T0y * M.bx + Txy);
  c.C.xz = 0.5 * (c.ax * M.bz + T0z * M.bx + Txz);
  c.C.yy = 0.5 * (c.ay * M.by + T0y * M.by + Tyy);
  c.C.yz = 0.5 * (c.ay * M.bz + T0z * M.by + Tyz);
  c.C.zz = 0.5 * (c.az * M.bz + T0z * M.bz + Tzz);
  c.T00a = T00 * M.a;
  // T^0_i = gamma_ik (T^{00} beta^k + T^{0k})
  lower(M, c.ax, c.ay, c.az, c.T0lx, c.T0ly, c.T0lz);
  return c;
}

__device__ __forceinline__ double contract(const Sym3& C, double xx, double xy, double xz,
                                           double yy, double yz, double zz) {
  return C.xx * xx + C.yy * yy + C.zz * zz + 2.0 * (C.xy * xy + C.xz * xz + C.yz * yz);
}

}  // namespace gk

// recon_c2p.cuh -- con2prim (R14) and source terms (R9/G11).
// Device-only restatements of PAPER.md:256-295 + PAPER.md:326 (con2prim + atmosphere) and
// eq. (19) PAPER.md:125 (sources).  (The reconstruction lives in flux_face.cuh.)
#pragma once
#include "phys.cuh"
#include "c2p_1d.cuh"

namespace gk {

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

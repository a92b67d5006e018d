// flux_tma.cuh -- A3 + A4: reconstruction + Riemann flux along direction D; marching form
// fed asynchronously (TMA ring for the face data, register prefetch for the cell data).
//
// Same thread mapping as flux_march.cuh (a block of 128 threads = 32 pencils x chunks of
// TC = 4 faces; phase A: warp = 2 reconstructed variables, lane = pencil; phase B: one thread
// per face), with what the ncu capture r1b asked for:
//  * no global load is waited for in the loop.  The face metric stencil (10 fields x 4 layers
//    along D, R4) and the staggered normal field arrive through a 3-slot shared-memory ring
//    filled by cp.async.bulk.tensor (one 4-D box [field][.][.][.] per chunk, completion on an
//    mbarrier), issued one chunk ahead by thread 0.  The cell-centred primitives of phase A are
//    prefetched one chunk ahead into registers (32-byte vector loads for D = x).
//  * the PPM limiter is branch free (selects), in the |b| > 2|a| form of the Colella-Woodward
//    monotonicity conditions (algebraically the conditions of DESIGN.md G8(d));
//    reciprocal, square root and reciprocal square root are the hardware seed + Newton steps
//    without special-case paths (operands are normal numbers by construction).
//  * all offsets inside a field are 32-bit.
// The block owns 32 consecutive transverse positions t0 (x for D = y, z; y for D = x) at one
// position t1 of the other transverse axis; the 1-cell flux-CT apron (R10) along t1 is part of
// the grid, the two apron columns along t0 are left to k_flux_march (apron mode).
#pragma once
#include <cuda.h>

#include "flux_math.cuh"
#include "flux_march.cuh"

namespace gk {

constexpr int FT_THREADS = 128;
constexpr int FT_TC = 4;
constexpr int FT_SLOTS = 3;
constexpr int FT_NMET = 10;
#ifndef FT_MINB
#define FT_MINB 3
#endif

template <int D>
struct FtSmem {
  static constexpr int P = D == 0 ? 36 : 32;  // pencil pitch of the exchange buffer
  // ring slots (TMA destinations, dense boxes): D = 0: [field][pencil][layer];
  // D = 1, 2: [field][layer][pencil]
  alignas(128) double met[FT_SLOTS][FT_NMET * FT_TC * 32];
  alignas(128) double bf[FT_SLOTS][FT_TC * 32];
  double q[2][FM_NV][2][FT_TC][P];  // [buffer][variable][L/R][face][pencil]
  double fl[2][FT_TC][32];
  double fl0[32];
  alignas(8) unsigned long long bar[FT_SLOTS];
};

// ---- PTX wrappers -------------------------------------------------------------------------
__device__ __forceinline__ unsigned ft_saddr(const void* p) {
  return (unsigned)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void ft_mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(ft_saddr(bar)), "r"(count));
}
__device__ __forceinline__ void ft_mbar_expect(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(ft_saddr(bar)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void ft_mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "FT_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra FT_DONE_%=;\n"
      "bra FT_WAIT_%=;\n"
      "FT_DONE_%=:\n"
      "}\n" ::"r"(ft_saddr(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void ft_tma_4d(void* dst, const CUtensorMap* tm,
                                          unsigned long long* bar, int c0, int c1, int c2,
                                          int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes "
      "[%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(ft_saddr(dst)),
      "l"(tm), "r"(ft_saddr(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}

// ---- branch-free reconstruction state of one variable on one pencil -------------------------

// select that stays a select (the compiler turns ?: chains of the limiter into branches)
__device__ __forceinline__ double ft_sel(bool c, double a, double b) {
  double r;
  asm("{\n.reg .pred p;\nsetp.ne.s32 p, %3, 0;\nselp.f64 %0, %1, %2, p;\n}"
      : "=d"(r) : "d"(a), "d"(b), "r"((int)c));
  return r;
}

// G8(a): monotonised-central slope from the two one-sided differences.  For same-signed
// dm, dp the candidates d = (dp+dm)/2 and 2 min(|dp|,|dm|) carry the sign of d already; if
// one of them is zero so is the candidate chosen, so "dp dm > 0" reduces to a sign-bit test.
__device__ __forceinline__ double ft_slope(double dm, double dp) {
  const double d = 0.5 * (dp + dm);
  const double m = fabs(dp) < fabs(dm) ? dp : dm;
  const double m2 = m + m;
  const double r = fabs(d) < fabs(m2) ? d : m2;
  return ft_opposite(dp, dm) ? 0.0 : r;
}

template <int RECON>
struct FtMarch {
  double qa, qb;  // q_c, q_{c+1}
  double dl;      // q_c - q_{c-1}
  double s0;      // PPM: limited slope of cell c
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
      const double dmA = ft_slope(d01, dl);
      s0 = ft_slope(dl, q3 - q2);
      il = 0.5 * (q1 + q2) - (s0 - dmA) * (1.0 / 6.0);
    }
  }
  // process cell c given qn = q_{c+2}, the flattening coefficient f of cell c and whether
  // any lane of the warp has f != 0
  __device__ __forceinline__ void step(double qn, double f, bool anyf, double& qm, double& qp) {
    const double dr = qb - qa;
    if (RECON == 0) {
      // G7
      const double m = fabs(dl) < fabs(dr) ? dl : dr;
      const double s = dl * dr > 0.0 ? m : 0.0;
      qm = fma(-0.5, s, qa);
      qp = fma(0.5, s, qa);
    } else {
      const double dmn = ft_slope(dr, qn - qb);                        // slope of cell c+1
      const double ir = 0.5 * (qa + qb) - (dmn - s0) * (1.0 / 6.0);  // interface c + 1/2
      qm = il; qp = ir;
      if (RECON == 2 && anyf) {  // G8(c); f = 0 leaves the values untouched exactly
        const double qpf = f * qa + (1.0 - f) * qp;
        const double qmf = f * qa + (1.0 - f) * qm;
        qp = f != 0.0 ? qpf : qp;
        qm = f != 0.0 ? qmf : qm;
      }
      // G8(d) with a = q^+ - q, b = q - q^-: a b <= 0 -> flat; |b| > 2|a| -> q^- = q - 2a;
      // |a| > 2|b| -> q^+ = q + 2b
      const double a = qp - qa, b = qa - qm;
      const double aa = fabs(a), ab = fabs(b);
      // a b <= 0: with a = 0 or b = 0 the two fixes below give q as well, so the sign bits decide
      const bool flat = ft_opposite(a, b);
      const bool fixm = ab > 2.0 * aa;
      const bool fixp = aa > 2.0 * ab;
      const double qm2 = fma(-2.0, a, qa);
      const double qp2 = fma(2.0, b, qa);
#ifndef FT_NO_SELP
      qm = ft_sel(flat, qa, ft_sel(fixm, qm2, qm));
      qp = ft_sel(flat, qa, ft_sel(fixp, qp2, qp));
#else
      qm = flat ? qa : (fixm ? qm2 : qm);
      qp = flat ? qa : (fixp ? qp2 : qp);
#endif
      s0 = dmn; il = ir;
    }
    dl = dr; qa = qb; qb = qn;
  }
};

// G8(c): flattening coefficient of cell c; marching over p_{c-2..c+2}, v_{c-1}, v_{c+1}
struct FtFlat {
  double pm2, pm1, p0, pp1, vm1, v0;
  __device__ __forceinline__ void init(double a, double b, double c, double d, double va,
                                       double vb) {
    pm2 = a; pm1 = b; p0 = c; pp1 = d; vm1 = va; v0 = vb;
  }
  // pn = p_{c+2}, vn = v_{c+1}
  __device__ __forceinline__ double step(double pn, double vn) {
    const double dp1 = pp1 - pm1;
    const double dp2 = pn - pm2;
    const bool on = fabs(dp1) > 0.33 * ft_min(pp1, pm1) && vm1 > vn;
    const bool z = dp2 == 0.0;
    const double r = ft_rcp(z ? 1.0 : dp2);
    double f = 10.0 * fma(dp1, r, -0.75);
    f = ft_min(1.0, ft_max(0.0, f));
    f = z ? 1.0 : f;
    pm2 = pm1; pm1 = p0; p0 = pp1; pp1 = pn;
    vm1 = v0; v0 = vn;
    return on ? f : 0.0;
  }
};

// one side of a face, as side_rows (flux_math.cuh) with the call-free special functions
template <int D>
__device__ __forceinline__ void ft_side(double rho, double vx, double vy, double vz, double p,
                                        double Bx, double By, double Bz, const Met& M,
                                        double gdd, const Eos& E, double U[7], double Gf[7],
                                        double& lm, double& lp, double* vt = nullptr) {
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
  double Blx, Bly, Blz;
  lower(M, Bx, By, Bz, Blx, Bly, Blz);
  const double B2 = Blx * Bx + Bly * By + Blz * Bz;
  const double Bv = Bx * vlx + By * vly + Bz * vlz;
  const double iW2 = 1.0 - v2;
  const double W = ft_rsqrt(iW2);
  const double iW = iW2 * W;
  const double ab0 = W * Bv;
  const double b2 = (B2 + ab0 * ab0) * iW2;
  const double blx = Blx * iW + ab0 * vlx;
  const double bly = Bly * iW + ab0 * vly;
  const double blz = Blz * iW + ab0 * vlz;
  const double rhoh = rho + E.GoGm1 * p;
  const double e = rhoh + b2;
  const double eW2 = e * W * W;
  const double ptot = p + 0.5 * b2;
  U[0] = rho * W;
  U[1] = eW2 * vlx - ab0 * blx;
  U[2] = eW2 * vly - ab0 * bly;
  U[3] = eW2 * vlz - ab0 * blz;
  U[4] = eW2 - ptot - ab0 * ab0 - U[0];
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
  if (vt) { vt[0] = vt1; vt[1] = vt2; }  // v~^{(D+1)%3}, v~^{(D+2)%3} for eq. (33)
  U[5] = B1; U[6] = B2t;
  Gf[5] = B1 * vtd - Bd * vt1;
  Gf[6] = B2t * vtd - Bd * vt2;
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

// R7 (eq. 29 / eq. 30): out[r] = sqrt(gamma_f) * F^[r]
__device__ __forceinline__ void ft_hll(const double UL[7], const double GL[7], double lmL,
                                       double lpL, const double UR[7], const double GR[7],
                                       double lmR, double lpR, double sgf, int riemann,
                                       double out[7], double* apm = nullptr) {
  const double cmax = ft_max(0.0, ft_max(lpL, lpR));
  const double cmin = -ft_min(0.0, ft_min(lmL, lmR));
  if (apm) { apm[0] = cmax; apm[1] = cmin; }  // a_+, a_- of eq. (34)
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

// Upwind-CT face data of direction D (row F1): a_+, a_- and eq. (33)
// vbar^j = (a_+ v~^jL + a_- v~^jR)/(a_+ + a_-), their mean when a_+ + a_- vanishes.
// o = address of this face in field F_W + 4 D.
__device__ __forceinline__ void ft_store_uct(double* o, size_t NPA, const double apm[2],
                                             const double vtL[2], const double vtR[2]) {
  const double cs = apm[0] + apm[1];
  const bool deg = cs < 1e-300;
  const double w = ft_rcp(deg ? 1.0 : cs);
  const double a = deg ? 0.5 : apm[0] * w, b = deg ? 0.5 : apm[1] * w;
  o[0] = apm[0];
  o[NPA] = apm[1];
  o[2 * NPA] = a * vtL[0] + b * vtR[0];
  o[3 * NPA] = a * vtL[1] + b * vtR[1];
}

// 32-byte global load of 4 consecutive doubles (address 32-byte aligned)
__device__ __forceinline__ void ft_ld4(const double* p, double& a, double& b, double& c,
                                       double& d) {
  asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];"
               : "=d"(a), "=d"(b), "=d"(c), "=d"(d)
               : "l"(p));
}

// RECON: 0 minmod, 1 PPM without flattening, 2 PPM with flattening.
// grid: x = (groups of 32 along t0) * (n_t1 + 2), y = segments of `seglen` faces (seglen a
// multiple of 4).  For D = 0 the march starts at face -2 so that every 4-cell group of a row
// is one 32-byte sector.
// UCT (compile time, so that the default kernel keeps its register budget): also store the
// upwind-CT face rows of F_W.
template <int D, int RECON, bool UCT>
__global__ void __launch_bounds__(FT_THREADS, UCT ? 2 : FT_MINB)
k_flux_tma(double* __restrict__ base, Geom g, Eos E, int seglen, int ngx, int ap,
           const __grid_constant__ CUtensorMap tmMet, const __grid_constant__ CUtensorMap tmBf) {
  using Smem = FtSmem<D>;
  constexpr int TC = FT_TC;
  constexpr int P = Smem::P;
  extern __shared__ __align__(128) unsigned char ft_smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(ft_smem_raw);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nD = g.n(D);
  const int nt0 = D == 0 ? g.ny : g.nx;
  const int sd = D == 0 ? 1 : (D == 1 ? (int)g.sy : (int)g.sz);
  const int gx = (int)blockIdx.x % ngx;
  const int t1 = (int)blockIdx.x / ngx - ap;  // ap = transverse apron: 1 (flux-CT), 3 (UCT)
  const int g0 = gx * 32;
  const int fbeg = D == 0 ? -2 : 0;
  const int f0 = fbeg + (int)blockIdx.y * seglen;
  const int f1 = min(f0 + seglen, nD + 1);
  const int cmax = nD + G - 1;  // last valid cell index along D
  const int nchunk = (f1 - f0 + TC - 1) / TC;

  // ---- ring: stage m holds layers f0 - 2 + 4m .. + 3 of the metric and of B~^D
  constexpr unsigned STAGE_BYTES = (FT_NMET + 1) * TC * 32 * sizeof(double);
  auto issue_stage = [&](int m) {
    const int slot = m % FT_SLOTS;
    const int L = f0 - 2 + TC * m;
    int c0, c1, c2;
    if (D == 0) { c0 = L + X0; c1 = g0 + G; c2 = t1 + G; }
    else if (D == 1) { c0 = g0 + X0; c1 = L + G; c2 = t1 + G; }
    else { c0 = g0 + X0; c1 = t1 + G; c2 = L + G; }
    ft_mbar_expect(&sm.bar[slot], STAGE_BYTES);
    ft_tma_4d(sm.met[slot], &tmMet, &sm.bar[slot], c0, c1, c2, F_MET);
    ft_tma_4d(sm.bf[slot], &tmBf, &sm.bar[slot], c0, c1, c2, F_BF + D);
  };
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < FT_SLOTS; s++) ft_mbar_init(&sm.bar[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
#pragma unroll
    for (int m = 0; m < FT_SLOTS; m++)
      if (m <= nchunk) issue_stage(m);
  }

  // ---- phase-A identity: lane = pencil
  const int pA = min(g0 + lane, nt0 - 1);
  const int baseA = (int)(D == 0 ? g.at(0, pA, t1) : (D == 1 ? g.at(pA, 0, t1) : g.at(pA, t1, 0)));
  const int s0 = 2 * warp, nslot = warp == 3 ? 1 : 2;
  const double* qsrc[2];
  qsrc[0] = fld(base, g, fm_var_field(D, s0)) + baseA;
  qsrc[1] = fld(base, g, fm_var_field(D, s0 + (nslot > 1 ? 1 : 0))) + baseA;
  const double* psrc = fld(base, g, F_P + 4) + baseA;
  const double* vsrc = fld(base, g, F_P + 1 + D) + baseA;

  // new cells of the chunk whose first face is F: cells F+2 .. F+5
  auto load_cells = [&](const double* q, int F, double out[TC]) {
    if (D == 0) {
      ft_ld4(q + (F + 2), out[0], out[1], out[2], out[3]);
    } else {
#pragma unroll
      for (int cl = 0; cl < TC; cl++) out[cl] = q[min(F + cl + 2, cmax) * sd];
    }
  };

  FtMarch<RECON> mv[2];
  FtFlat fmch;
  double nxt[2][TC];        // cells of the next chunk (prefetched)
  // ---- prologue: state before cell f0-1, flattening of f0-1 and of chunk 0
#pragma unroll
  for (int s = 0; s < 2; s++) {
    if (s < nslot) {
      const double* q = qsrc[s];
      mv[s].init(q[(f0 - 3) * sd], q[(f0 - 2) * sd], q[(f0 - 1) * sd], q[f0 * sd]);
    }
  }
  if (RECON == 2 && warp == 3) {
    const int c = f0 - 1;
    fmch.init(psrc[(c - 2) * sd], psrc[(c - 1) * sd], psrc[c * sd], psrc[(c + 1) * sd],
              vsrc[(c - 1) * sd], vsrc[c * sd]);
    sm.fl0[lane] = fmch.step(psrc[min(c + 2, cmax) * sd], vsrc[min(c + 1, cmax) * sd]);
#pragma unroll
    for (int cl = 0; cl < TC; cl++) {
      const int cc = f0 + cl;
      sm.fl[0][cl][lane] = fmch.step(psrc[min(cc + 2, cmax) * sd], vsrc[min(cc + 1, cmax) * sd]);
    }
  }
  __syncthreads();  // barrier init + fl0 / fl[0] visible
  {
    const bool anyf = RECON == 2 && __any_sync(0xffffffffu, sm.fl0[lane] != 0.0);
#pragma unroll
    for (int s = 0; s < 2; s++) {
      if (s < nslot) {
        double qm, qp;
        mv[s].step(qsrc[s][min(f0 + 1, cmax) * sd], RECON == 2 ? sm.fl0[lane] : 0.0, anyf, qm, qp);
        mv[s].qpp = qp;
        load_cells(qsrc[s], f0, nxt[s]);
      }
    }
  }

  // ---- phase-B identity: one thread per face of the chunk, lanes along x
  int clB, plB;
  if (D == 0) { clB = tid % TC; plB = tid / TC; }
  else { plB = lane; clB = warp; }
  const bool okB = g0 + plB < nt0;
  // output offset = block-uniform part + a term rebuilt from the thread index when needed
  // (nothing to keep in a register across the loop)
  const long long ublk = D == 0 ? g.at(0, g0, t1) : (D == 1 ? g.at(g0, 0, t1) : g.at(g0, t1, 0));
  double* const outb = fld(base, g, D == 0 ? F_FX : (D == 1 ? F_FY : F_FZ)) + ublk;
  const size_t NPA = (size_t)g.NPA;
  // ring offsets of the thread: layer j = clB + k of the 8 resident ones
  constexpr int MF = TC * 32;  // doubles per field in a slot
  const int ringp = D == 0 ? plB * TC : plB;
  constexpr int ringl = D == 0 ? 1 : 32;

  int buf = 0;
  for (int n = 0; n < nchunk; n++, buf ^= 1) {
    const int F = f0 + n * TC;
    // ================= phase A: cells F .. F+TC-1 =================
    double cur[2][TC];
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
      for (int cl = 0; cl < TC; cl++) cur[s][cl] = nxt[s][cl];
    const bool more = n + 1 < nchunk;
#pragma unroll
    for (int s = 0; s < 2; s++)
      if (s < nslot && more) load_cells(qsrc[s], F + TC, nxt[s]);
    // warp 3 (one variable): inputs p_{c+2}, v_{c+1} of the flattening of the next chunk's
    // cells, in flight while its variable is reconstructed
    double pc[TC], vc[TC];
    if (RECON == 2 && warp == 3 && more) {
      load_cells(psrc, F + TC, pc);
#pragma unroll
      for (int cl = 0; cl < TC; cl++) vc[cl] = vsrc[min(F + TC + cl + 1, cmax) * sd];
    }
#pragma unroll
    for (int s = 0; s < 2; s++) {
      if (s < nslot) {
#pragma unroll
        for (int cl = 0; cl < TC; cl++) {
          const double f = RECON == 2 ? sm.fl[buf][cl][lane] : 0.0;
          const bool anyf = RECON == 2 && __any_sync(0xffffffffu, f != 0.0);
          double qm, qp;
          mv[s].step(cur[s][cl], f, anyf, qm, qp);
          sm.q[buf][s0 + s][0][cl][lane] = mv[s].qpp;  // left state of face F+cl
          sm.q[buf][s0 + s][1][cl][lane] = qm;         // right state of face F+cl
          mv[s].qpp = qp;
        }
      }
    }
    if (RECON == 2 && warp == 3 && more) {
#pragma unroll
      for (int cl = 0; cl < TC; cl++) sm.fl[buf ^ 1][cl][lane] = fmch.step(pc[cl], vc[cl]);
    }
    __syncthreads();  // A(n) and B(n-1) are complete in every warp
    if (tid == 0 && n >= 1 && n + 2 <= nchunk) issue_stage(n + 2);  // slot of stage n-1
    // ================= phase B: faces F .. F+TC-1 =================
    {
      const int sA = n % FT_SLOTS, sB = (n + 1) % FT_SLOTS;
      ft_mbar_wait(&sm.bar[sA], (unsigned)((n / FT_SLOTS) & 1));
      ft_mbar_wait(&sm.bar[sB], (unsigned)(((n + 1) / FT_SLOTS) & 1));
      const int f = F + clB;
      // layers f-2 .. f+1 = ring layers clB .. clB+3 counted from the first layer of stage n
      int off[4];
#pragma unroll
      for (int k = 0; k < 4; k++) {
        const int j = clB + k;
        off[k] = (j < TC ? sA : sB) * (FT_NMET * MF) + (j & (TC - 1)) * ringl + ringp;
      }
      const double* mr = &sm.met[0][0];
      double mq[FT_NMET];
#pragma unroll
      for (int v = 0; v < FT_NMET; v++) {
        const double q0 = mr[off[0] + v * MF], q1 = mr[off[1] + v * MF], q2 = mr[off[2] + v * MF],
                     q3 = mr[off[3] + v * MF];
        mq[v] = (-q0 + 9.0 * q1 + 9.0 * q2 - q3) * 0.0625;  // R4
      }
      Met M;
      M.a = mq[0]; M.bx = mq[1]; M.by = mq[2]; M.bz = mq[3];
      M.gxx = mq[4]; M.gxy = mq[5]; M.gxz = mq[6]; M.gyy = mq[7]; M.gyz = mq[8]; M.gzz = mq[9];
      const double det = det_gamma(M);
      const double isg = ft_rsqrt(det);
      const double sgf = det * isg;
      const double gdd = inv_gamma_dd<D>(M, isg * isg);
      const int jb = clB + 2;
      const double Bn =
          sm.bf[jb < TC ? sA : sB][(jb & (TC - 1)) * ringl + ringp] * isg;  // G6
      double qL[FM_NV], qR[FM_NV];
#pragma unroll
      for (int v = 0; v < FM_NV; v++) {
        qL[v] = sm.q[buf][v][0][clB][plB];
        qR[v] = sm.q[buf][v][1][clB][plB];
      }
      double UL[7], GL[7], UR[7], GR[7], lmL, lpL, lmR, lpR;
      double vtL[2], vtR[2], apm[2];
      ft_side<D>(qL[0], qL[1], qL[2], qL[3], qL[4], D == 0 ? Bn : (D == 1 ? qL[6] : qL[5]),
                 D == 1 ? Bn : (D == 2 ? qL[6] : qL[5]), D == 2 ? Bn : (D == 0 ? qL[6] : qL[5]),
                 M, gdd, E, UL, GL, lmL, lpL, UCT ? vtL : nullptr);
      ft_side<D>(qR[0], qR[1], qR[2], qR[3], qR[4], D == 0 ? Bn : (D == 1 ? qR[6] : qR[5]),
                 D == 1 ? Bn : (D == 2 ? qR[6] : qR[5]), D == 2 ? Bn : (D == 0 ? qR[6] : qR[5]),
                 M, gdd, E, UR, GR, lmR, lpR, UCT ? vtR : nullptr);
      double out[7];
      ft_hll(UL, GL, lmL, lpL, UR, GR, lmR, lpR, sgf, E.riemann, out, UCT ? apm : nullptr);
      if (okB && f >= 0 && f < f1) {
        const int pl = D == 0 ? tid / TC : (tid & 31);
        double* o = outb + (D == 0 ? pl * (int)g.sy + f : pl + f * sd);
#pragma unroll
        for (int r = 0; r < 7; r++) o[r * NPA] = out[r];
        if (UCT) {
          constexpr int fid = D == 0 ? F_FX : (D == 1 ? F_FY : F_FZ);
          ft_store_uct(o + (size_t)(F_W + 4 * D - fid) * NPA, NPA, apm, vtL, vtR);
        }
      }
    }
    // no barrier here: the next phase A writes the other exchange buffer
  }
}

}  // namespace gk

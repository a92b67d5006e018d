// flux_march.cuh -- A3 + A4: reconstruction + Riemann flux along direction D, marching form.
//
// Thread mapping.  A block of 128 threads (4 warps) owns one "pencil group": 32 pencils of cells
// running along D (transverse positions incl. the 1-cell apron flux-CT needs, R10, flattened
// to one index so that no lane idles at row ends) and a segment of faces [f0, f1) along D.
// It walks the segment in chunks of TC faces; face f is the face between cells f-1 and f.
//
//  phase A (reconstruction, R5): warp w owns the variables {2w, 2w+1} of the 7 reconstructed
//    ones (rho, v^x, v^y, v^z, p and the two transverse B; the normal B is the staggered face
//    value, G6); lane = pencil.  The PPM / minmod state of a variable is carried in
//    registers from cell to cell: every limited slope, interface value and parabola is
//    computed exactly once and every input double is loaded exactly once.  Cell c yields
//    q^-_c (right state of face c) and q^+_c (left state of face c+1); both go to shared
//    memory.  Warp 3 (one variable only) also computes the PPM flattening coefficients of the
//    NEXT chunk.
//  phase B (Riemann, R4 + R7): one thread per face (lanes along x, so global accesses are
//    coalesced for every D) reads both states from shared memory, interpolates the metric
//    to the face and stores the 7 flux rows.
// Shared memory is double buffered: one __syncthreads per chunk.
#pragma once
#include "flux_math.cuh"
#include "kernels_aux.cuh"

namespace gk {

constexpr int FM_THREADS = 128;
constexpr int FM_NV = 7;  // reconstructed variables

template <int D, int TC>
struct FluxSmem {
  // pitch of one chunk-local face index in doubles: 32 pencils (+ padding for D = 0, where
  // phase B walks c fastest: TC*pitch' = 16 mod ... see DESIGN.md 5.1)
  static constexpr int P = D == 0 ? 32 + 16 / TC : 32;
  double q[2][FM_NV][2][TC][P];  // [buffer][variable][0 = L state, 1 = R state][face][pencil]
  double fl[2][TC][32];          // flattening coefficient of cell c (chunk-local), per pencil
  double fl0[32];                // ... of the prologue cell f0-1
};

// ---- the carried reconstruction state of one variable on one pencil ---------------------
template <int RECON>
struct March {
  double qa, qb;  // q_c, q_{c+1}
  double s0;      // PPM: limited slope dm_c;  minmod: q_c - q_{c-1}
  double il;      // PPM: interface value at c - 1/2
  double qpp;     // q^+ of the previous cell, not yet stored
  // q0..q3 = cells c-2, c-1, c, c+1 where c is the first cell to be processed
  __device__ __forceinline__ void init(double q0, double q1, double q2, double q3) {
    if (RECON == 0) {
      s0 = q2 - q1;
      il = 0.0;
    } else {
      const double dmA = ppm_slope(q0, q1, q2);
      s0 = ppm_slope(q1, q2, q3);
      il = ppm_iface(q1, q2, dmA, s0);
    }
    qa = q2; qb = q3; qpp = 0.0;
  }
  // process cell c given qn = q_{c+2} and the flattening coefficient f of cell c
  __device__ __forceinline__ void step(double qn, double f, double& qm, double& qp) {
    if (RECON == 0) {
      const double d = qb - qa;
      const double s = minmod(s0, d);
      qm = qa - 0.5 * s;
      qp = qa + 0.5 * s;
      s0 = d;
    } else {
      const double dmn = ppm_slope(qa, qb, qn);
      const double ir = ppm_iface(qa, qb, s0, dmn);
      qm = il; qp = ir;
      if (RECON == 2) {
        if (f != 0.0) {  // G8(c); f = 0 leaves the values untouched exactly
          qp = f * qa + (1.0 - f) * qp;
          qm = f * qa + (1.0 - f) * qm;
        }
      }
      // G8(d)
      if ((qp - qa) * (qa - qm) <= 0.0) {
        qp = qa; qm = qa;
      } else {
        const double Dq = qp - qm;
        const double m = qa - 0.5 * (qp + qm);
        const double D26 = Dq * Dq * (1.0 / 6.0);
        if (Dq * m > D26) qm = 3.0 * qa - 2.0 * qp;
        else if (-D26 > Dq * m) qp = 3.0 * qa - 2.0 * qm;
      }
      s0 = dmn; il = ir;
    }
    qa = qb; qb = qn;
  }
};

// flattening coefficient marcher (G8c): f_c from p_{c-2..c+2} and v^D_{c-1}, v^D_{c+1}
struct FlatMarch {
  double pm2, pm1, p0, pp1, vm1, v0;
  // p[0..3] = p_{c-2..c+1}, v[0..1] = v_{c-1}, v_c for the first cell c
  __device__ __forceinline__ void init(double a, double b, double c, double d, double va,
                                       double vb) {
    pm2 = a; pm1 = b; p0 = c; pp1 = d; vm1 = va; v0 = vb;
  }
  // pn = p_{c+2}, vn = v_{c+1}
  __device__ __forceinline__ double step(double pn, double vn) {
    const double f = ppm_flatten(pm2, pm1, pp1, pn, vm1, vn);
    pm2 = pm1; pm1 = p0; p0 = pp1; pp1 = pn;
    vm1 = v0; v0 = vn;
    return f;
  }
};

__device__ __forceinline__ int fm_var_field(int D, int slot) {
  // slots 0..4 = rho, v^x, v^y, v^z, p; 5, 6 = B^{(D+1)%3}, B^{(D+2)%3} at cell centres
  return slot < 5 ? F_P + slot : F_BC + (D + 1 + (slot - 5)) % 3;
}

// index of cell 0 of pencil r along D (r = flattened transverse index incl. the apron).
// apron != 0: only the two apron columns t0 = -1 and t0 = n_t0 (t0 = y for D = x, else x) at
// every t1 in [-1, n_t1] -- the pencils k_flux_tma (flux_tma.cuh) leaves out.
template <int D>
__device__ __forceinline__ long long fm_pencil_base(const Geom& g, int r, int apron) {
  if (apron) {
    const int t1 = (r >> 1) - 1;
    if (D == 0) return g.at(0, (r & 1) ? g.ny : -1, t1);
    const int i = (r & 1) ? g.nx : -1;
    return D == 1 ? g.at(i, 0, t1) : g.at(i, t1, 0);
  }
  if (D == 0) {
    const int na = g.ny + 2;
    return g.at(0, r % na - 1, r / na - 1);
  } else if (D == 1) {
    const int na = g.nx + 2;
    return g.at(r % na - 1, 0, r / na - 1);
  } else {
    const int na = g.nx + 2;
    return g.at(r % na - 1, r / na - 1, 0);
  }
}

__host__ __device__ inline int fm_npencils(const Geom& g, int D, int apron) {
  if (apron) return 2 * ((D == 2 ? g.ny : g.nz) + 2);
  return D == 0 ? (g.ny + 2) * (g.nz + 2)
                : (D == 1 ? (g.nx + 2) * (g.nz + 2) : (g.nx + 2) * (g.ny + 2));
}

// RECON: 0 minmod, 1 PPM without flattening, 2 PPM with flattening.
// grid: x = pencil groups, y = segments of `seglen` faces (seglen a multiple of TC).
template <int D, int RECON, int TC>
__global__ void __launch_bounds__(FM_THREADS, 4)
k_flux_march(double* __restrict__ base, Geom g, Eos E, int seglen, int apron) {
  using Smem = FluxSmem<D, TC>;
  extern __shared__ __align__(16) unsigned char fm_smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(fm_smem_raw);
  constexpr int P = Smem::P;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nD = g.n(D);
  const long long sd = D == 0 ? 1 : (D == 1 ? g.sy : g.sz);
  const int npen = fm_npencils(g, D, apron);
  const int f0 = blockIdx.y * seglen;
  const int f1 = min(f0 + seglen, nD + 1);
  const int cmax = nD + G - 1;  // last valid cell index along D

  // ---- phase-A identity: lane = pencil
  const int rA = min((int)blockIdx.x * 32 + lane, npen - 1);
  const long long baseA = fm_pencil_base<D>(g, rA, apron);
  const int s0 = 2 * warp, nslot = warp == 3 ? 1 : 2;
  const double* qsrc[2];
  qsrc[0] = fld(base, g, fm_var_field(D, s0)) + baseA;
  qsrc[1] = fld(base, g, fm_var_field(D, s0 + (nslot > 1 ? 1 : 0))) + baseA;
  const double* psrc = fld(base, g, F_P + 4) + baseA;
  const double* vsrc = fld(base, g, F_P + 1 + D) + baseA;

  March<RECON> mv[2];
  FlatMarch fmch;
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
  if (RECON == 2) __syncthreads();
#pragma unroll
  for (int s = 0; s < 2; s++) {
    if (s < nslot) {
      double qm, qp;
      mv[s].step(qsrc[s][min(f0 + 1, cmax) * sd], RECON == 2 ? sm.fl0[lane] : 0.0, qm, qp);
      mv[s].qpp = qp;
    }
  }

  // ---- phase-B identity: one thread per face of the chunk, lanes along x
  constexpr int NIT = TC * 32 / FM_THREADS;
  static_assert(TC * 32 % FM_THREADS == 0, "TC must be a multiple of 4");
  long long baseB[NIT];
  bool okB[NIT];
  int clB[NIT], plB[NIT];
#pragma unroll
  for (int it = 0; it < NIT; it++) {
    if (D == 0) { clB[it] = tid % TC; plB[it] = tid / TC + it * (FM_THREADS / TC); }
    else { plB[it] = lane; clB[it] = warp + 4 * it; }
    const int r = (int)blockIdx.x * 32 + plB[it];
    okB[it] = r < npen;
    baseB[it] = fm_pencil_base<D>(g, min(r, npen - 1), apron);
  }
  const int fid = D == 0 ? F_FX : (D == 1 ? F_FY : F_FZ);

  int buf = 0;
  for (int F = f0; F < f1; F += TC, buf ^= 1) {
    // ================= phase A: cells F .. F+TC-1 =================
    double qn[2][TC];
#pragma unroll
    for (int s = 0; s < 2; s++) {
      if (s < nslot) {
        if (D == 0) {
          // consecutive x: 16-byte vector loads (F + 2 + X0 is even)
#pragma unroll
          for (int cl = 0; cl < TC; cl += 2) {
            const int c2 = min(F + cl + 2, cmax & ~1);  // even: stays 16-byte aligned, in-row
            const double2 v = *reinterpret_cast<const double2*>(qsrc[s] + c2);
            qn[s][cl] = v.x; qn[s][cl + 1] = v.y;
          }
        } else {
#pragma unroll
          for (int cl = 0; cl < TC; cl++) qn[s][cl] = qsrc[s][min(F + cl + 2, cmax) * sd];
        }
      }
    }
#pragma unroll
    for (int s = 0; s < 2; s++) {
      if (s < nslot) {
#pragma unroll
        for (int cl = 0; cl < TC; cl++) {
          double qm, qp;
          mv[s].step(qn[s][cl], RECON == 2 ? sm.fl[buf][cl][lane] : 0.0, qm, qp);
          sm.q[buf][s0 + s][0][cl][lane] = mv[s].qpp;  // left state of face F+cl
          sm.q[buf][s0 + s][1][cl][lane] = qm;         // right state of face F+cl
          mv[s].qpp = qp;
        }
      }
    }
    if (RECON == 2 && warp == 3 && F + TC < f1) {
#pragma unroll
      for (int cl = 0; cl < TC; cl++) {
        const int cc = F + TC + cl;
        sm.fl[buf ^ 1][cl][lane] =
            fmch.step(psrc[min(cc + 2, cmax) * sd], vsrc[min(cc + 1, cmax) * sd]);
      }
    }
    __syncthreads();
    // ================= phase B: faces F .. F+TC-1 =================
#pragma unroll
    for (int it = 0; it < NIT; it++) {
      const int cl = clB[it], pl = plB[it];
      const int f = F + cl;
      if (f < f1 && okB[it]) {
        const long long c = baseB[it] + f * sd;
        const Met M = face_metric(base, g, c, sd);
        const double det = det_gamma(M);
        const double isg = rsqrt(det);
        const double sgf = det * isg;
        const double gdd = inv_gamma_dd<D>(M, isg * isg);
        const double Bn = fld(base, g, F_BF + D)[c] * isg;  // G6
        double qL[FM_NV], qR[FM_NV];
#pragma unroll
        for (int v = 0; v < FM_NV; v++) {
          qL[v] = sm.q[buf][v][0][cl][pl];
          qR[v] = sm.q[buf][v][1][cl][pl];
        }
        double UL[7], GL[7], UR[7], GR[7], lmL, lpL, lmR, lpR;
        side_rows<D>(qL[0], qL[1], qL[2], qL[3], qL[4], D == 0 ? Bn : (D == 1 ? qL[6] : qL[5]),
                     D == 1 ? Bn : (D == 2 ? qL[6] : qL[5]),
                     D == 2 ? Bn : (D == 0 ? qL[6] : qL[5]), M, gdd, E, UL, GL, lmL, lpL);
        side_rows<D>(qR[0], qR[1], qR[2], qR[3], qR[4], D == 0 ? Bn : (D == 1 ? qR[6] : qR[5]),
                     D == 1 ? Bn : (D == 2 ? qR[6] : qR[5]),
                     D == 2 ? Bn : (D == 0 ? qR[6] : qR[5]), M, gdd, E, UR, GR, lmR, lpR);
        double out[7];
        hll_rows(UL, GL, lmL, lpL, UR, GR, lmR, lpR, sgf, E.riemann, out);
#pragma unroll
        for (int r = 0; r < 7; r++) fld(base, g, fid + r)[c] = out[r];
      }
    }
    // no barrier here: the next phase A writes the other buffer
  }
}

}  // namespace gk

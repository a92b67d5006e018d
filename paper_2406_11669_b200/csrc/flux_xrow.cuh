// flux_xrow.cuh -- A3 + A4 along x with the lanes of a warp ALONG x.
//
// x is the contiguous axis: a kernel that marches along x (flux_tma.cuh, D = 0) can only
// touch 32 bytes of a row at a time, which HBM serves badly (ncu capture r1g: the prefetched
// cells arrive late, DRAM reads 1.45x the algorithmic bytes).  Here a warp owns 32 consecutive
// cells c0 .. c0+31 of one row (j, k); lane = cell.  Every load and store is a contiguous
// 256-byte row segment.  The reconstruction recurrences run across lanes: the limited slope,
// the interface value and the parabola of a cell are computed once, by the cell's lane, and
// handed to the neighbour with warp shuffles (R5/G8: slope of c+1 from the lane above,
// interface c-1/2 and q^+_{c-1} from the lane below).  The lane of cell c then solves the
// Riemann problem of face c-1/2.  The 3 lowest and 2 highest lanes have incomplete stencils:
// a warp yields 27 faces; consecutive warps overlap by 5 cells.  No shared memory, no block
// barrier, nothing carried from one row segment to the next.
#pragma once
#include "flux_tma.cuh"

namespace gk {

constexpr int FX_THREADS = 128;
constexpr int FX_VALID = 27;  // faces per warp: lanes 3 .. 29
#ifndef FX_MINB
#define FX_MINB 4
#endif

__device__ __forceinline__ double fx_up(double v, int d) {
  return __shfl_up_sync(0xffffffffu, v, d);
}
__device__ __forceinline__ double fx_dn(double v, int d) {
  return __shfl_down_sync(0xffffffffu, v, d);
}

// q^-_c (right state of face c-1/2) and q^+_c of the lane's cell; qm1, qp1 = neighbours
template <int RECON>
__device__ __forceinline__ void fx_recon(double q, double qm1, double qp1, double f, bool anyf,
                                         double& qm, double& qp) {
  const double dl = q - qm1, dr = qp1 - q;
  if (RECON == 0) {  // G7
    const double m = fabs(dl) < fabs(dr) ? dl : dr;
    const double s = dl * dr > 0.0 ? m : 0.0;
    qm = fma(-0.5, s, q);
    qp = fma(0.5, s, q);
  } else {  // G8(a)-(d), same arithmetic as FtMarch::step
    const double dm = ft_slope(dl, dr);
    const double dmp = fx_dn(dm, 1);                             // slope of cell c+1
    const double ir = 0.5 * (q + qp1) - (dmp - dm) * (1.0 / 6.0);  // interface c + 1/2
    const double il = fx_up(ir, 1);                              // interface c - 1/2
    qm = il; qp = ir;
    if (RECON == 2 && anyf) {
      const double qpf = f * q + (1.0 - f) * qp;
      const double qmf = f * q + (1.0 - f) * qm;
      qp = f != 0.0 ? qpf : qp;
      qm = f != 0.0 ? qmf : qm;
    }
    const double a = qp - q, b = q - qm;
    const double aa = fabs(a), ab = fabs(b);
    const bool flat = ft_opposite(a, b);
    const bool fixm = ab > 2.0 * aa;
    const bool fixp = aa > 2.0 * ab;
    const double qm2 = fma(-2.0, a, q);
    const double qp2 = fma(2.0, b, q);
    qm = ft_sel(flat, q, ft_sel(fixm, qm2, qm));
    qp = ft_sel(flat, q, ft_sel(fixp, qp2, qp));
  }
}

// grid: one warp per (pencil, segment) item: item = pencil * nsd + seg.  With (t0, t1) the
// transverse axes -- (y, z) for D = x, (x, z) for D = y, (x, y) for D = z -- and `ap` the
// transverse apron (1 for flux-CT, R10; 3 for the upwind CT, G27):
//   mode 0: every pencil t0 in [-ap, n_t0 + ap), t1 in [-ap, n_t1 + ap).  The x fluxes; for
//           D = y, z the lanes then run along y or z with a stride (uncoalesced: small
//           blocks and option combinations only).
//   mode 1: only the 2 ap apron columns t0 < 0 and t0 >= n_t0 that the 32-wide groups of
//           k_flux_tma leave out.
// UCT (compile time, as in k_flux_tma): also store the upwind-CT face rows of F_W.
template <int D, int RECON, bool UCT>
__global__ void __launch_bounds__(FX_THREADS, FX_MINB)
k_flux_xrow(double* __restrict__ base, Geom g, Eos E, int nsd, long long nitems, int ap,
            int mode) {
  const int lane = threadIdx.x & 31;
  const long long nwarp = (long long)gridDim.x * (FX_THREADS / 32);
  const int nD = g.n(D);
  const int nt0 = D == 0 ? g.ny : g.nx;
  const int w0 = mode ? 2 * ap : nt0 + 2 * ap;
  const int sd = D == 0 ? 1 : (D == 1 ? (int)g.sy : (int)g.sz);
  // grid-stride loop over the items (the launch gives every warp one item)
  for (long long item = (long long)blockIdx.x * (FX_THREADS / 32) + (threadIdx.x >> 5);
       item < nitems; item += nwarp) {
  const int seg = (int)(item % nsd);
  const int row = (int)(item / nsd);
  const int c = seg * FX_VALID - 3 + lane;  // this lane's cell along D; its face is c - 1/2
  const int cc = min(c, nD + G - 1);        // lanes past the last ghost cell reuse it
  const int q0 = row % w0, t1 = row / w0 - ap;
  const int t0 = mode ? (q0 < ap ? q0 - ap : nt0 + q0 - ap) : q0 - ap;
  const int idx = (int)(D == 0 ? g.at(cc, t0, t1) : (D == 1 ? g.at(t0, cc, t1) : g.at(t0, t1, cc)));

  // ---- cell data of the lane: rho, v^x, v^y, v^z, p, B^y, B^z
  double q[FM_NV];
#pragma unroll
  for (int v = 0; v < FM_NV; v++) q[v] = fld(base, g, fm_var_field(D, v))[idx];
  const double bfx = fld(base, g, F_BF + D)[idx];
  // ---- face metric (R4): 4-point Lagrange along D.  Lanes 0-2 have no face to solve: their
  // stencil base is moved to cell -1 so that it stays inside the padded array.
  const int idxm = idx + (max(cc, -1) - cc) * sd;
  Met M;
  {
    double mq[FT_NMET];
#pragma unroll
    for (int v = 0; v < FT_NMET; v++) {
      const double* m = fld(base, g, F_MET + v) + idxm;
      mq[v] = (-m[-2 * sd] + 9.0 * m[-sd] + 9.0 * m[0] - m[sd]) * 0.0625;
    }
    M.a = mq[0]; M.bx = mq[1]; M.by = mq[2]; M.bz = mq[3];
    M.gxx = mq[4]; M.gxy = mq[5]; M.gxz = mq[6]; M.gyy = mq[7]; M.gyz = mq[8]; M.gzz = mq[9];
  }
  // ---- neighbours across lanes
  double qm1[FM_NV], qp1[FM_NV];
#pragma unroll
  for (int v = 0; v < FM_NV; v++) { qm1[v] = fx_up(q[v], 1); qp1[v] = fx_dn(q[v], 1); }
  // G8(c): flattening coefficient of the lane's cell from p_{c-2..c+2}, v^D_{c-1}, v^D_{c+1}
  double f = 0.0;
  bool anyf = false;
  if (RECON == 2) {
    const double pm2 = fx_up(q[4], 2), pp2 = fx_dn(q[4], 2);
    const double dp1 = qp1[4] - qm1[4];
    const double dp2 = pp2 - pm2;
    const bool on = fabs(dp1) > 0.33 * ft_min(qp1[4], qm1[4]) && qm1[1 + D] > qp1[1 + D];
    const bool z = dp2 == 0.0;
    const double r = ft_rcp(z ? 1.0 : dp2);
    double ff = 10.0 * fma(dp1, r, -0.75);
    ff = ft_min(1.0, ft_max(0.0, ff));
    ff = z ? 1.0 : ff;
    f = on ? ff : 0.0;
    anyf = __any_sync(0xffffffffu, f != 0.0);
  }
  double qL[FM_NV], qR[FM_NV];
#pragma unroll
  for (int v = 0; v < FM_NV; v++) {
    double qm, qp;
    fx_recon<RECON>(q[v], qm1[v], qp1[v], f, anyf, qm, qp);
    qL[v] = fx_up(qp, 1);  // q^+ of cell c-1
    qR[v] = qm;
  }
  // ---- Riemann problem of face c - 1/2 (R7)
  const double det = det_gamma(M);
  const double isg = ft_rsqrt(det);
  const double sgf = det * isg;
  const double gdd = inv_gamma_dd<D>(M, isg * isg);
  const double Bn = bfx * isg;  // G6
  double UL[7], GL[7], UR[7], GR[7], lmL, lpL, lmR, lpR, vtL[2], vtR[2], apm[2];
  // slots 5, 6 hold B^{(D+1)%3}, B^{(D+2)%3}
  ft_side<D>(qL[0], qL[1], qL[2], qL[3], qL[4], D == 0 ? Bn : (D == 1 ? qL[6] : qL[5]),
             D == 1 ? Bn : (D == 2 ? qL[6] : qL[5]), D == 2 ? Bn : (D == 0 ? qL[6] : qL[5]), M,
             gdd, E, UL, GL, lmL, lpL, UCT ? vtL : nullptr);
  ft_side<D>(qR[0], qR[1], qR[2], qR[3], qR[4], D == 0 ? Bn : (D == 1 ? qR[6] : qR[5]),
             D == 1 ? Bn : (D == 2 ? qR[6] : qR[5]), D == 2 ? Bn : (D == 0 ? qR[6] : qR[5]), M,
             gdd, E, UR, GR, lmR, lpR, UCT ? vtR : nullptr);
  double out[7];
  ft_hll(UL, GL, lmL, lpL, UR, GR, lmR, lpR, sgf, E.riemann, out, UCT ? apm : nullptr);
  if (lane >= 3 && lane < 3 + FX_VALID && c <= nD) {
    double* o = fld(base, g, D == 0 ? F_FX : (D == 1 ? F_FY : F_FZ)) + idx;
    const size_t NPA = (size_t)g.NPA;
#pragma unroll
    for (int r = 0; r < 7; r++) o[r * NPA] = out[r];
    if (UCT) ft_store_uct(fld(base, g, F_W + 4 * D) + idx, NPA, apm, vtL, vtR);
  }
  }  // items
}

}  // namespace gk

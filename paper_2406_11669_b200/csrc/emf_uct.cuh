// emf_uct.cuh -- row F1: the electric field on the edges by the upwind constrained transport
// (eqs 33-35; readings G26-G28 of DESIGN.md) and the update of A_i.
#pragma once
#include "flux_xrow.cuh"
#include "kernels_flux.cuh"

namespace gk {

// ---------------------------------------------------------- upwind constrained transport
// Row F1, eqs (33)-(35), readings G26-G28 of DESIGN.md.  One bracket of
// eq. (35): the quantities on the b-faces -- vbar^a (eq. 33, stored by the b-direction flux
// kernel in F_W) and the staggered B~^b -- reconstructed along a to the edge (PPM of G8, no
// flattening: L from the lower, R from the upper side), combined with the larger a_+, a_- of
// the two a-faces that share the edge.  c = index of the edge, sa / sb = strides of a and b.
// G8 without flattening on the 6 values s[0..5] around a position: L = q^+ of cell 2, R = q^- of
// cell 3; branch free, same arithmetic as FtMarch::step (flux_face.cuh).
// monotonised q^+ (UPPER = true) or q^- of a cell from its two interface values
template <bool UPPER>
__device__ __forceinline__ double uct_limit(double q, double qm, double qp) {
  const double a = qp - q, b = q - qm;
  const bool flat = ft_opposite(a, b);
  if (UPPER) {
    const bool fixp = fabs(a) > 2.0 * fabs(b);
    return ft_sel(flat, q, ft_sel(fixp, fma(2.0, b, q), qp));
  } else {
    const bool fixm = fabs(b) > 2.0 * fabs(a);
    return ft_sel(flat, q, ft_sel(fixm, fma(-2.0, a, q), qm));
  }
}
__device__ __forceinline__ void uct_recon6(const double s[6], double& L, double& R) {
  const double d0 = s[1] - s[0], d1 = s[2] - s[1], d2 = s[3] - s[2], d3 = s[4] - s[3],
               d4 = s[5] - s[4];
  const double m1 = ft_slope2(d0, d1), m2 = ft_slope2(d1, d2), m3 = ft_slope2(d2, d3),
               m4 = ft_slope2(d3, d4);
  const double i12 = ft_iface(s[1], s[2], m1, m2);
  const double i23 = ft_iface(s[2], s[3], m2, m3);
  const double i34 = ft_iface(s[3], s[4], m3, m4);
  L = uct_limit<true>(s[2], i12, i23);   // q^+ of the lower cell
  R = uct_limit<false>(s[3], i23, i34);  // q^- of the upper cell
}

__device__ __forceinline__ double uct_bracket(const double* __restrict__ base, const Geom& g,
                                              int a, int b, long long c, long long sa,
                                              long long sb) {
  const double* vb = fld(base, g, F_W + 4 * b + (a == (b + 1) % 3 ? 2 : 3));
  const double* Bb = fld(base, g, F_BF + b);
  double sv[6], sB[6];
#pragma unroll
  for (int m = 0; m < 6; m++) {
    sv[m] = vb[c + (m - 3) * sa];
    sB[m] = Bb[c + (m - 3) * sa];
  }
  double vL, vR, BL, BR;
  uct_recon6(sv, vL, vR);
  uct_recon6(sB, BL, BR);
  const double* Ap = fld(base, g, F_W + 4 * a);
  const double* Am = fld(base, g, F_W + 4 * a + 1);
  const double ap = ft_max(Ap[c], Ap[c - sb]);
  const double am = ft_max(Am[c], Am[c - sb]);
  const double cs = ap + am;
  const bool deg = cs < 1e-300;
  const double w = ft_rcp(deg ? 1.0 : cs);
  const double full = (ap * vL * BL + am * vR * BR - ap * am * (BR - BL)) * w;
  return deg ? 0.5 * (vL * BL + vR * BR) : full;
}

// One thread per edge: blockIdx.z = 3 k + comp; E_comp = -[a-bracket] + [b-bracket] with
// (a, b, comp) cyclic, then R11 d_t A_comp = -E_comp and the RK combination.
__global__ void __launch_bounds__(256)
k_emf_uct(double* __restrict__ base, Geom g, const DevState* __restrict__ st, RkStage rk,
          int gauge) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z / 3;
  const int comp = blockIdx.z % 3;
  if (i > g.nx || j > g.ny) return;
  if ((comp == 0 && i >= g.nx) || (comp == 1 && j >= g.ny) || (comp == 2 && k >= g.nz)) return;
  const long long c = g.at(i, j, k);
  const int a = (comp + 1) % 3, b = (comp + 2) % 3;
  const long long sa = g.stride(a), sb = g.stride(b);
  const double E = -uct_bracket(base, g, a, b, c, sa, sb) + uct_bracket(base, g, b, a, c, sb, sa);
  double rhs = -E;
  if (gauge) {  // eq. (31): - d_comp G_A
    const double* GA = fld(base, g, F_GV);
    rhs -= (GA[c + g.stride(comp)] - GA[c]) * g.idx[comp];
  }
  rk_apply(base, g, 5 + comp, c, rhs, st->dt, rk);
}

// ---- the same electric field, every face -> edge parabola built once --------------------
// k_emf_uct above rebuilds each parabola in both edges that use it (and each slope four
// times).  The passes below take one reconstruction axis A at a time and compute the two
// brackets of eq. (35) that reconstruct along A, for every edge index (i,j,k) in [0, n]:
//   br(A, A+1) -> -E_{A+2},   br(A, A+2) -> +E_{A+1}
// into three scratch fields (the flux-CT B rows F_FX+5, F_FY+5, F_FZ+5, unused with the upwind
// CT, hold E_x, E_y, E_z).  Pass order x, y, z; `wr` bit 0 / bit 1 = the first / second
// bracket writes (first contribution) instead of adding; the last one goes into R11 + RK.
__device__ __forceinline__ double* uct_escratch(double* base, const Geom& g, int comp) {
  return fld(base, g, comp == 0 ? F_FX + 5 : (comp == 1 ? F_FY + 5 : F_FZ + 5));
}
__device__ __forceinline__ double uct_combine(double ap, double am, double vL, double vR,
                                              double BL, double BR) {
  const double cs = ap + am;
  const bool deg = cs < 1e-300;
  const double w = ft_rcp(deg ? 1.0 : cs);
  const double full = (ap * vL * BL + am * vR * BR - ap * am * (BR - BL)) * w;
  return deg ? 0.5 * (vL * BL + vR * BR) : full;
}
__device__ __forceinline__ int uct_vbar_field(int a, int b) {  // vbar^a on the b-faces
  return F_W + 4 * b + (a == (b + 1) % 3 ? 2 : 3);
}

// A = 1, 2: lanes along x, one thread per (i, t) column and bracket (blockIdx.y = 2 t + w:
// w = 0 the bracket br(A, A+1) -> -E_{A+2}, w = 1 br(A, A+2) -> +E_{A+1}) marching along A with
// the PPM state of its two quantities carried in registers (FtMarch, as in the flux kernels).
// `wr` bit w: this bracket is the first contribution (write), else add; `fin` bit w: it is the
// last one -- the component goes straight into R11 + the RK combination.
#ifndef UM_MINB
#define UM_MINB 6
#endif
#ifndef UM_CHUNK
#define UM_CHUNK 2
#endif
template <int A>
__global__ void __launch_bounds__(128, UM_MINB)
k_uct_march(double* __restrict__ base, Geom g, int seglen, int wr, int fin,
            const DevState* __restrict__ st, RkStage rk, int gauge) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int t = blockIdx.y >> 1;
  const int w = blockIdx.y & 1;
  if (i > g.nx) return;
  const int nA = g.n(A);
  const int m0 = (int)blockIdx.z * seglen, m1 = min(m0 + seglen, nA + 1);
  const int b = (A + 1 + w) % 3;     // the faces whose quantities are reconstructed along A
  const int comp = (A + 2 - w) % 3;  // the edge component this bracket belongs to
  const double sign = w ? 1.0 : -1.0;
  const long long sA = g.stride(A), sb = g.stride(b);
  const long long c0 = A == 1 ? g.at(i, 0, t) : g.at(i, t, 0);  // position 0 along A
  const double* q[2] = {fld(base, g, uct_vbar_field(A, b)) + c0, fld(base, g, F_BF + b) + c0};
  const double* Ap = fld(base, g, F_W + 4 * A) + c0;
  const double* Am = fld(base, g, F_W + 4 * A + 1) + c0;
  double* Ec = uct_escratch(base, g, comp) + c0;
  // does the component exist at this (i, t)?  E_x needs i < nx; otherwise the index along the
  // component's own axis, which is t's axis here (comp != A)
  const bool ok = comp == 0 ? i < g.nx : t < g.n(comp);
  const bool first = (wr >> w) & 1, last = (fin >> w) & 1;
  const double h = st->dt;
  const double* GA = fld(base, g, F_GV) + c0;
  const long long sc = g.stride(comp);
  FtMarch<1> mv[2];
#pragma unroll
  for (int v = 0; v < 2; v++) {
    mv[v].init(q[v][(m0 - 3) * sA], q[v][(m0 - 2) * sA], q[v][(m0 - 1) * sA], q[v][m0 * sA]);
    double qm, qp;
    mv[v].step(q[v][(m0 + 1) * sA], 0.0, false, qm, qp);  // position m0 - 1
    mv[v].qpp = qp;
  }
  // The march is serial along A, so its loads are what can overlap: the inputs of a chunk of
  // UM_CHUNK steps (2 reconstructed values, 4 a+- values and the pending first bracket each) are
  // all requested before the first of them is used.
  const int need_e = !first;
  for (int mb = m0; mb < m1; mb += UM_CHUNK) {
    double cq[UM_CHUNK][2], ca[UM_CHUNK][4], ce[UM_CHUNK];
#pragma unroll
    for (int u = 0; u < UM_CHUNK; u++) {
      const long long c = (long long)min(mb + u, m1 - 1) * sA;  // the tail repeats its last step
      cq[u][0] = q[0][c + 2 * sA]; cq[u][1] = q[1][c + 2 * sA];
      ca[u][0] = Ap[c]; ca[u][1] = Ap[c - sb]; ca[u][2] = Am[c]; ca[u][3] = Am[c - sb];
      ce[u] = need_e ? Ec[c] : 0.0;
    }
#pragma unroll
    for (int u = 0; u < UM_CHUNK; u++) {
      const int m = mb + u;
      if (m >= m1) break;
      const double ap = ft_max(ca[u][0], ca[u][1]), am = ft_max(ca[u][2], ca[u][3]);
      double L[2], R[2];
      {
        double qm, qp;
        mv[0].step(cq[u][0], 0.0, false, qm, qp);
        L[0] = mv[0].qpp; R[0] = qm; mv[0].qpp = qp;  // q^+ of position m-1, q^- of position m
        mv[1].step(cq[u][1], 0.0, false, qm, qp);
        L[1] = mv[1].qpp; R[1] = qm; mv[1].qpp = qp;
      }
      const long long c = m * sA;
      const double br = sign * uct_combine(ap, am, L[0], R[0], L[1], R[1]);
      const double e = first ? br : ce[u] + br;
      if (last) {
        if (ok) {
          double rhs = -e;
          if (gauge) rhs -= (GA[c + sc] - GA[c]) * g.idx[comp];
          rk_apply(base, g, 5 + comp, c0 + c, rhs, h, rk);
        }
      } else {
        Ec[c] = e;
      }
    }
  }
}

// A = 0: lanes along x, the recurrences across lanes by shuffles (fx_recon, as k_flux_xrow):
// one warp per 27 edge positions of a row (j, k) in [0, ny] x [0, nz].
__global__ void __launch_bounds__(128)
k_uct_xrow(double* __restrict__ base, Geom g, int nsd, long long nitems, int wr) {
  const int lane = threadIdx.x & 31;
  const long long item = (long long)blockIdx.x * 4 + (threadIdx.x >> 5);
  if (item >= nitems) return;  // warp uniform
  const int seg = (int)(item % nsd);
  const int row = (int)(item / nsd);
  const int j = row % (g.ny + 1), k = row / (g.ny + 1);
  const int p = seg * FX_VALID - 3 + lane;
  const long long c = g.at(min(p, g.nx + G - 1), j, k);
  constexpr int b1 = 1, b2 = 2;
  const double qv[4] = {fld(base, g, uct_vbar_field(0, b1))[c], fld(base, g, F_BF + b1)[c],
                        fld(base, g, uct_vbar_field(0, b2))[c], fld(base, g, F_BF + b2)[c]};
  double L[4], R[4];
#pragma unroll
  for (int v = 0; v < 4; v++) {
    double qm, qp;
    fx_recon<1>(qv[v], fx_up(qv[v], 1), fx_dn(qv[v], 1), 0.0, false, qm, qp);
    L[v] = fx_up(qp, 1);
    R[v] = qm;
  }
  if (lane >= 3 && lane < 3 + FX_VALID && p <= g.nx) {
    const double* Ap = fld(base, g, F_W + 0);
    const double* Am = fld(base, g, F_W + 1);
    const long long s1 = g.sy, s2 = g.sz;
    const double br1 = uct_combine(ft_max(Ap[c], Ap[c - s1]), ft_max(Am[c], Am[c - s1]), L[0],
                                   R[0], L[1], R[1]);
    const double br2 = uct_combine(ft_max(Ap[c], Ap[c - s2]), ft_max(Am[c], Am[c - s2]), L[2],
                                   R[2], L[3], R[3]);
    double* E1 = uct_escratch(base, g, 2);
    double* E2 = uct_escratch(base, g, 1);
    E1[c] = (wr & 1) ? -br1 : E1[c] - br1;
    E2[c] = (wr & 2) ? br2 : E2[c] + br2;
  }
}

// ------------------------------------------------------------ generalised Lorenz gauge
// Row F3; readings G29-G32 of DESIGN.md.  One thread per vertex
// (i-1/2, j-1/2, k-1/2), i in [-1, nx+1] etc.: the metric as the mean of the 8 cells around the
// vertex (G29), A_j as the mean of the two edges of its own axis ending there (G30), then
//   G_A = alpha Psi/sqrt(gamma) - beta^j A_j                    (eq. 31)
//   F_Psi^d = alpha sqrt(gamma) gamma^{dl} A_l - beta^d Psi     (eq. 32)
// stored with alpha in the five vertex fields F_GV for k_update / k_emf_uct.
__global__ void __launch_bounds__(128)
k_gauge_vertex(double* __restrict__ base, Geom g) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x - 1;
  const int j = blockIdx.y * blockDim.y + threadIdx.y - 1;
  const int k = blockIdx.z - 1;
  if (i > g.nx + 1 || j > g.ny + 1) return;
  const long long c = g.at(i, j, k);
  const long long sy = g.sy, sz = g.sz;
  double m[10];
#pragma unroll
  for (int f = 0; f < 10; f++) {
    const double* q = fld(base, g, F_MET + f) + c;
    double acc = 0.0;
#pragma unroll
    for (int b = 0; b < 8; b++) acc += q[-(b & 1) - ((b >> 1) & 1) * sy - ((b >> 2) & 1) * sz];
    m[f] = 0.125 * acc;
  }
  Met M;
  M.a = m[0]; M.bx = m[1]; M.by = m[2]; M.bz = m[3];
  M.gxx = m[4]; M.gxy = m[5]; M.gxz = m[6]; M.gyy = m[7]; M.gyz = m[8]; M.gzz = m[9];
  const double det = det_gamma(M);
  const double sg = sqrt(det);
  const Sym3 gu = inv_gamma(M, 1.0 / det);
  const double* Ax = fld(base, g, F_Y + 5);
  const double* Ay = fld(base, g, F_Y + 6);
  const double* Az = fld(base, g, F_Y + 7);
  const double ax = 0.5 * (Ax[c - 1] + Ax[c]);
  const double ay = 0.5 * (Ay[c - sy] + Ay[c]);
  const double az = 0.5 * (Az[c - sz] + Az[c]);
  const double psi = fld(base, g, F_Y + 8)[c];
  fld(base, g, F_GV + 0)[c] = M.a * psi / sg - (M.bx * ax + M.by * ay + M.bz * az);
  const double asg = M.a * sg;
  fld(base, g, F_GV + 1)[c] = asg * (gu.xx * ax + gu.xy * ay + gu.xz * az) - M.bx * psi;
  fld(base, g, F_GV + 2)[c] = asg * (gu.xy * ax + gu.yy * ay + gu.yz * az) - M.by * psi;
  fld(base, g, F_GV + 3)[c] = asg * (gu.xz * ax + gu.yz * ay + gu.zz * az) - M.bz * psi;
  fld(base, g, F_GV + 4)[c] = M.a;
}

}  // namespace gk

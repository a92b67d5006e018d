// emf_uct.cuh -- row F1: the electric field on the edges by the upwind constrained transport
// (eqs 33-35; readings G26-G28 of DESIGN.md) and the update of A_i.
#pragma once
#include "flux_tma.cuh"
#include "kernels_flux.cuh"

namespace gk {

// ---------------------------------------------------------- upwind constrained transport
// Row F1, eqs (33)-(35), readings G26-G28 of DESIGN.md.  One bracket of
// eq. (35): the quantities on the b-faces -- vbar^a (eq. 33, stored by the b-direction flux
// kernel in F_W) and the staggered B~^b -- reconstructed along a to the edge (PPM of G8, no
// flattening: L from the lower, R from the upper side), combined with the larger a_+, a_- of
// the two a-faces that share the edge.  c = index of the edge, sa / sb = strides of a and b.
// G8 without flattening on the 6 values s[0..5] around a position: L = q^+ of cell 2, R = q^- of
// cell 3; branch free, same arithmetic as FtMarch::step.
__device__ __forceinline__ void uct_limit(double q, double& qm, double& qp) {
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
__device__ __forceinline__ void uct_recon6(const double s[6], double& L, double& R) {
  const double d0 = s[1] - s[0], d1 = s[2] - s[1], d2 = s[3] - s[2], d3 = s[4] - s[3],
               d4 = s[5] - s[4];
  const double m1 = ft_slope(d0, d1), m2 = ft_slope(d1, d2), m3 = ft_slope(d2, d3),
               m4 = ft_slope(d3, d4);
  const double i12 = 0.5 * (s[1] + s[2]) - (m2 - m1) * (1.0 / 6.0);
  const double i23 = 0.5 * (s[2] + s[3]) - (m3 - m2) * (1.0 / 6.0);
  const double i34 = 0.5 * (s[3] + s[4]) - (m4 - m3) * (1.0 / 6.0);
  double qm = i12, qp = i23;
  uct_limit(s[2], qm, qp);
  L = qp;
  qm = i23; qp = i34;
  uct_limit(s[3], qm, qp);
  R = qm;
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
k_emf_uct(double* __restrict__ base, Geom g, const DevState* __restrict__ st, RkStage rk) {
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
  rk_apply(base, g, 5 + comp, c, -E, st->dt, rk);
}

}  // namespace gk

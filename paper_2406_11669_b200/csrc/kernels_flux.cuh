// kernels_flux.cuh -- divergence + flux-CT + RK update (A5, A6, A7; the sources of A5 are
// evaluated by k_src, kernels_aux.cuh).
#pragma once
#include "kernels_aux.cuh"

namespace gk {

// ------------------------------------------------------------------------------ update
// RK stage combination (R12 / G15).  mode: 0 first SSP stage (saves Y0), 1 later SSP stage
// y = a Y0 + b (y + dt k), 2 first RK4 stage, 3 middle RK4 stages y = Y0 + (c dt) k,
// 4 last RK4 stage y = Y0 + dt/6 (k1 + 2 k2 + 2 k3 + k4).
struct RkStage {
  int mode;
  double a, b, c;
};

__device__ __forceinline__ void rk_apply(double* __restrict__ base, const Geom& g, int r,
                                         long long c, double k, double h, const RkStage& s) {
  double* y = fld(base, g, F_Y + r) + c;
  double* y0 = fld(base, g, F_Y0 + r) + c;
  double* ks = fld(base, g, F_KS + r) + c;
  const double yc = *y;
  switch (s.mode) {
    case 0: *y0 = yc; *y = yc + h * k; break;
    case 1: *y = s.a * (*y0) + s.b * (yc + h * k); break;
    case 2: *y0 = yc; *ks = k; *y = yc + (0.5 * h) * k; break;
    case 3: *ks += 2.0 * k; *y = *y0 + (s.c * h) * k; break;
    default: *y = *y0 + (h / 6.0) * (*ks + k); break;
  }
}

// One thread per evolved value: blockIdx.z = 8 k + r, r = row of Y (0-4 hydro rows of cell
// (i,j,k); 5-7 the edges A_x, A_y, A_z attached to index (i,j,k) in the lower convention).
// Each thread streams at most 6 flux values, one source, Y and Y0 -- all accesses are
// coalesced along x, the row is uniform per block (no divergence) and the register need is
// small enough for full occupancy.  The sources alpha sqrt(gamma) S were stored by k_post
// (kernels_aux.cuh) when the primitives they depend on were recovered.
template <int NROWS, bool GAUGE>
__global__ void __launch_bounds__(256)
k_update(double* __restrict__ base, Geom g, const DevState* __restrict__ st, RkStage rk,
         double lorenz_xi) {
  constexpr int nrows = NROWS;
  constexpr bool gauge = GAUGE;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  // nrows = 8 (5 hydro rows + 3 edges), 5 when k_emf_uct updates the edges; in the Lorenz gauge
  // one more row, the last: Psi_mhd on the vertices
  const int k = blockIdx.z / nrows;
  const int r = blockIdx.z % nrows;
  if (i > g.nx || j > g.ny) return;
  const long long c = g.at(i, j, k);
  const double h = st->dt;
  const long long sy = g.sy, sz = g.sz;
  double rhs;
  if (gauge && r == nrows - 1) {
    // eq. (32): d_t Psi = -d_j F_Psi^j - xi alpha Psi at the vertex (G32), xi = lorenz_xi / dt
    const double* Fx = fld(base, g, F_GV + 1);
    const double* Fy = fld(base, g, F_GV + 2);
    const double* Fz = fld(base, g, F_GV + 3);
    double div = (Fx[c + 1] - Fx[c - 1]) * (0.5 * g.idx[0]);
    div += (Fy[c + sy] - Fy[c - sy]) * (0.5 * g.idx[1]);
    div += (Fz[c + sz] - Fz[c - sz]) * (0.5 * g.idx[2]);
    const double xi = h > 0.0 ? lorenz_xi / h : 0.0;
    rhs = -div - xi * fld(base, g, F_GV + 4)[c] * fld(base, g, F_Y + 8)[c];
    rk_apply(base, g, 8, c, rhs, h, rk);
    return;
  }
  const double* GA = fld(base, g, F_GV);  // eq. (31): d_t A_i = -E_i - d_i G_A (G31)
  if (r < 5) {
    if (i >= g.nx || j >= g.ny || k >= g.nz) return;
    // R8: L(U~) = -sum_d (F~_{i+1/2} - F~_{i-1/2})/dx_d + alpha sqrt(gamma) S, eq. (17)
    const double* Fx = fld(base, g, F_FX + r);
    const double* Fy = fld(base, g, F_FY + r);
    const double* Fz = fld(base, g, F_FZ + r);
    double div = (Fx[c + 1] - Fx[c]) * g.idx[0];
    div += (Fy[c + sy] - Fy[c]) * g.idx[1];
    div += (Fz[c + sz] - Fz[c]) * g.idx[2];
    const double src = r == 0 ? 0.0 : fld(base, g, F_SRC + r - 1)[c];  // S_D = 0
    rhs = -div + src;
  } else if (r == 5) {
    // R10 (flux-CT, G13/G14) and R11 (d_t A_i = -E_i).  Stored B rows:
    // FX+5 = F~x(B~y), FX+6 = F~x(B~z); FY+5 = F~y(B~z), FY+6 = F~y(B~x);
    // FZ+5 = F~z(B~x), FZ+6 = F~z(B~y).
    if (i >= g.nx) return;  // E_x at (i, j-1/2, k-1/2)
    const double* FyBz = fld(base, g, F_FY + 5);
    const double* FzBy = fld(base, g, F_FZ + 6);
    rhs = -0.25 * (-FyBz[c - sz] - FyBz[c] + FzBy[c - sy] + FzBy[c]);
    if (gauge) rhs -= (GA[c + 1] - GA[c]) * g.idx[0];
  } else if (r == 6) {
    if (j >= g.ny) return;  // E_y at (i-1/2, j, k-1/2)
    const double* FzBx = fld(base, g, F_FZ + 5);
    const double* FxBz = fld(base, g, F_FX + 6);
    rhs = -0.25 * (-FzBx[c - 1] - FzBx[c] + FxBz[c - sz] + FxBz[c]);
    if (gauge) rhs -= (GA[c + sy] - GA[c]) * g.idx[1];
  } else {
    if (k >= g.nz) return;  // E_z at (i-1/2, j-1/2, k)
    const double* FxBy = fld(base, g, F_FX + 5);
    const double* FyBx = fld(base, g, F_FY + 6);
    rhs = -0.25 * (-FxBy[c - sy] - FxBy[c] + FyBx[c - 1] + FyBx[c]);
    if (gauge) rhs -= (GA[c + sz] - GA[c]) * g.idx[2];
  }
  rk_apply(base, g, r, c, rhs, h, rk);
}

}  // namespace gk

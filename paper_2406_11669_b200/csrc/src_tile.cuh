// src_tile.cuh -- A5: alpha sqrt(gamma) S of eq. (19) (R9 / G11) with the x-y stencils of the
// metric derivatives served from a TMA-staged shared-memory tile.
//
// k_src (kernels_aux.cuh) issues 144 global loads per cell, 120 of them the 4th-order stencils
// of the 10 differentiated fields alpha, beta^i, gamma_ij in x, y and z, and spends a third of
// its instructions on their 64-bit addresses.  Here a block of 32 x 8 cells of one z-plane gets
// the (32+4) x (8+4) tile of all 10 fields with ONE cp.async.bulk.tensor (a 4-D box
// [field][1][12][36] of the workspace tensor map, 34.5 KB, completion on an mbarrier): the cell
// metric and the 80 x and y stencil values become shared-memory reads at immediate offsets.  The
// 40 z-stencil values, K_ij and the primitives stay plain loads, issued before the tile is
// waited for.  Same arithmetic, in the same order, as k_src (src_axis): the two are bit-identical.
#pragma once
#include "kernels_aux.cuh"
#include "tma.cuh"

namespace gk {

constexpr int ST_BX = 32, ST_BY = 8;
constexpr int ST_TX = ST_BX + 4, ST_TY = ST_BY + 4;   // tile extent incl. the 2-cell halo
constexpr int ST_NF = 10;                             // alpha, beta^i, gamma_ij

struct SrcTileSmem {
  alignas(128) double tile[ST_NF][ST_TY][ST_TX];
  alignas(8) unsigned long long bar;
};

__global__ void __launch_bounds__(ST_BX * ST_BY, 2)
k_src_tile(double* __restrict__ base, Geom g, Eos E, const __grid_constant__ CUtensorMap tm) {
  extern __shared__ __align__(128) unsigned char st_smem_raw[];
  SrcTileSmem& sm = *reinterpret_cast<SrcTileSmem*>(st_smem_raw);
  const int tx = threadIdx.x, ty = threadIdx.y;
  const int i0 = blockIdx.x * ST_BX, j0 = blockIdx.y * ST_BY, k = blockIdx.z;
  if (tx == 0 && ty == 0) {
    ft_mbar_init(&sm.bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    ft_mbar_expect(&sm.bar, (unsigned)sizeof(sm.tile));
    ft_tma_4d(&sm.tile[0][0][0], &tm, &sm.bar, i0 - 2 + X0, j0 - 2 + G, k + G, F_MET);
  }
  const int i = i0 + tx, j = j0 + ty;
  const bool in = i < g.nx && j < g.ny;
  const int c = (int)g.at(min(i, g.nx - 1), min(j, g.ny - 1), k);
  // ---- plain loads first: primitives, K_ij, z stencils (they overlap the tile's flight)
  const Prim P = load_prim(base, g, c);
  double Kc[6];
#pragma unroll
  for (int q = 0; q < 6; q++) Kc[q] = fld(base, g, F_MET + 10 + q)[c];
  const int sz = (int)g.sz;
  double dz[ST_NF];
  {
    const double w = g.idx[2] * (1.0 / 12.0);
#pragma unroll
    for (int f = 0; f < ST_NF; f++) dz[f] = d4(fld(base, g, F_MET + f), c, sz, w);
  }
  __syncthreads();            // the mbarrier is initialised
  ft_mbar_wait(&sm.bar, 0u);  // the tile has landed
  const int sx = tx + 2, sy = ty + 2;
  double m[ST_NF], dx[ST_NF], dy[ST_NF];
  {
    const double wx = g.idx[0] * (1.0 / 12.0), wy = g.idx[1] * (1.0 / 12.0);
#pragma unroll
    for (int f = 0; f < ST_NF; f++) {
      const double (*t)[ST_TX] = sm.tile[f];
      m[f] = t[sy][sx];
      dx[f] = (8.0 * (t[sy][sx + 1] - t[sy][sx - 1]) - (t[sy][sx + 2] - t[sy][sx - 2])) * wx;
      dy[f] = (8.0 * (t[sy + 1][sx] - t[sy - 1][sx]) - (t[sy + 2][sx] - t[sy - 2][sx])) * wy;
    }
  }
  if (!in) return;
  Met M;
  M.a = m[0]; M.bx = m[1]; M.by = m[2]; M.bz = m[3];
  M.gxx = m[4]; M.gxy = m[5]; M.gxz = m[6]; M.gyy = m[7]; M.gyz = m[8]; M.gzz = m[9];
  const double det = det_gamma(M);
  const double sg = det * ft_rsqrt(det);
  const SrcCoef sc = source_coef(P, M, E);
  double St = 2.0 * contract(sc.C, Kc[0], Kc[1], Kc[2], Kc[3], Kc[4], Kc[5]);
  const double asg = M.a * sg;
  double S[4];
  src_axis(sc, 0, dx, asg, S, St);
  src_axis(sc, 1, dy, asg, S, St);
  src_axis(sc, 2, dz, asg, S, St);
  S[3] = asg * St;
#pragma unroll
  for (int r = 0; r < 4; r++) fld(base, g, F_SRC + r)[c] = S[r];
}

}  // namespace gk

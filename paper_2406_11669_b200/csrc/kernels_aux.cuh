// kernels_aux.cuh -- layout conversion, ghost fill (A1), B from A (A6/R13), con2prim (A2),
// max-speed reduction (A8), dt.
#pragma once
#include "layout.cuh"
#include "recon_c2p.cuh"

namespace gk {

__device__ __forceinline__ const double* fld(const double* base, const Geom& g, int id) {
  return base + (size_t)id * g.NPA;
}
__device__ __forceinline__ double* fld(double* base, const Geom& g, int id) {
  return base + (size_t)id * g.NPA;
}

__device__ __forceinline__ Met load_met(const double* base, const Geom& g, long long c) {
  Met M;
  M.a = fld(base, g, F_MET + 0)[c];
  M.bx = fld(base, g, F_MET + 1)[c]; M.by = fld(base, g, F_MET + 2)[c];
  M.bz = fld(base, g, F_MET + 3)[c];
  M.gxx = fld(base, g, F_MET + 4)[c]; M.gxy = fld(base, g, F_MET + 5)[c];
  M.gxz = fld(base, g, F_MET + 6)[c]; M.gyy = fld(base, g, F_MET + 7)[c];
  M.gyz = fld(base, g, F_MET + 8)[c]; M.gzz = fld(base, g, F_MET + 9)[c];
  return M;
}

__device__ __forceinline__ Prim load_prim(const double* base, const Geom& g, long long c) {
  Prim P;
  P.rho = fld(base, g, F_P + 0)[c]; P.vx = fld(base, g, F_P + 1)[c];
  P.vy = fld(base, g, F_P + 2)[c]; P.vz = fld(base, g, F_P + 3)[c];
  P.p = fld(base, g, F_P + 4)[c];
  P.Bx = fld(base, g, F_BC + 0)[c]; P.By = fld(base, g, F_BC + 1)[c];
  P.Bz = fld(base, g, F_BC + 2)[c];
  return P;
}

// ------------------------------------------------------------------ layout conversion
// external array (ez, ey, ex), x fastest, element (0,0,0) = grid index (-G,-G,-G)
// <-> internal padded array.  One thread per external element.
__global__ void k_repack_in(const double* __restrict__ ext, double* __restrict__ dst, Geom g,
                            int ex, int ey, int ez) {
  const long long n = (long long)ex * ey * ez;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < n;
       q += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(q % ex), j = (int)((q / ex) % ey), k = (int)(q / ((long long)ex * ey));
    dst[g.at(i - G, j - G, k - G)] = ext[q];
  }
}

// mode 0: plain copy; mode 1: interior cells only, divided by sqrt(gamma) of the cell
// (get_cons rows D,S_j,tau), ghosts 0; mode 2: interior cells only, ghosts 0.
__global__ void k_repack_out(const double* __restrict__ src, double* __restrict__ ext,
                             const double* __restrict__ base, Geom g, int ex, int ey, int ez,
                             int mode) {
  const long long n = (long long)ex * ey * ez;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < n;
       q += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(q % ex) - G, j = (int)((q / ex) % ey) - G,
              k = (int)(q / ((long long)ex * ey)) - G;
    const long long c = g.at(i, j, k);
    double v = src[c];
    if (mode != 0) {
      const bool in = i >= 0 && i < g.nx && j >= 0 && j < g.ny && k >= 0 && k < g.nz;
      if (!in) v = 0.0;
      else if (mode == 1) v = v / sqrt(det_gamma(load_met(base, g, c)));
    }
    ext[q] = v;
  }
}

__global__ void k_repack_mask(const unsigned char* __restrict__ ext,
                              unsigned char* __restrict__ dst, Geom g) {
  const int ex = g.nx + 2 * G, ey = g.ny + 2 * G, ez = g.nz + 2 * G;
  const long long n = (long long)ex * ey * ez;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < n;
       q += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(q % ex), j = (int)((q / ex) % ey), k = (int)(q / ((long long)ex * ey));
    dst[g.at(i - G, j - G, k - G)] = ext[q];
  }
}

__global__ void k_fill_zero(double* __restrict__ p, long long n) {
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < n;
       q += (long long)gridDim.x * blockDim.x)
    p[q] = 0.0;
}

// ------------------------------------------------------------------------- ghost fill
// R15 / PAPER.md:350: one pass along axis `a` for up to 8 fields (blockIdx.z = field).
// The transverse range is the full padded extent on axes already filled (< a) and the
// valid range on axes still to come (> a), so that edges and corners end up filled after
// the x, y, z passes.  stag bit b = field staggered along axis b; kind 0 = copy of the
// nearest valid value (outflow) , 1 = linear extrapolation layer by layer (A_i); periodic
// axes wrap with period n (staggered index n = image of 0).
struct FillArgs {
  int id[8];
  int stag[8];  // bit mask
  int kind[8];
  int nf;
};

// one item of the pass along axis a: field f, transverse position tid (false: past the end)
__device__ __forceinline__ bool fill_axis_item(double* __restrict__ base, const Geom& g,
                                               const FillArgs& fa, int a, int f, long long tid) {
  double* q = fld(base, g, fa.id[f]);
  const int st = fa.stag[f], kind = fa.kind[f];
  const int b0 = (a + 1) % 3, b1 = (a + 2) % 3;
  const int lo0 = b0 < a ? -G : 0, hi0 = g.n(b0) - 1 + ((st >> b0) & 1) + (b0 < a ? G : 0);
  const int lo1 = b1 < a ? -G : 0, hi1 = g.n(b1) - 1 + ((st >> b1) & 1) + (b1 < a ? G : 0);
  const int n0 = hi0 - lo0 + 1, n1 = hi1 - lo1 + 1;
  if (tid >= (long long)n0 * n1) return false;
  // make the x-like axis the fast thread index whenever it is transverse
  int t0, t1;
  if (b0 == 0 || (b1 != 0 && b0 < b1)) { t0 = (int)(tid % n0); t1 = (int)(tid / n0); }
  else { t1 = (int)(tid % n1); t0 = (int)(tid / n1); }
  int I[3];
  I[b0] = lo0 + t0; I[b1] = lo1 + t1;
  const int na = g.n(a), sa = (st >> a) & 1;
  const bool periodic = g.bc[a] == 0;
  const int hi = na - 1 + sa, ghi = na + G - 1 + sa;
  const long long sd = g.stride(a);
  I[a] = 0;
  const long long c0 = g.at(I[0], I[1], I[2]);  // index of layer 0 along a
  if (periodic) {
    for (int gl = -1; gl >= -G; gl--) {
      const int src = ((gl % na) + na) % na;
      q[c0 + gl * sd] = q[c0 + src * sd];
    }
    for (int gl = na; gl <= ghi; gl++) {
      const int src = gl % na;
      q[c0 + gl * sd] = q[c0 + src * sd];
    }
  } else if (kind == 0) {
    const double vlo = q[c0], vhi = q[c0 + hi * sd];
    for (int gl = -1; gl >= -G; gl--) q[c0 + gl * sd] = vlo;
    for (int gl = hi + 1; gl <= ghi; gl++) q[c0 + gl * sd] = vhi;
  } else {
    double q1 = q[c0], q2 = q[c0 + sd];
    for (int gl = -1; gl >= -G; gl--) {
      const double v = 2.0 * q1 - q2;
      q[c0 + gl * sd] = v;
      q2 = q1; q1 = v;
    }
    q1 = q[c0 + hi * sd]; q2 = q[c0 + (hi - 1) * sd];
    for (int gl = hi + 1; gl <= ghi; gl++) {
      const double v = 2.0 * q1 - q2;
      q[c0 + gl * sd] = v;
      q2 = q1; q1 = v;
    }
  }
  return true;
}

__global__ void k_fill_axis(double* __restrict__ base, Geom g, FillArgs fa, int a) {
  const int f = blockIdx.z;
  if (f >= fa.nf) return;
  fill_axis_item(base, g, fa, a, f, blockIdx.x * (long long)blockDim.x + threadIdx.x);
}

// The x, y, z passes in ONE launch (launch-bound small blocks): one thread-block CLUSTER of
// FILL1_CTAS blocks walks the items of a pass, then a cluster barrier (arrive.release /
// wait.acquire: the global writes of every block of the cluster are ordered before the reads of
// the next pass).  Same items, same arithmetic: bit-identical to three k_fill_axis launches.
constexpr int FILL1_THREADS = 512;
constexpr int FILL1_CTAS = 8;
__global__ void __launch_bounds__(FILL1_THREADS) k_fill_axes1(double* __restrict__ base, Geom g,
                                                               FillArgs fa) {
  const int t0 = blockIdx.x * FILL1_THREADS + threadIdx.x;
  for (int a = 0; a < 3; a++) {
    const int b0 = (a + 1) % 3, b1 = (a + 2) % 3;
    const long long nt = (long long)(g.n(b0) + 2 * G + 1) * (g.n(b1) + 2 * G + 1);
    for (long long w = t0; w < nt * fa.nf; w += FILL1_THREADS * FILL1_CTAS)
      fill_axis_item(base, g, fa, a, (int)(w / nt), w % nt);
    asm volatile("barrier.cluster.arrive.release.aligned;\n"
                 "barrier.cluster.wait.acquire.aligned;" ::: "memory");
  }
}

// R15 for unstaggered copy / wrap fields (the primitives) in one launch: the x, y, z passes of
// k_fill_axis compose to one index map per axis (wrap with period n, or clamp to the nearest
// interior cell), so every ghost cell reads its interior source directly -- bit-identical, and
// two launches fewer per substep on blocks that are launch bound.  One thread per padded cell.
__global__ void k_fill_copy3(double* __restrict__ base, Geom g, FillArgs fa) {
  const int W0 = g.nx + 2 * G, W1 = g.ny + 2 * G, W2 = g.nz + 2 * G;
  const long long tid = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (tid >= (long long)W0 * W1 * W2) return;
  const int i = (int)(tid % W0) - G, j = (int)((tid / W0) % W1) - G;
  const int k = (int)(tid / ((long long)W0 * W1)) - G;
  if (i >= 0 && i < g.nx && j >= 0 && j < g.ny && k >= 0 && k < g.nz) return;
  const int I[3] = {i, j, k};
  int S[3];
#pragma unroll
  for (int a = 0; a < 3; a++) {
    const int n = g.n(a);
    S[a] = g.bc[a] == 0 ? ((I[a] % n) + n) % n : min(max(I[a], 0), n - 1);
  }
  double* q = fld(base, g, fa.id[blockIdx.z]);
  q[g.at(i, j, k)] = q[g.at(S[0], S[1], S[2])];
}

// ------------------------------------------------------------------ static face metric
// R4 (adapted per G3), once per grmhd_set_metric since the ADM variables are held
// fixed: for the lower D-face of every padded index, the 4-point Lagrange values
// q_f = (-q_{i-2} + 9 q_{i-1} + 9 q_i - q_{i+1})/16 of alpha, beta^k, gamma_kl along D and
// sqrt(det gamma_f) -> field family F_FM + NFM D.  Faces whose stencil leaves the cells the
// caller supplied (i_D outside [-1, n_D + 1], or a transverse index outside [-G, n + G)) take
// the value of the nearest face inside: never used by a stored flux, but finite.
template <int D>
__global__ void __launch_bounds__(128)
k_face_metric(double* __restrict__ base, Geom g) {
  const int ix = blockIdx.x * blockDim.x + threadIdx.x;
  const int iy = blockIdx.y * blockDim.y + threadIdx.y;
  const int iz = blockIdx.z;
  if (ix >= g.PXP || iy >= g.PY) return;
  const long long dst = (long long)iz * g.sz + (long long)iy * g.sy + ix;
  int I[3] = {ix - X0, iy - G, iz - G};
#pragma unroll
  for (int a = 0; a < 3; a++) {
    const int lo = a == D ? -1 : -G, hi = a == D ? g.n(a) + 1 : g.n(a) + G - 1;
    I[a] = min(max(I[a], lo), hi);
  }
  const long long c = g.at(I[0], I[1], I[2]);
  const long long sd = g.stride(D);
  double m[10];
#pragma unroll
  for (int v = 0; v < 10; v++) {
    const double* q = fld(base, g, F_MET + v);
    m[v] = (-q[c - 2 * sd] + 9.0 * q[c - sd] + 9.0 * q[c] - q[c + sd]) * 0.0625;
    fld(base, g, F_FM + NFM * D + v)[dst] = m[v];
  }
  Met M;
  M.a = m[0]; M.bx = m[1]; M.by = m[2]; M.bz = m[3];
  M.gxx = m[4]; M.gxy = m[5]; M.gxz = m[6]; M.gyy = m[7]; M.gyz = m[8]; M.gzz = m[9];
  fld(base, g, F_FM + NFM * D + 10)[dst] = sqrt(det_gamma(M));
}

// --------------------------------------------------------------------------- B from A
// R13: B~^i = B~0^i + [ijk] d_j A_k on faces (eq. 24 PAPER.md:149 with
// epsilon^{ijk} = [ijk]/sqrt(gamma)), then the cell-centre value as the mean
// of the two faces divided by sqrt(gamma).  One thread per padded index
// (i,j,k) in [-G, n+G]; a face whose edges do not all exist keeps the static value.
__device__ __forceinline__ double face_bx(const double* Ay, const double* Az, const double* B0x,
                                          const Geom& g, long long c) {
  return B0x[c] + (Az[c + g.sy] - Az[c]) * g.idx[1] - (Ay[c + g.sz] - Ay[c]) * g.idx[2];
}
__device__ __forceinline__ double face_by(const double* Ax, const double* Az, const double* B0y,
                                          const Geom& g, long long c) {
  return B0y[c] + (Ax[c + g.sz] - Ax[c]) * g.idx[2] - (Az[c + 1] - Az[c]) * g.idx[0];
}
__device__ __forceinline__ double face_bz(const double* Ax, const double* Ay, const double* B0z,
                                          const Geom& g, long long c) {
  return B0z[c] + (Ay[c + 1] - Ay[c]) * g.idx[0] - (Ax[c + g.sy] - Ax[c]) * g.idx[1];
}

// G16: static face field B~0^d = mean over the two cells sharing the face of
// sqrt(gamma_c) B^d_c, for faces 0..n_d along d and interior transverse indices.
// Bin = ghost-filled cell-centred input component (temporarily held in F_BF + d).
__global__ void k_b0_from_centred(double* __restrict__ base, Geom g, int d) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  if (i >= g.nx + (d == 0) || j >= g.ny + (d == 1) || k >= g.nz + (d == 2)) return;
  const long long c = g.at(i, j, k), cm = c - g.stride(d);
  const double* Bin = fld(base, g, F_BF + d);
  const double sgc = sqrt(det_gamma(load_met(base, g, c)));
  const double sgm = sqrt(det_gamma(load_met(base, g, cm)));
  fld(base, g, F_B0 + d)[c] = 0.5 * (sgm * Bin[cm] + sgc * Bin[c]);
}

// ------------------------------------------------------------------------- reductions
__device__ __forceinline__ void block_max3_atomic(double m0, double m1, double m2,
                                                  unsigned long long* acc) {
  __shared__ double sm[3][32];
  const int lane = threadIdx.x & 31;
  const int tid = threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z);
  const int warp = tid >> 5;
  const int nw = (blockDim.x * blockDim.y * blockDim.z + 31) >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    m0 = fmax(m0, __shfl_xor_sync(0xffffffffu, m0, o));
    m1 = fmax(m1, __shfl_xor_sync(0xffffffffu, m1, o));
    m2 = fmax(m2, __shfl_xor_sync(0xffffffffu, m2, o));
  }
  if ((tid & 31) == 0) { sm[0][warp] = m0; sm[1][warp] = m1; sm[2][warp] = m2; }
  __syncthreads();
  if (warp == 0) {
    m0 = (tid < nw) ? sm[0][tid] : 0.0;
    m1 = (tid < nw) ? sm[1][tid] : 0.0;
    m2 = (tid < nw) ? sm[2][tid] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      m0 = fmax(m0, __shfl_xor_sync(0xffffffffu, m0, o));
      m1 = fmax(m1, __shfl_xor_sync(0xffffffffu, m1, o));
      m2 = fmax(m2, __shfl_xor_sync(0xffffffffu, m2, o));
    }
    if (tid == 0) {
      // non-negative doubles order like their bit patterns: the max is exact and
      // independent of the order of arrival
      atomicMax(acc + 0, (unsigned long long)__double_as_longlong(m0));
      atomicMax(acc + 1, (unsigned long long)__double_as_longlong(m1));
      atomicMax(acc + 2, (unsigned long long)__double_as_longlong(m2));
    }
  }
  (void)lane;
}

// R16: max(|lambda_-|, |lambda_+|) per direction at a cell centre
__device__ __forceinline__ void cell_speeds(const Prim& P, const Met& M, const Eos& E,
                                            double s[3]) {
  const double idet = ft_rcp(det_gamma(M));
  const Pt pt = point_state(P, M, E);
  double lm, lp;
  char_speeds<0>(P, pt, M, inv_gamma_dd<0>(M, idet), E, lm, lp);
  s[0] = fmax(fabs(lm), fabs(lp));
  char_speeds<1>(P, pt, M, inv_gamma_dd<1>(M, idet), E, lm, lp);
  s[1] = fmax(fabs(lm), fabs(lp));
  char_speeds<2>(P, pt, M, inv_gamma_dd<2>(M, idet), E, lm, lp);
  s[2] = fmax(fabs(lm), fabs(lp));
#pragma unroll
  for (int d = 0; d < 3; d++)
    if (!(s[d] == s[d])) s[d] = 0.0;  // a NaN never wins the max (same as `s > m`)
}

// ------------------------------------------------------------ fused post-update kernel
// 4th-order centred derivative (G12); this operand order gives exactly 0 on constants
__device__ __forceinline__ double d4(const double* __restrict__ q, int c, int sd, double i12dx) {
  return (8.0 * (q[c + sd] - q[c - sd]) - (q[c + 2 * sd] - q[c - 2 * sd])) * i12dx;
}

// One axis of R9: d[0..9] = d_a of alpha, beta^x, beta^y, beta^z, gamma_xx .. gamma_zz at the cell.
// S_a = alpha sqrt(gamma) (C^{ik} d_a gamma_ik - T^{00} alpha d_a alpha + T^0_i d_a beta^i) and
// the d_a alpha part of S_tau.
__device__ __forceinline__ void src_axis(const SrcCoef& sc, int a, const double d[10], double asg,
                                         double S[4], double& St) {
  const double cg = contract(sc.C, d[4], d[5], d[6], d[7], d[8], d[9]);
  S[a] = asg * (cg - sc.T00a * d[0] + sc.T0lx * d[1] + sc.T0ly * d[2] + sc.T0lz * d[3]);
  St -= (a == 0 ? sc.ax : (a == 1 ? sc.ay : sc.az)) * d[0];
}

// R9 / G11: alpha sqrt(gamma) S for the rows S_x, S_y, S_z, tau at an interior cell
// (eq. (19) PAPER.md:125 in 3+1 form; metric derivatives PAPER.md:384)
__device__ __forceinline__ void cell_sources(const double* __restrict__ base, const Geom& g, int c,
                                             const Prim& P, const Met& M, double sg,
                                             const Eos& E, double S[4]) {
  const SrcCoef sc = source_coef(P, M, E);
  // S_tau, curvature part: 2 C^{ik} K_ik
  double St = 2.0 * contract(sc.C, fld(base, g, F_MET + 10)[c], fld(base, g, F_MET + 11)[c],
                             fld(base, g, F_MET + 12)[c], fld(base, g, F_MET + 13)[c],
                             fld(base, g, F_MET + 14)[c], fld(base, g, F_MET + 15)[c]);
  const double asg = M.a * sg;
#pragma unroll
  for (int a = 0; a < 3; a++) {
    const int sd = a == 0 ? 1 : (a == 1 ? (int)g.sy : (int)g.sz);
    const double w = g.idx[a] * (1.0 / 12.0);
    double d[10];
#pragma unroll
    for (int f = 0; f < 10; f++) d[f] = d4(fld(base, g, F_MET + f), c, sd, w);
    src_axis(sc, a, d, asg, S, St);
  }
  S[3] = asg * St;
}

// After a change of (U~, A) (an RK stage) or of the initial data: one pass that
//   R13  builds B~ = B~0 + curl A on the lower faces of every padded index and the
//        cell-centred B^i (mean of the two faces / sqrt(gamma)),
//   R14  recovers the primitives of the interior cells (INIT: takes the given primitives
//        and forms U~ = sqrt(gamma) U(P, B_c) instead, eqs (20)-(22)),
//   R9   stores alpha sqrt(gamma) S of those primitives for the next k_update,
//   R16  accumulates the max characteristic speeds when want_speed.
// One thread per padded index (i,j,k) in [-G, n+G].
#ifndef KP_BY
#define KP_BY 4
#endif
#ifndef KP_BZ
#define KP_BZ 1
#endif
constexpr int KP_THREADS = 32 * KP_BY * KP_BZ;
#ifndef KP_MINB
#define KP_MINB 5
#endif
// The metric and U~ rows are first used after the stores of B~ and B_c, which the compiler cannot
// move loads across (one workspace: it must assume aliasing): their lines are asked for at kernel
// entry with prefetch.global.L2, at no register cost.  Measured at 256^3: 1.350 ms without,
// 1.315 ms with (L1 instead of L2: 1.320 ms).
#ifndef KP_PREFETCH
#define KP_PREFETCH 1
#endif
__device__ __forceinline__ void kp_opaque(double& x) { asm volatile("" : "+d"(x)); }
__device__ __forceinline__ void kp_prefetch(const double* p) {
  asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}
// SRC (launch-bound small blocks): also R9, the sources of the recovered primitives (otherwise
// k_src / k_src_tile).  flags: bit 0 = accumulate the max speeds, bit 1 = end of a step, t += dt
// (otherwise k_dt mode 1).
template <bool INIT, bool BACKUP, bool SRC = false>
__global__ void __launch_bounds__(KP_THREADS, SRC ? 1 : KP_MINB)
k_post(double* __restrict__ base, const unsigned char* __restrict__ mask, Geom g, Eos E,
       DevState* __restrict__ st, int flags) {
  const int want_speed = flags & 1;
  if ((flags & 2) && blockIdx.x + blockIdx.y + blockIdx.z == 0 &&
      threadIdx.x + threadIdx.y + threadIdx.z == 0)
    st->t += st->dt;
  const int i = blockIdx.x * 32 + threadIdx.x - G;
  const int j = blockIdx.y * KP_BY + threadIdx.y - G;
  const int kraw = blockIdx.z * KP_BZ + threadIdx.z - G;
  const int k = min(kraw, g.nz + G);
  const bool inpad = i <= g.nx + G && j <= g.ny + G && kraw <= g.nz + G;
  const int c = (int)g.at(min(i, g.nx + G), min(j, g.ny + G), k);
  const bool ix = i < g.nx + G, jy = j < g.ny + G, kz = k < g.nz + G;
  double Bx = 0.0, By = 0.0, Bz = 0.0;
  Met M;
  double sg = 1.0;
#if KP_PREFETCH
  if (!INIT && (threadIdx.x & 15) == 0) {  // one request per 128-byte line (c is clamped: valid)
#pragma unroll
    for (int f = 0; f < 10; f++) kp_prefetch(fld(base, g, F_MET + f) + c);
#pragma unroll
    for (int r = 0; r < 5; r++) kp_prefetch(fld(base, g, F_Y + r) + c);
  }
#endif
  if (inpad) {
    const double* Ax = fld(base, g, F_Y + 5);
    const double* Ay = fld(base, g, F_Y + 6);
    const double* Az = fld(base, g, F_Y + 7);
    const double* B0x = fld(base, g, F_B0 + 0);
    const double* B0y = fld(base, g, F_B0 + 1);
    const double* B0z = fld(base, g, F_B0 + 2);
    const double bx = (jy && kz) ? face_bx(Ay, Az, B0x, g, c) : B0x[c];
    const double by = (ix && kz) ? face_by(Ax, Az, B0y, g, c) : B0y[c];
    const double bz = (ix && jy) ? face_bz(Ax, Ay, B0z, g, c) : B0z[c];
    fld(base, g, F_BF + 0)[c] = bx;
    fld(base, g, F_BF + 1)[c] = by;
    fld(base, g, F_BF + 2)[c] = bz;
    if (ix && jy && kz) {
      M = load_met(base, g, c);
      const double det = det_gamma(M);
      const double isg = ft_rsqrt(det);
      sg = det * isg;
      Bx = 0.5 * (bx + face_bx(Ay, Az, B0x, g, c + 1)) * isg;
      By = 0.5 * (by + face_by(Ax, Az, B0y, g, c + g.sy)) * isg;
      Bz = 0.5 * (bz + face_bz(Ax, Ay, B0z, g, c + g.sz)) * isg;
      fld(base, g, F_BC + 0)[c] = Bx;
      fld(base, g, F_BC + 1)[c] = By;
      fld(base, g, F_BC + 2)[c] = Bz;
    }
  }
  const bool in = inpad && i >= 0 && i < g.nx && j >= 0 && j < g.ny && k >= 0 && k < g.nz;
  double s[3] = {0.0, 0.0, 0.0};
  int bits = 0, iters = 0;
  if (in) {
    double P5[5];
    if (INIT) {
#pragma unroll
      for (int r = 0; r < 5; r++) P5[r] = fld(base, g, F_P + r)[c];
      const Prim P = {P5[0], P5[1], P5[2], P5[3], P5[4], Bx, By, Bz};
      double U[5];
      prim2con(P, M, E, U);
#pragma unroll
      for (int r = 0; r < 5; r++) fld(base, g, F_Y + r)[c] = sg * U[r];
    } else {
      const double isg = ft_rcp(sg);
      double U[5];
#pragma unroll
      for (int r = 0; r < 5; r++) U[r] = fld(base, g, F_Y + r)[c] * isg;  // undensitise, eq. (17)
      int rewrite;
      bits = con2prim<BACKUP>(U, Bx, By, Bz, M, E, mask != nullptr && mask[c] != 0, P5, iters,
                              rewrite);
#pragma unroll
      for (int r = 0; r < 5; r++) fld(base, g, F_P + r)[c] = P5[r];
      if (rewrite & 1) fld(base, g, F_Y + 0)[c] = sg * U[0];
      if (rewrite & 2) {
#pragma unroll
        for (int r = 1; r < 5; r++) fld(base, g, F_Y + r)[c] = sg * U[r];
      }
    }
    const Prim P = {P5[0], P5[1], P5[2], P5[3], P5[4], Bx, By, Bz};
    if (want_speed) cell_speeds(P, M, E, s);
    if (SRC) {
      // The inputs pass through an opaque barrier: without it the compiler shares sub-expressions
      // (point_state, det gamma, gamma^ij) with con2prim / prim2con above and contracts other
      // products into FMAs than in the stand-alone k_src -- the results then differ in the last
      // bit.  With it cell_sources is compiled as in k_src: bit-identical.
      Prim Ps = P;
      Met Ms = M;
      double sgs = sg;
      kp_opaque(Ps.rho); kp_opaque(Ps.vx); kp_opaque(Ps.vy); kp_opaque(Ps.vz); kp_opaque(Ps.p);
      kp_opaque(Ps.Bx); kp_opaque(Ps.By); kp_opaque(Ps.Bz);
      kp_opaque(Ms.a); kp_opaque(Ms.bx); kp_opaque(Ms.by); kp_opaque(Ms.bz);
      kp_opaque(Ms.gxx); kp_opaque(Ms.gxy); kp_opaque(Ms.gxz);
      kp_opaque(Ms.gyy); kp_opaque(Ms.gyz); kp_opaque(Ms.gzz);
      kp_opaque(sgs);
      double S[4];
      cell_sources(base, g, c, Ps, Ms, sgs, E, S);
#pragma unroll
      for (int r = 0; r < 4; r++) fld(base, g, F_SRC + r)[c] = S[r];
    }
  }
  if (!INIT) {
    // counters: integer sums and maxima, order independent
    const unsigned any = __ballot_sync(0xffffffffu, bits != 0);
    if (any) {
      const int nf = __popc(__ballot_sync(0xffffffffu, (bits & 2) != 0));
      const int np = __popc(__ballot_sync(0xffffffffu, (bits & 4) != 0));
      const int na = __popc(__ballot_sync(0xffffffffu, (bits & 1) != 0));
      const int nw = __popc(__ballot_sync(0xffffffffu, (bits & 8) != 0));
      const int nb = __popc(__ballot_sync(0xffffffffu, (bits & 16) != 0));
      if (threadIdx.x == 0) {
        if (nf) atomicAdd((unsigned long long*)&st->c2p_fail, (unsigned long long)nf);
        if (np) atomicAdd((unsigned long long*)&st->p_fix, (unsigned long long)np);
        if (na) atomicAdd((unsigned long long*)&st->atmo, (unsigned long long)na);
        if (nw) atomicAdd((unsigned long long*)&st->w_cap, (unsigned long long)nw);
        if (nb) atomicAdd((unsigned long long*)&st->c2p_backup, (unsigned long long)nb);
      }
    }
    int mi = iters;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mi = max(mi, __shfl_xor_sync(0xffffffffu, mi, o));
    if (threadIdx.x == 0 && mi > 0)
      atomicMax((long long*)&st->c2p_maxiter, (long long)mi);
  }
  if (want_speed) block_max3_atomic(s[0], s[1], s[2], st->ms_acc);
}

// R9: alpha sqrt(gamma) S of the interior cells from the primitives k_post just stored, for
// the next k_update.  Its own kernel: the 120 stencil loads of the metric derivatives want
// L1 and registers that the Newton iteration of k_post would otherwise hold.
#ifndef KS_MINB
#define KS_MINB 4
#endif
#ifndef KS_BX
#define KS_BX 32
#endif
#ifndef KS_BY
#define KS_BY 4
#endif
__global__ void __launch_bounds__(KS_BX * KS_BY, KS_MINB)
k_src(double* __restrict__ base, Geom g, Eos E) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  if (i >= g.nx || j >= g.ny) return;
  const int c = (int)g.at(i, j, k);
  const Met M = load_met(base, g, c);
  const Prim P = load_prim(base, g, c);
  const double det = det_gamma(M);
  const double sg = det * ft_rsqrt(det);
  double S[4];
  cell_sources(base, g, c, P, M, sg, E, S);
#pragma unroll
  for (int r = 0; r < 4; r++) fld(base, g, F_SRC + r)[c] = S[r];
}

// ---------------------------------------------------------------------------------- dt
// R16 / G22: dt = cfl * min_d dx_d / maxspeed_d (or fixed_dt), clipped to t_end when
// t_end >= 0.  mode 0: start of a step (compute dt, reset the accumulator);
// mode 1: end of a step (t += dt).
__global__ void k_dt(DevState* st, Geom g, int mode) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  if (mode == 1) { st->t += st->dt; return; }
  double dt;
  double ms[3];
  for (int d = 0; d < 3; d++) {
    ms[d] = __longlong_as_double((long long)st->ms_acc[d]);
    st->ms_used[d] = ms[d];
    st->ms_acc[d] = 0ull;
  }
  if (st->fixed_dt > 0.0) dt = st->fixed_dt;
  else {
    double m = INFINITY;
    for (int d = 0; d < 3; d++) m = fmin(m, g.dx[d] / ms[d]);
    dt = st->cfl * m;
  }
  if (!(dt > 0.0) || !isfinite(dt)) { st->bad_dt = 1; dt = 0.0; }
  else if (st->t_end >= 0.0 && dt > st->t_end - st->t) dt = st->t_end - st->t;
  st->dt = dt;
}

}  // namespace gk

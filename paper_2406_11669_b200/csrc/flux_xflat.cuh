// flux_xflat.cuh -- A3 + A4 along x: one thread per cell, a block of 128 threads owns 128
// CONSECUTIVE array positions of a z-plane swept in memory order (rows follow one another: the
// row pitch is nx + 8, so 257 of every 264 positions carry a face that is needed).
//
// Every load and store of the block is one contiguous, aligned 1 KB segment.  The cell of a
// thread yields its own limited slope, interface value and parabola exactly once (R5 / G8);
// what a thread needs from its neighbours -- slope of c+1, interface c-1/2, q^+ of c-1 -- goes
// through two small shared-memory arrays with one __syncthreads per exchange (three per block).
// Raw neighbour values (q_{c-1}, q_{c+1}, p_{c-2}, p_{c+2}) are plain loads: the lines are the
// block's own.  Thread t then solves the Riemann problem of the face below its cell (R7).  Since
// every slope comes from loaded values, only the 2 lowest threads and the highest one of a block
// lack a neighbour's interface value: 125 faces per 128 threads, against 27 per 32 when a warp
// works alone with shuffles (flux_xrow.cuh, which still serves y and z on blocks narrower than 32
// cells and the apron columns).
#pragma once
#include "flux_face.cuh"

namespace gk {

#ifndef XF_NTHREADS
#define XF_NTHREADS 128
#endif
constexpr int XF_THREADS = XF_NTHREADS;
constexpr int XF_VALID = XF_THREADS - 3;  // faces per block: threads 2 .. 126
#ifndef XF_MINB
#define XF_MINB 5
#endif

// faces of one z-plane: rows j in [-ap, ny + ap), flat offsets o = (j + ap) * sy + (x index)
__host__ __device__ inline long long xf_items_per_plane(const Geom& g, int ap) {
  const long long last = (long long)(g.ny + 2 * ap - 1) * g.sy + X0 + g.nx;  // last needed offset
  return (last + XF_VALID) / XF_VALID;
}

// RECON: 0 minmod, 1 PPM without flattening, 2 PPM with flattening.  grid: x = items, one block
// per item; item = plane * items_per_plane + segment, plane k = item / ipp - ap.
template <int RECON, bool UCT>
__global__ void __launch_bounds__(XF_THREADS, XF_MINB)
k_flux_xflat(double* __restrict__ base, Geom g, Eos E, int ap, int ipp) {
  __shared__ double sa[FX_NV][XF_THREADS + 2], sb[FX_NV][XF_THREADS + 2];
  const int t = threadIdx.x;
  const int plane = (int)(blockIdx.x / ipp), seg = (int)(blockIdx.x % ipp);
  const int sy = (int)g.sy;
  const int o = seg * XF_VALID - 2 + t;              // flat offset inside the plane's rows
  const int p0 = (int)g.at(-X0, -ap, plane - ap);    // x index 0 of row -ap
  const int np1 = (int)g.NP - 1;
  const int idx = min(max(p0 + o, 0), np1);
  const int im1 = max(idx - 1, 0), ip1 = min(idx + 1, np1);

  // ---- cell data of the thread and its raw neighbours
  double q[FX_NV], qm1[FX_NV], qp1[FX_NV];
#pragma unroll
  for (int v = 0; v < FX_NV; v++) {
    const double* f = fld(base, g, flux_var_field(0, v));
    q[v] = f[idx]; qm1[v] = f[im1]; qp1[v] = f[ip1];
  }
  const double bfx = fld(base, g, F_BF)[idx];
  double mv11[NFM];
#pragma unroll
  for (int v = 0; v < NFM; v++) mv11[v] = fld(base, g, F_FM + v)[idx];
  // G8(c): flattening coefficient of the thread's cell
  double f = 0.0;
  bool anyf = false;
  if (RECON == 2) {
    const double* pp = fld(base, g, F_P + 4);
    f = ft_flatten(pp[max(idx - 2, 0)], qm1[4], qp1[4], pp[min(idx + 2, np1)], qm1[1], qp1[1]);
    anyf = __any_sync(0xffffffffu, f != 0.0);
  }
  // ---- reconstruction: q^-_c -> qR (right state of the thread's face), q^+_{c-1} -> qL
  double qL[FX_NV], qR[FX_NV], qp[FX_NV];
  if (RECON == 0) {  // G7
#pragma unroll
    for (int v = 0; v < FX_NV; v++) {
      const double dl = q[v] - qm1[v], dr = qp1[v] - q[v];
      const double m = fabs(dl) < fabs(dr) ? dl : dr;
      const double s = dl * dr > 0.0 ? m : 0.0;
      qR[v] = fma(-0.5, s, q[v]);
      qp[v] = fma(0.5, s, q[v]);
    }
  } else {  // G8(a)-(d), same arithmetic as FtMarch::step
    double dm[FX_NV], ir[FX_NV];
#pragma unroll
    for (int v = 0; v < FX_NV; v++) {
      dm[v] = ft_slope2(q[v] - qm1[v], qp1[v] - q[v]);
      sa[v][t + 1] = dm[v];
    }
    __syncthreads();
#pragma unroll
    for (int v = 0; v < FX_NV; v++) {
      const double dmp = sa[v][t + 2];                                   // slope of cell c+1
      ir[v] = ft_iface(q[v], qp1[v], dm[v], dmp);                        // interface c + 1/2
      sb[v][t + 1] = ir[v];
    }
    __syncthreads();
#pragma unroll
    for (int v = 0; v < FX_NV; v++) {
      double qm = sb[v][t];                                              // interface c - 1/2
      qp[v] = ir[v];
      ft_parabola<RECON == 2>(q[v], f, anyf, qm, qp[v]);
      qR[v] = qm;
    }
  }
#pragma unroll
  for (int v = 0; v < FX_NV; v++) sa[v][t + 1] = qp[v];  // (every reader of sa passed the 2nd barrier)
  __syncthreads();
#pragma unroll
  for (int v = 0; v < FX_NV; v++) qL[v] = sa[v][t];      // q^+ of cell c-1

  // ---- Riemann problem of face c - 1/2 (R7)
  const FaceMet fmet = face_met<0>(mv11);
  double out[7], w[4];
  ft_face<0, UCT>(qL, qR, bfx, fmet, E, out, w);
  const int xi = o >= 0 ? o % sy : -1;
  const int row = o >= 0 ? o / sy : -1;
  if (t >= 2 && t < 2 + XF_VALID && xi >= X0 && xi <= X0 + g.nx && row < g.ny + 2 * ap) {
    double* ob = fld(base, g, F_FX) + idx;
    const size_t NPA = (size_t)g.NPA;
#pragma unroll
    for (int r = 0; r < 7; r++) ob[r * NPA] = out[r];
    if (UCT) {
      double* ow = fld(base, g, F_W) + idx;
#pragma unroll
      for (int r = 0; r < 4; r++) ow[r * NPA] = w[r];
    }
  }
}

}  // namespace gk

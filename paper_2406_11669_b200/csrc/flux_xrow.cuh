// flux_xrow.cuh -- A3 + A4 along x with the lanes of a warp ALONG x.
//
// x is the contiguous axis: a kernel that marches along x can only touch 32 bytes of a row at
// a time, which HBM serves badly (measured in round 1: 1.45x DRAM over-fetch, 1.7 ms against
// 1.0 ms).  Here a warp owns 32 consecutive cells c0 .. c0+31 of one row (j, k); lane = cell.  Every load and store is a contiguous
// 256-byte row segment.  The reconstruction recurrences run across lanes: the limited slope,
// the interface value and the parabola of a cell are computed once, by the cell's lane, and
// handed to the neighbour with warp shuffles (R5/G8: slope of c+1 from the lane above,
// interface c-1/2 and q^+_{c-1} from the lane below).  The lane of cell c then solves the
// Riemann problem of face c-1/2.  The 3 lowest and 2 highest lanes have incomplete stencils:
// a warp yields 27 faces; consecutive warps overlap by 5 cells.  No shared memory, no block
// barrier, nothing carried from one row segment to the next.
#pragma once
#include "flux_face.cuh"

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
    const double dm = ft_slope2(dl, dr);
    const double dmp = fx_dn(dm, 1);                             // slope of cell c+1
    const double ir = ft_iface(q, qp1, dm, dmp);                 // interface c + 1/2
    qm = fx_up(ir, 1);                                           // interface c - 1/2
    qp = ir;
    ft_parabola<RECON == 2>(q, f, anyf, qm, qp);
  }
}

// One item: the warp's 32 lanes are the cells c0 .. c0+31 along D of the pencil (t0, t1) -- with
// (t0, t1) the transverse axes: (y, z) for D = x, (x, z) for D = y, (x, y) for D = z -- and the
// lane of cell c solves face c - 1/2.  Faces outside [flo, fhi) are not stored.  Call with whole
// warps.  UCT (compile time): also store the upwind-CT face rows of F_W.
template <int D, int RECON, bool UCT>
__device__ __forceinline__ void fx_item(double* __restrict__ base, const Geom& g, const Eos& E,
                                        int c0, int t0, int t1, int flo, int fhi) {
  const int lane = threadIdx.x & 31;
  const int nD = g.n(D);
  const int c = c0 + lane;                  // this lane's cell along D; its face is c - 1/2
  const int cc = min(c, nD + G - 1);        // lanes past the last ghost cell reuse it
  const int idx = (int)(D == 0 ? g.at(cc, t0, t1) : (D == 1 ? g.at(t0, cc, t1) : g.at(t0, t1, cc)));

  // ---- cell data of the lane: rho, v^x, v^y, v^z, p and the two transverse B; the static face
  // metric and the staggered normal field of the lane's face c - 1/2
  double q[FX_NV];
#pragma unroll
  for (int v = 0; v < FX_NV; v++) q[v] = fld(base, g, flux_var_field(D, v))[idx];
  const double bfx = fld(base, g, F_BF + D)[idx];
  double mv11[NFM];
#pragma unroll
  for (int v = 0; v < NFM; v++) mv11[v] = fld(base, g, F_FM + NFM * D + v)[idx];
  // ---- neighbours across lanes
  double qm1[FX_NV], qp1[FX_NV];
#pragma unroll
  for (int v = 0; v < FX_NV; v++) { qm1[v] = fx_up(q[v], 1); qp1[v] = fx_dn(q[v], 1); }
  // G8(c): flattening coefficient of the lane's cell from p_{c-2..c+2}, v^D_{c-1}, v^D_{c+1}
  double f = 0.0;
  bool anyf = false;
  if (RECON == 2) {
    f = ft_flatten(fx_up(q[4], 2), qm1[4], qp1[4], fx_dn(q[4], 2), qm1[1 + D], qp1[1 + D]);
    anyf = __any_sync(0xffffffffu, f != 0.0);
  }
  double qL[FX_NV], qR[FX_NV];
#pragma unroll
  for (int v = 0; v < FX_NV; v++) {
    double qm, qp;
    fx_recon<RECON>(q[v], qm1[v], qp1[v], f, anyf, qm, qp);
    qL[v] = fx_up(qp, 1);  // q^+ of cell c-1
    qR[v] = qm;
  }
  // ---- Riemann problem of face c - 1/2 (R7)
  const FaceMet fmet = face_met<D>(mv11);
  double out[7], w[4];
  ft_face<D, UCT>(qL, qR, bfx, fmet, E, out, w);
  if (lane >= 3 && lane < 3 + FX_VALID && c >= flo && c < fhi) {
    double* o = fld(base, g, flux_field(D)) + idx;
    const size_t NPA = (size_t)g.NPA;
#pragma unroll
    for (int r = 0; r < 7; r++) o[r * NPA] = out[r];
    if (UCT) {
      double* ow = fld(base, g, F_W + 4 * D) + idx;
#pragma unroll
      for (int r = 0; r < 4; r++) ow[r * NPA] = w[r];
    }
  }
}

// grid: one warp per (pencil, segment) item: item = pencil * nsd + seg.  `ap` = the transverse
// apron (1 for flux-CT, R10; 3 for the upwind CT, G27):
//   mode 0: every pencil t0 in [-ap, n_t0 + ap), t1 in [-ap, n_t1 + ap).  For D = y, z the lanes
//           then run along y or z with a stride (uncoalesced: small blocks and option
//           combinations only).
//   mode 1: only the 2 ap apron columns t0 < 0 and t0 >= n_t0.
template <int D, int RECON, bool UCT>
__global__ void __launch_bounds__(FX_THREADS, FX_MINB)
k_flux_xrow(double* __restrict__ base, Geom g, Eos E, int nsd, long long nitems, int ap,
            int mode) {
  const long long nwarp = (long long)gridDim.x * (FX_THREADS / 32);
  const int nt0 = D == 0 ? g.ny : g.nx;
  const int w0 = mode ? 2 * ap : nt0 + 2 * ap;
  // grid-stride loop over the items (the launch gives every warp one item)
  for (long long item = (long long)blockIdx.x * (FX_THREADS / 32) + (threadIdx.x >> 5);
       item < nitems; item += nwarp) {
    const int seg = (int)(item % nsd);
    const int row = (int)(item / nsd);
    const int q0 = row % w0, t1 = row / w0 - ap;
    const int t0 = mode ? (q0 < ap ? q0 - ap : nt0 + q0 - ap) : q0 - ap;
    fx_item<D, RECON, UCT>(base, g, E, seg * FX_VALID - 3, t0, t1, 0, g.n(D) + 1);
  }
}

// The three directions in ONE launch (launch-bound small blocks): the items of x, then y, then z,
// every pencil of each (mode 0 above); same per-item code, so the stored fluxes are bit-identical
// to three k_flux_xrow launches.
struct FluxAllArgs {
  int nsd[3];          // segments per pencil
  long long first[4];  // first item of direction d; first[3] = all items
};
template <int RECON, bool UCT>
__global__ void __launch_bounds__(FX_THREADS, FX_MINB)
k_flux_all(double* __restrict__ base, Geom g, Eos E, FluxAllArgs fa, int ap) {
  const long long item = (long long)blockIdx.x * (FX_THREADS / 32) + (threadIdx.x >> 5);
  if (item >= fa.first[3]) return;
  const int d = item >= fa.first[2] ? 2 : (item >= fa.first[1] ? 1 : 0);
  const long long it = item - fa.first[d];
  const int nsd = fa.nsd[d];
  const int seg = (int)(it % nsd);
  const int row = (int)(it / nsd);
  const int w0 = (d == 0 ? g.ny : g.nx) + 2 * ap;
  const int t0 = row % w0 - ap, t1 = row / w0 - ap;
  if (d == 0) fx_item<0, RECON, UCT>(base, g, E, seg * FX_VALID - 3, t0, t1, 0, g.nx + 1);
  else if (d == 1) fx_item<1, RECON, UCT>(base, g, E, seg * FX_VALID - 3, t0, t1, 0, g.ny + 1);
  else fx_item<2, RECON, UCT>(base, g, E, seg * FX_VALID - 3, t0, t1, 0, g.nz + 1);
}

}  // namespace gk

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

// Where an item's data live.  FxPadded: the padded [field][z][y][x] arrays of the workspace.
struct FxPadded {
  const double* base;
  long long NPA;
  static constexpr bool compact = false;
  template <int D>
  __device__ __forceinline__ int index(const Geom& g, int cc, int t0, int t1) const {
    return (int)(D == 0 ? g.at(cc, t0, t1) : (D == 1 ? g.at(t0, cc, t1) : g.at(t0, t1, cc)));
  }
  __device__ __forceinline__ double load(int field, int idx) const {
    return base[(size_t)field * NPA + idx];
  }
};

// FxXcol: the COMPACT COPIES of the two x-apron columns x = -1 (side 0) and x = nx (side 1).
// In the padded arrays consecutive cells of such a column are a row pitch apart: one useful
// double per DRAM atom.  k_xcol_gather copies the columns of the XC_NSLOT fields an apron face
// needs into [slot][side][z][y] arrays (y fastest) in one spare field of the workspace -- the 22
// static face-metric fields once per grmhd_set_metric, the 10 dynamic ones once per substep for
// both the y and the z fluxes -- and the apron faces are then computed from contiguous data.
constexpr int XC_NSLOT = 32;
__host__ __device__ constexpr int xc_slot(int field) {
  // P 0-4, B_c 5-7, B~^y 8, B~^z 9, static face metric of y 10-20, of z 21-31
  return field >= F_FM + 2 * NFM ? 21 + (field - F_FM - 2 * NFM)
       : field >= F_FM + NFM     ? 10 + (field - F_FM - NFM)
       : field >= F_BF           ? 8 + (field - F_BF - 1)
       : field >= F_BC           ? 5 + (field - F_BC)
                                 : field - F_P;
}
__host__ __device__ constexpr int xc_field(int slot) {
  return slot < 5 ? F_P + slot : slot < 8 ? F_BC + slot - 5 : slot < 10 ? F_BF + 1 + slot - 8
       : slot < 21 ? F_FM + NFM + slot - 10 : F_FM + 2 * NFM + slot - 21;
}
struct FxXcol {
  const double* xc;  // the spare field
  int PY, PZ;
  static constexpr bool compact = true;
  // pencils of direction y: (t0, t1) = (x, z), lanes along y; of direction z: (x, y), along z
  template <int D>
  __device__ __forceinline__ int index(const Geom& g, int cc, int t0, int t1) const {
    const int side = t0 < 0 ? 0 : 1;
    const int jj = (D == 1 ? cc : t1) + G, kk = (D == 1 ? t1 : cc) + G;
    return (side * PZ + kk) * PY + jj;
  }
  __device__ __forceinline__ double load(int field, int idx) const {
    return xc[(size_t)xc_slot(field) * 2 * PZ * PY + idx];
  }
};

// columns of the slots [s0, s0 + gridDim.z / 2) -> compact; blockIdx.z = 2 (slot - s0) + side
__global__ void k_xcol_gather(double* __restrict__ base, Geom g, long long xc_off, int s0) {
  const int jj = blockIdx.x * blockDim.x + threadIdx.x;
  const int kk = blockIdx.y * blockDim.y + threadIdx.y;
  if (jj >= g.PY || kk >= g.PZ) return;
  const int slot = s0 + (int)(blockIdx.z >> 1), side = (int)(blockIdx.z & 1);
  const int x = side ? g.nx + X0 : X0 - 1;
  const double v = base[(size_t)xc_field(slot) * g.NPA + (long long)kk * g.sz + (long long)jj * g.sy + x];
  base[xc_off + ((size_t)(slot * 2 + side) * g.PZ + kk) * g.PY + jj] = v;
}

// One item: the warp's 32 lanes are the cells c0 .. c0+31 along D of the pencil (t0, t1) -- with
// (t0, t1) the transverse axes: (y, z) for D = x, (x, z) for D = y, (x, y) for D = z -- and the
// lane of cell c solves face c - 1/2.  Faces outside [flo, fhi) are not stored.  Call with whole
// warps.  UCT (compile time): also store the upwind-CT face rows of F_W.
template <int D, int RECON, bool UCT, class AD>
__device__ __forceinline__ void fx_item_at(double* __restrict__ base, const Geom& g, const Eos& E,
                                           const AD& ad, int c0, int t0, int t1, int flo, int fhi) {
  const int lane = threadIdx.x & 31;
  const int nD = g.n(D);
  const int c = c0 + lane;                  // this lane's cell along D; its face is c - 1/2
  const int cc = min(c, nD + G - 1);        // lanes past the last ghost cell reuse it
  const int idx = ad.template index<D>(g, cc, t0, t1);

  // ---- cell data of the lane: rho, v^x, v^y, v^z, p and the two transverse B; the static face
  // metric and the staggered normal field of the lane's face c - 1/2
  double q[FX_NV];
#pragma unroll
  for (int v = 0; v < FX_NV; v++) q[v] = ad.load(flux_var_field(D, v), idx);
  const double bfx = ad.load(F_BF + D, idx);
  double mv11[NFM];
#pragma unroll
  for (int v = 0; v < NFM; v++) mv11[v] = ad.load(F_FM + NFM * D + v, idx);
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
  if constexpr (AD::compact) {
    // x-apron columns: flux-CT (R10) reads there only the row of B~^x -- F~y(B~x) is row 6 of the
    // y fluxes, F~z(B~x) row 5 of the z fluxes (k_update) -- stored at its place in the padded array
    static_assert(D != 0 && !UCT, "compact columns: y / z fluxes with flux-CT");
    if (lane >= 3 && lane < 3 + FX_VALID && c >= flo && c < fhi) {
      const long long pidx = D == 1 ? g.at(t0, cc, t1) : g.at(t0, t1, cc);
      constexpr int row = D == 1 ? 6 : 5;
      fld(base, g, flux_field(D) + row)[pidx] = out[row];
    }
  } else if (lane >= 3 && lane < 3 + FX_VALID && c >= flo && c < fhi) {
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

template <int D, int RECON, bool UCT>
__device__ __forceinline__ void fx_item(double* __restrict__ base, const Geom& g, const Eos& E,
                                        int c0, int t0, int t1, int flo, int fhi) {
  const FxPadded ad = {base, g.NPA};
  fx_item_at<D, RECON, UCT>(base, g, E, ad, c0, t0, t1, flo, fhi);
}

// The 2 x-apron columns of the y or z fluxes (flux-CT) from the compact column copies: one warp
// per (column, t1, segment) item as mode 1 of k_flux_xrow with ap = 1; same per-face code.
template <int D, int RECON>
__global__ void __launch_bounds__(FX_THREADS, FX_MINB)
k_flux_xcol(double* __restrict__ base, Geom g, Eos E, int nsd, long long nitems, long long xc_off) {
  const long long item = (long long)blockIdx.x * (FX_THREADS / 32) + (threadIdx.x >> 5);
  if (item >= nitems) return;  // warp uniform
  const int seg = (int)(item % nsd);
  const int row = (int)(item / nsd);
  const int q0 = row % 2, t1 = row / 2 - 1;
  const int t0 = q0 == 0 ? -1 : g.nx;
  const FxXcol ad = {base + xc_off, g.PY, g.PZ};
  fx_item_at<D, RECON, false>(base, g, E, ad, seg * FX_VALID - 3, t0, t1, 0, g.n(D) + 1);
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

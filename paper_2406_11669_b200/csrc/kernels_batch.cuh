// kernels_batch.cuh -- scalar-state helpers and the stand-alone pointwise batches exposed by
// include/grmhd.h for unit parity tests and the FP64 micro-benchmarks.
#pragma once
#include "kernels_aux.cuh"

namespace gk {

__global__ void k_set_params(DevState* st, double cfl, double fixed_dt, double t_end) {
  st->cfl = cfl; st->fixed_dt = fixed_dt; st->t_end = t_end;
}

// full = 1: new initial data (t, counters); always: clear the max-speed accumulator
__global__ void k_reset_state(DevState* st, int full) {
  for (int d = 0; d < 3; d++) st->ms_acc[d] = 0ull;
  if (full) {
    st->t = 0.0; st->dt = 0.0;
    st->c2p_fail = st->p_fix = st->atmo = st->w_cap = st->c2p_maxiter = st->c2p_backup = 0;
    st->bad_dt = 0;
  }
}

struct BatchPtrs {
  const double* prim[8];  // prim2con: prim in   | con2prim: cons in
  const double* met[10];
  double* cons[8];        // prim2con: cons out  | con2prim: prim out (5)
};

__device__ __forceinline__ Met batch_met(const BatchPtrs& b, long long q) {
  Met M;
  M.a = b.met[0][q]; M.bx = b.met[1][q]; M.by = b.met[2][q]; M.bz = b.met[3][q];
  M.gxx = b.met[4][q]; M.gxy = b.met[5][q]; M.gxz = b.met[6][q];
  M.gyy = b.met[7][q]; M.gyz = b.met[8][q]; M.gzz = b.met[9][q];
  return M;
}

__global__ void k_prim2con_batch(BatchPtrs b, long long n, Eos E) {
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < n;
       q += (long long)gridDim.x * blockDim.x) {
    const Prim P = {b.prim[0][q], b.prim[1][q], b.prim[2][q], b.prim[3][q],
                    b.prim[4][q], b.prim[5][q], b.prim[6][q], b.prim[7][q]};
    double U[5];
    prim2con(P, batch_met(b, q), E, U);
#pragma unroll
    for (int r = 0; r < 5; r++) b.cons[r][q] = U[r];
    b.cons[5][q] = P.Bx; b.cons[6][q] = P.By; b.cons[7][q] = P.Bz;
  }
}

__global__ void __launch_bounds__(128)
k_con2prim_batch(BatchPtrs b, int* __restrict__ status, int* __restrict__ iters, long long n,
                 Eos E) {
  const long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (q >= n) return;
  double U[5] = {b.prim[0][q], b.prim[1][q], b.prim[2][q], b.prim[3][q], b.prim[4][q]};
  double P5[5];
  int it, rw;
  const int bits = con2prim(U, b.prim[5][q], b.prim[6][q], b.prim[7][q], batch_met(b, q), E,
                            false, P5, it, rw);
#pragma unroll
  for (int r = 0; r < 5; r++) b.cons[r][q] = P5[r];
  status[q] = bits;
  iters[q] = it;
}

__global__ void __launch_bounds__(128)
k_con2prim1d_batch(BatchPtrs b, int* __restrict__ status, int* __restrict__ iters, long long n,
                   Eos E) {
  const long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (q >= n) return;
  const double U[5] = {b.prim[0][q], b.prim[1][q], b.prim[2][q], b.prim[3][q], b.prim[4][q]};
  double rho = 0, vx = 0, vy = 0, vz = 0, eps = 0;
  int it = 0;
  const bool ok = con2prim_1d(U, b.prim[5][q], b.prim[6][q], b.prim[7][q], batch_met(b, q), E,
                              rho, vx, vy, vz, eps, it);
  b.cons[0][q] = rho; b.cons[1][q] = vx; b.cons[2][q] = vy; b.cons[3][q] = vz;
  b.cons[4][q] = (E.Gamma - 1.0) * rho * eps;
  status[q] = ok ? 0 : 2;
  iters[q] = it;
}

// FP64 pipe peak: 16 independent DFMA chains per thread, iters rounds.
__global__ void k_dfma_peak(double* __restrict__ out, long long threads, int iters) {
  const long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  double a[16];
#pragma unroll
  for (int r = 0; r < 16; r++) a[r] = 1.0 + 1e-3 * (double)(r + (q & 7));
  const double m = 1.0 - 1e-9, c = 1e-9;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int r = 0; r < 16; r++) a[r] = fma(a[r], m, c);
  }
  double s = 0.0;
#pragma unroll
  for (int r = 0; r < 16; r++) s += a[r];
  if (q < threads) out[q] = s;
}

}  // namespace gk

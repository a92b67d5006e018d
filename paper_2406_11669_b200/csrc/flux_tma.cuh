// flux_tma.cuh -- A3 + A4 along y and z: reconstruction + Riemann flux, marching form, the face
// data fed by TMA.
//
// A block of 128 threads owns 32 pencils of cells running along D (32 consecutive x at one
// position t1 of the other transverse axis: every global access is a full 256-byte row) and a
// segment of faces [f0, f1) along D, which it walks in chunks of TC = 4 faces; face f is the
// face between cells f-1 and f.
//  phase A (reconstruction, R5): warp w owns the variables {2w, 2w+1} of the 7 reconstructed
//    ones, lane = pencil.  The PPM / minmod state of a variable is carried in registers from
//    cell to cell (FtMarch): every slope, interface value and parabola is computed exactly once
//    and every cell value is loaded exactly once, one chunk ahead.  Cell c yields q^-_c (right
//    state of face c) and q^+_c (left state of face c+1); both go to a double-buffered exchange
//    buffer in shared memory.  Warp 3 (one variable) also computes the flattening coefficients
//    of the next chunk.
//  phase B (Riemann, R7): one thread per face reads both states from the exchange buffer and
//    the STATIC face metric (11 values, field family F_FM) plus the staggered normal field from
//    a 2-slot shared-memory ring that thread 0 fills one chunk ahead with cp.async.bulk.tensor
//    (two 4-D boxes [field][.][.][x] of the workspace tensor map per chunk, completion on an
//    mbarrier): no global load is waited for in the loop, and the ring costs no registers.
// One __syncthreads per chunk.  Slot reuse: stage n+1 is issued after the barrier of iteration n,
// i.e. after every thread has finished phase B of chunk n-1, the last reader of that slot.
// The 2 ap apron columns x < 0, x >= nx (ap = 1 flux-CT, R10; 3 upwind CT, G27) are not 32-wide
// groups; they go through k_flux_xrow (flux_xrow.cuh, mode 1), a launch of its own after this
// one.  (Solved at the end of the first and last group's blocks instead -- where their loads hit
// L2 -- they cost more: 0.98 against 0.91 ms, the blocks of those groups finish late.)
#pragma once
#include "flux_face.cuh"
#include "tma.cuh"

namespace gk {

constexpr int FT_THREADS = 128;
constexpr int FT_TC = 4;
#ifndef FT_NSLOTS
#define FT_NSLOTS 3
#endif
constexpr int FT_SLOTS = FT_NSLOTS;
#ifndef FT_MINB
#define FT_MINB 3
#endif
#ifndef FT_UCT_MINB
#define FT_UCT_MINB 3
#endif

struct FtSmem {
  // ring slots (TMA destinations, dense boxes [field][face][pencil])
  alignas(128) double fm[FT_SLOTS][NFM * FT_TC * 32];
  alignas(128) double bf[FT_SLOTS][FT_TC * 32];
  double q[2][FX_NV][2][FT_TC][32];  // [buffer][variable][L/R][face][pencil]
  double fl[2][FT_TC][32];           // flattening coefficient of the chunk's cells
  double fl0[32];                    // ... of the prologue cell f0 - 1
  alignas(8) unsigned long long bar[FT_SLOTS];
};

// RECON: 0 minmod, 1 PPM without flattening, 2 PPM with flattening.  D = 1 (y) or 2 (z).
// grid: x = (groups of 32 along x) * (n_t1 + 2 ap), y = segments of `seglen` faces (a multiple
// of TC).  UCT (compile time, so that the default kernel keeps its register budget): also store
// the upwind-CT face rows of F_W.
template <int D, int RECON, bool UCT>
__global__ void __launch_bounds__(FT_THREADS, UCT ? FT_UCT_MINB : FT_MINB)
k_flux_tma(double* __restrict__ base, Geom g, Eos E, int seglen, int ngx, int ap,
           const __grid_constant__ CUtensorMap tmMet, const __grid_constant__ CUtensorMap tmBf) {
  static_assert(D == 1 || D == 2, "x fluxes: k_flux_xrow");
  constexpr int TC = FT_TC;
  extern __shared__ __align__(128) unsigned char ft_smem_raw[];
  FtSmem& sm = *reinterpret_cast<FtSmem*>(ft_smem_raw);

  const int tid = threadIdx.x, lane = tid & 31;
  // warp index as a warp-uniform value: field offsets that depend on it can live in uniform
  // registers instead of the (scarce) per-thread ones
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int nD = g.n(D);
  const int sd = D == 1 ? (int)g.sy : (int)g.sz;
  const int gx = (int)blockIdx.x % ngx;
  const int t1 = (int)blockIdx.x / ngx - ap;
  const int g0 = gx * 32;
  const int f0 = (int)blockIdx.y * seglen;
  const int f1 = min(f0 + seglen, nD + 1);
  const int cmax = nD + G - 1;  // last valid cell index along D
  const int nchunk = (f1 - f0 + TC - 1) / TC;

  // ---- ring: stage m holds the faces f0 + 4m .. + 3
  constexpr unsigned STAGE_BYTES = (NFM + 1) * TC * 32 * sizeof(double);
  auto issue_stage = [&](int m) {
    const int slot = m % FT_SLOTS;
    const int L = f0 + TC * m;
    const int c0 = g0 + X0;
    const int c1 = D == 1 ? L + G : t1 + G;
    const int c2 = D == 1 ? t1 + G : L + G;
    ft_mbar_expect(&sm.bar[slot], STAGE_BYTES);
    ft_tma_4d(sm.fm[slot], &tmMet, &sm.bar[slot], c0, c1, c2, F_FM + NFM * D);
    ft_tma_4d(sm.bf[slot], &tmBf, &sm.bar[slot], c0, c1, c2, F_BF + D);
  };
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < FT_SLOTS; s++) ft_mbar_init(&sm.bar[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
#pragma unroll
    for (int m = 0; m < FT_SLOTS; m++)
      if (m < nchunk) issue_stage(m);
  }

  // ---- phase-A identity: lane = pencil
  const int pA = min(g0 + lane, g.nx - 1);
  const int baseA = (int)(D == 1 ? g.at(pA, 0, t1) : g.at(pA, t1, 0));
  // variables of the warp (slots of flux_var_field): {rho, v^x}, {v^y, v^z}, the two transverse
  // B, and warp 3 the pressure alone -- with the pressure window of its own march in registers
  // it also forms the flattening coefficients (G8c) of the NEXT chunk's cells
  const int sA = warp == 0 ? 0 : (warp == 1 ? 2 : (warp == 2 ? 5 : 4));
  const int nslot = warp == 3 ? 1 : 2;
  const double* qsrc[2];
  qsrc[0] = fld(base, g, flux_var_field(D, sA)) + baseA;
  qsrc[1] = fld(base, g, flux_var_field(D, sA + (nslot > 1 ? 1 : 0))) + baseA;
  const double* vsrc = fld(base, g, F_P + 1 + D) + baseA;  // warp 3: normal velocity

  // new cells of the chunk whose first face is F: cells F+2 .. F+5
  auto load_cells = [&](const double* q, int F, double out[TC]) {
#pragma unroll
    for (int cl = 0; cl < TC; cl++) out[cl] = q[min(F + cl + 2, cmax) * sd];
  };

  FtMarch<RECON> mv[2];
  double vm1 = 0.0, v0 = 0.0;  // warp 3: v_{c-1}, v_c behind the next cell to be flattened
  double nxt[2][TC];           // cells of the next chunk (prefetched)
  // ---- prologue: state before cell f0-1, flattening of f0-1 and of chunk 0
#pragma unroll
  for (int s = 0; s < 2; s++) {
    if (s < nslot) {
      const double* q = qsrc[s];
      mv[s].init(q[(f0 - 3) * sd], q[(f0 - 2) * sd], q[(f0 - 1) * sd], q[f0 * sd]);
    }
  }
  if (RECON == 2 && warp == 3) {
    const double* ps = qsrc[0];
    double pw[TC + 5], vw[TC + 3];  // p_{f0-3 .. f0+5}, v_{f0-2 .. f0+4}
#pragma unroll
    for (int m = 0; m < TC + 5; m++) pw[m] = ps[min(f0 - 3 + m, cmax) * sd];
#pragma unroll
    for (int m = 0; m < TC + 3; m++) vw[m] = vsrc[min(f0 - 2 + m, cmax) * sd];
    sm.fl0[lane] = ft_flatten(pw[0], pw[1], pw[3], pw[4], vw[0], vw[2]);  // cell f0 - 1
#pragma unroll
    for (int cl = 0; cl < TC; cl++)  // cell f0 + cl
      sm.fl[0][cl][lane] = ft_flatten(pw[cl + 1], pw[cl + 2], pw[cl + 4], pw[cl + 5], vw[cl + 1],
                                      vw[cl + 3]);
    vm1 = vw[TC + 1]; v0 = vw[TC + 2];  // v_{f0+3}, v_{f0+4}
  }
  __syncthreads();  // barrier init + fl0 / fl[0] visible
  {
    const bool anyf = RECON == 2 && __any_sync(0xffffffffu, sm.fl0[lane] != 0.0);
#pragma unroll
    for (int s = 0; s < 2; s++) {
      if (s < nslot) {
        double qm, qp;
        mv[s].step(qsrc[s][min(f0 + 1, cmax) * sd], RECON == 2 ? sm.fl0[lane] : 0.0, anyf, qm, qp);
        mv[s].qpp = qp;
        load_cells(qsrc[s], f0, nxt[s]);
      }
    }
  }

  // ---- phase-B identity: warp = face of the chunk, lane = pencil
  const int plB = lane, clB = warp;
  const bool okB = g0 + plB < g.nx;
  const long long ublk = D == 1 ? g.at(g0, 0, t1) : g.at(g0, t1, 0);
  double* const outb = fld(base, g, flux_field(D)) + ublk;
  const size_t NPA = (size_t)g.NPA;
  const int ringo = clB * 32 + plB;  // offset of the thread's face inside a field of a slot
  constexpr int MF = TC * 32;        // doubles per field in a slot

  int buf = 0;
  for (int n = 0; n < nchunk; n++, buf ^= 1) {
    const int F = f0 + n * TC;
    // ================= phase A: cells F .. F+TC-1 =================
    double cur[2][TC];
#pragma unroll
    for (int s = 0; s < 2; s++)
#pragma unroll
      for (int cl = 0; cl < TC; cl++) cur[s][cl] = nxt[s][cl];
    const bool more = n + 1 < nchunk;
#pragma unroll
    for (int s = 0; s < 2; s++)
      if (s < nslot && more) load_cells(qsrc[s], F + TC, nxt[s]);
    // warp 3: v_{F+5 .. F+8}, the only inputs of the next chunk's flattening that its own march
    // does not hold (in flight while the pressure is reconstructed)
    double vc[TC];
    if (RECON == 2 && warp == 3 && more) {
#pragma unroll
      for (int cl = 0; cl < TC; cl++) vc[cl] = vsrc[min(F + TC + cl + 1, cmax) * sd];
    }
#pragma unroll
    for (int s = 0; s < 2; s++) {
      if (s < nslot) {
        const int slot = sA + s;
#pragma unroll
        for (int cl = 0; cl < TC; cl++) {
          const double f = RECON == 2 ? sm.fl[buf][cl][lane] : 0.0;
          const bool anyf = RECON == 2 && __any_sync(0xffffffffu, f != 0.0);
          double qm, qp;
          mv[s].step(cur[s][cl], f, anyf, qm, qp);
          sm.q[buf][slot][0][cl][lane] = mv[s].qpp;  // left state of face F+cl
          sm.q[buf][slot][1][cl][lane] = qm;         // right state of face F+cl
          mv[s].qpp = qp;
        }
      }
    }
    if (RECON == 2 && warp == 3 && more) {
      // cells c' = F+TC+cl: p_{c'-2 .. c'+2} = p_{F+2 .. F+9} are cur[0] and nxt[0]
      double pw[2 * TC];
#pragma unroll
      for (int m = 0; m < TC; m++) { pw[m] = cur[0][m]; pw[TC + m] = nxt[0][m]; }
      const double vw[TC + 2] = {vm1, v0, vc[0], vc[1], vc[2], vc[3]};  // v_{F+3 .. F+8}
#pragma unroll
      for (int cl = 0; cl < TC; cl++)
        sm.fl[buf ^ 1][cl][lane] =
            ft_flatten(pw[cl], pw[cl + 1], pw[cl + 3], pw[cl + 4], vw[cl], vw[cl + 2]);
      vm1 = vc[2]; v0 = vc[3];
    }
    __syncthreads();  // A(n) and B(n-1) are complete in every warp
    if (tid == 0 && n >= 1 && n + FT_SLOTS - 1 < nchunk) issue_stage(n + FT_SLOTS - 1);  // slot of stage n-1
    // ================= phase B: faces F .. F+TC-1 =================
    {
      const int slot = n % FT_SLOTS;
      ft_mbar_wait(&sm.bar[slot], (unsigned)((n / FT_SLOTS) & 1));
      double mv11[NFM];
#pragma unroll
      for (int v = 0; v < NFM; v++) mv11[v] = sm.fm[slot][v * MF + ringo];
      const FaceMet fmet = face_met<D>(mv11);
      const double bfn = sm.bf[slot][ringo];
      double qL[FX_NV], qR[FX_NV];
#pragma unroll
      for (int v = 0; v < FX_NV; v++) {
        qL[v] = sm.q[buf][v][0][clB][plB];
        qR[v] = sm.q[buf][v][1][clB][plB];
      }
      double out[7], w[4];
      ft_face<D, UCT>(qL, qR, bfn, fmet, E, out, w);
      const int f = F + clB;
      if (okB && f < f1) {
        double* o = outb + plB + f * sd;
#pragma unroll
        for (int r = 0; r < 7; r++) o[r * NPA] = out[r];
        if (UCT) {
          double* ow = o + (size_t)(F_W + 4 * D - flux_field(D)) * NPA;
#pragma unroll
          for (int r = 0; r < 4; r++) ow[r * NPA] = w[r];
        }
      }
    }
    // no barrier here: the next phase A writes the other exchange buffer
  }
}

}  // namespace gk

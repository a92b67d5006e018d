// grmhd.cu -- C ABI of libgrmhd.so (include/grmhd.h): host-side step driver that only
// enqueues kernels on the handle's stream; every numerical step runs in the CUDA kernels of
// kernels_*.cuh.  There is no CPU fallback: without a CUDA device every compute call
// returns GRMHD_ECUDA.
#include "../../include/grmhd.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "kernels_flux.cuh"
#include "flux_tma.cuh"
#include "flux_xrow.cuh"
#include "flux_xflat.cuh"
#include "src_tile.cuh"
#include "emf_uct.cuh"
#include "kernels_batch.cuh"

using namespace gk;

struct grmhd {
  Geom g;
  Eos E;
  grmhd_opts o;
  double* base = nullptr;
  double* stage = nullptr;
  unsigned char* mask = nullptr;
  DevState* dst = nullptr;
  cudaStream_t s = nullptr;
  int nfields = 0;
  long long stage_elems = 0;
  bool have_metric = false, have_prims = false, have_mask = false;
  bool dirty = false;  // set_prims / set_vecpot changed the inputs: (B, U~, sources, max speed)
                       // are rebuilt once, by the next call that needs them
  double cfl_set = -1.0, fixed_dt = 0.0, fixed_set = -1.0, tend_set = -2.0;
  long long steps = 0;
  long long launches = 0;
  int ft_conc[18] = {0};  // resident blocks of each k_flux_tma instantiation (0 = not queried)
  CUtensorMap tm_met[3], tm_bf[3];  // 4-D boxes [field][.][.][x] of the ring stages (y, z)
  CUtensorMap tm_src;               // [10 fields][1][12][36] tile of k_src_tile
  int src_impl = 1;                 // 1: k_src_tile (TMA-staged x-y stencils), 0: k_src
  bool tma_ok = false;
  int uct_nseg = 16;     // segments of the marching passes along y and z
  int uct_passes = 1;    // upwind CT: per-axis passes (1) or the per-edge kernel k_emf_uct (0)
  int nsm = 148;         // multiprocessors of the device (queried at create)
  int xcol = 1;          // 1: x-apron columns of the y/z fluxes from compact column copies
  int small_fuse = 1;    // 1: launch-bound blocks (<= SMALL_BLOCK_MAX padded cells) take the fused launches
  int flux_impl = 1;     // 1: y and z fluxes by k_flux_tma (blocks at least 32 cells wide in x),
                         // 0: k_flux_xrow (lanes along the flux direction) everywhere
  // CUDA graph of one RK step (launch-bound small blocks): the first step after a change of
  // options or mask runs eagerly (lazy attribute / occupancy queries happen there), the second
  // is captured on cap_s, later ones are one cudaGraphLaunch into the caller's stream.
  int use_graph = 1;
  int gstate = 0;        // 0 nothing run yet, 1 eager step done, 2 graph ready, 3 capture failed
  cudaStream_t cap_s = nullptr;
  cudaGraphExec_t gexec = nullptr;
  long long glaunches = 0;  // kernels per graph launch
  char err[256] = {0};
  // optional per-kernel-group timing ("kernel_timing" option): CUDA events on the stream
  bool ktime = false;
  std::vector<cudaEvent_t> ev;     // pool, used pairwise
  std::vector<int> ev_grp;         // group of each recorded pair
  size_t ev_used = 0;
  double kms[GRMHD_NKGROUPS] = {0};
  long long kcnt[GRMHD_NKGROUPS] = {0};
};

namespace {

int fail(grmhd* h, int code, const char* msg) {
  if (h) snprintf(h->err, sizeof h->err, "%s", msg);
  return code;
}

int cuda_fail(grmhd* h, cudaError_t e, const char* where) {
  if (h) snprintf(h->err, sizeof h->err, "%s: %s", where, cudaGetErrorString(e));
  return GRMHD_ECUDA;
}

#define CK(call)                                                     \
  do {                                                               \
    cudaError_t e_ = (call);                                         \
    if (e_ != cudaSuccess) return cuda_fail(h, e_, #call);           \
  } while (0)

#define CKL(name)                                                    \
  do {                                                               \
    h->launches++;                                                   \
    cudaError_t e_ = cudaGetLastError();                             \
    if (e_ != cudaSuccess) return cuda_fail(h, e_, name);            \
  } while (0)

// ---- kernel-group timing -------------------------------------------------------------
enum { KG_FLUX_X = 0, KG_FLUX_Y, KG_FLUX_Z, KG_UPDATE, KG_BFIELD, KG_C2P, KG_GHOST, KG_MISC, KG_SRC };

int kt_flush(grmhd* h) {
  if (h->ev_used == 0) return GRMHD_OK;
  CK(cudaStreamSynchronize(h->s));
  for (size_t q = 0; q < h->ev_used; q += 2) {
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, h->ev[q], h->ev[q + 1]));
    h->kms[h->ev_grp[q / 2]] += ms;
    h->kcnt[h->ev_grp[q / 2]]++;
  }
  h->ev_used = 0;
  return GRMHD_OK;
}

int kt_begin(grmhd* h, int grp) {
  if (!h->ktime) return GRMHD_OK;
  if (h->ev_used + 2 > h->ev.size()) {
    int rc = kt_flush(h);
    if (rc) return rc;
  }
  h->ev_grp[h->ev_used / 2] = grp;
  CK(cudaEventRecord(h->ev[h->ev_used], h->s));
  return GRMHD_OK;
}

int kt_end(grmhd* h) {
  if (!h->ktime) return GRMHD_OK;
  CK(cudaEventRecord(h->ev[h->ev_used + 1], h->s));
  h->ev_used += 2;
  return GRMHD_OK;
}

#define KT(grp, ...)                               \
  do {                                             \
    int rc_ = kt_begin(h, grp);                    \
    if (rc_) return rc_;                           \
    __VA_ARGS__;                                   \
    rc_ = kt_end(h);                               \
    if (rc_) return rc_;                           \
  } while (0)

bool valid_opts(const grmhd_opts* o) {
  if (!o) return false;
  for (int a = 0; a < 3; a++)
    if (o->bc[a] != 0 && o->bc[a] != 1) return false;
  return o->rk >= 2 && o->rk <= 4 && o->recon >= 0 && o->recon <= 1 && o->gamma_ad > 1.0 &&
         o->p_floor > 0 && o->rho_atm > 0 && o->w_max > 1.0 && o->c2p_maxit >= 1 &&
         o->c2p_tol > 0 && o->poly_k >= 0 && o->poly_gamma > 0 &&
         o->riemann >= 0 && o->riemann <= 1;
}

Eos make_eos(const grmhd_opts& o) {
  Eos E;
  E.Gamma = o.gamma_ad;
  E.GoGm1 = o.gamma_ad / (o.gamma_ad - 1.0);
  E.gm1oG = (o.gamma_ad - 1.0) / o.gamma_ad;
  E.rho_atm = o.rho_atm;
  E.p_atm = std::fmax(o.poly_k * std::pow(o.rho_atm, o.poly_gamma), o.p_floor);
  E.p_floor = o.p_floor;
  E.v2max = 1.0 - 1.0 / (o.w_max * o.w_max);
  E.c2p_tol = o.c2p_tol;
  E.c2p_maxit = o.c2p_maxit;
  E.recon = o.recon;
  E.flatten = o.ppm_flatten;
  E.riemann = o.riemann;
  E.c2p_backup = 0;
  E.emf = 0;
  E.gauge = 0;
  E.lorenz_xi = 1.5;
  return E;
}

bool make_geom(int nx, int ny, int nz, const double dx[3], const grmhd_opts* o, Geom* g) {
  if (nx < 1 || ny < 1 || nz < 1) return false;
  g->nx = nx; g->ny = ny; g->nz = nz;
  g->PXP = ((nx + 8 + 3) / 4) * 4;
  g->PY = ny + 2 * G + 1;
  g->PZ = nz + 2 * G + 1;
  g->sy = g->PXP;
  g->sz = (long long)g->PXP * g->PY;
  g->NP = g->sz * g->PZ;
  g->NPA = ((g->NP + 31) / 32) * 32;
  for (int a = 0; a < 3; a++) {
    g->dx[a] = dx ? dx[a] : 1.0;
    g->idx[a] = 1.0 / g->dx[a];
    g->bc[a] = o ? o->bc[a] : 0;
  }
  return true;
}

long long stage_elems_of(const Geom& g) {
  const long long n = (long long)(g.nx + 2 * G + 1) * (g.ny + 2 * G + 1) * (g.nz + 2 * G + 1);
  return ((n + 31) / 32) * 32;
}

// the fields of layout.cuh + one spare field: the compact x-apron columns (FxXcol, flux_xrow.cuh)
int nfields_of(const grmhd_opts* o) { return (o->rk == 4 ? F_END_RK4 : F_END_RK23) + 1; }

bool is_device_ptr(const void* p) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

// set_* calls stage host sources through cudaMemcpyAsync: wait for the copies before
// returning, so that the caller may reuse or free its host arrays at once (device sources stay
// asynchronous on the handle's stream)
int sync_if_host(grmhd* h, const void* p) {
  if (p && !is_device_ptr(p)) CK(cudaStreamSynchronize(h->s));
  return GRMHD_OK;
}

dim3 blk3() { return dim3(32, 4, 1); }
dim3 grd3(int ex, int ey, int ez) { return dim3((ex + 31) / 32, (ey + 3) / 4, ez); }
dim3 grd_post(const Geom& g) {
  return dim3((g.nx + 2 * G + 1 + 31) / 32, (g.ny + 2 * G + 1 + KP_BY - 1) / KP_BY,
              (g.nz + 2 * G + 1 + KP_BZ - 1) / KP_BZ);
}
dim3 grd_src(const Geom& g) {
  return dim3((g.nx + KS_BX - 1) / KS_BX, (g.ny + KS_BY - 1) / KS_BY, g.nz);
}
int grd1(long long n) {
  long long b = (n + 255) / 256;
  return (int)(b > 65535 * 16 ? 65535 * 16 : (b < 1 ? 1 : b));
}

// external array -> internal field (through the staging buffer when the source is host memory)
int copy_in(grmhd* h, const double* src, int id, bool stag) {
  const Geom& g = h->g;
  const int ex = g.nx + 2 * G + stag, ey = g.ny + 2 * G + stag, ez = g.nz + 2 * G + stag;
  const long long n = (long long)ex * ey * ez;
  const double* dsrc = src;
  if (!is_device_ptr(src)) {
    CK(cudaMemcpyAsync(h->stage, src, n * sizeof(double), cudaMemcpyDefault, h->s));
    dsrc = h->stage;
  }
  k_repack_in<<<grd1(n), 256, 0, h->s>>>(dsrc, h->base + (size_t)id * g.NPA, g, ex, ey, ez);
  CKL("k_repack_in");
  return GRMHD_OK;
}

int copy_out(grmhd* h, int id, double* dst, bool stag, int mode) {
  const Geom& g = h->g;
  const int ex = g.nx + 2 * G + stag, ey = g.ny + 2 * G + stag, ez = g.nz + 2 * G + stag;
  const long long n = (long long)ex * ey * ez;
  const bool dev = is_device_ptr(dst);
  double* ddst = dev ? dst : h->stage;
  k_repack_out<<<grd1(n), 256, 0, h->s>>>(h->base + (size_t)id * g.NPA, ddst, h->base, g, ex,
                                          ey, ez, mode);
  CKL("k_repack_out");
  if (!dev) CK(cudaMemcpyAsync(dst, h->stage, n * sizeof(double), cudaMemcpyDefault, h->s));
  return GRMHD_OK;
}

int zero_field(grmhd* h, int id) {
  k_fill_zero<<<grd1(h->g.NPA), 256, 0, h->s>>>(h->base + (size_t)id * h->g.NPA, h->g.NPA);
  CKL("k_fill_zero");
  return GRMHD_OK;
}

// R15: x, then y, then z pass
constexpr long long SMALL_BLOCK_MAX = 1LL << 16;  // padded cells: below, a step is launch bound
constexpr long long FILL_FUSE_MAX = 1LL << 20;  // padded cells: below, launches cost more than threads

int fill_ghosts(grmhd* h, const FillArgs& fa) {
  const Geom& g = h->g;
  bool plain = true;  // unstaggered copy / wrap fields only
  for (int f = 0; f < fa.nf; f++) plain = plain && fa.stag[f] == 0 && fa.kind[f] == 0;
  const long long npad = (long long)(g.nx + 2 * G) * (g.ny + 2 * G) * (g.nz + 2 * G);
  if (plain && npad <= FILL_FUSE_MAX) {
    k_fill_copy3<<<dim3((unsigned)((npad + 255) / 256), 1, fa.nf), 256, 0, h->s>>>(h->base, g, fa);
    CKL("k_fill_copy3");
    return GRMHD_OK;
  }
  if (h->small_fuse && npad <= SMALL_BLOCK_MAX) {  // staggered / extrapolated fields, small block:
    cudaLaunchConfig_t cfg = {};                    // the three passes by one cluster
    cfg.gridDim = dim3(FILL1_CTAS);
    cfg.blockDim = dim3(FILL1_THREADS);
    cfg.stream = h->s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = FILL1_CTAS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    CK(cudaLaunchKernelEx(&cfg, k_fill_axes1, h->base, g, fa));
    h->launches++;
    return GRMHD_OK;
  }
  for (int a = 0; a < 3; a++) {
    const int b0 = (a + 1) % 3, b1 = (a + 2) % 3;
    const long long nt = (long long)(g.n(b0) + 2 * G + 1) * (g.n(b1) + 2 * G + 1);
    dim3 grid((unsigned)((nt + 127) / 128), 1, fa.nf);
    k_fill_axis<<<grid, 128, 0, h->s>>>(h->base, g, fa, a);
    CKL("k_fill_axis");
  }
  return GRMHD_OK;
}

FillArgs fill_prims() {
  FillArgs fa{};
  fa.nf = 5;
  for (int r = 0; r < 5; r++) { fa.id[r] = F_P + r; fa.stag[r] = 0; fa.kind[r] = 0; }
  return fa;
}
FillArgs fill_vecpot(bool with_psi = false) {
  FillArgs fa{};
  fa.nf = 3;
  const int st[3] = {2 | 4, 1 | 4, 1 | 2};  // A_x on (y,z)-staggered edges, ...
  for (int d = 0; d < 3; d++) { fa.id[d] = F_Y + 5 + d; fa.stag[d] = st[d]; fa.kind[d] = 1; }
  if (with_psi) {  // Psi_mhd on the vertices: wrap / copy (G29)
    fa.id[3] = F_Y + 8; fa.stag[3] = 1 | 2 | 4; fa.kind[3] = 0;
    fa.nf = 4;
  }
  return fa;
}

int set_params(grmhd* h, double cfl, double t_end) {
  if (cfl != h->cfl_set || h->fixed_dt != h->fixed_set || t_end != h->tend_set) {
    k_set_params<<<1, 1, 0, h->s>>>(h->dst, cfl, h->fixed_dt, t_end);
    CKL("k_set_params");
    h->cfl_set = cfl; h->fixed_set = h->fixed_dt; h->tend_set = t_end;
  }
  return GRMHD_OK;
}

int launch_src(grmhd* h);

// launch-bound blocks take fused launches: k_flux_all, k_fill_axes1, k_post with sources and t += dt
bool small_block(const grmhd* h) {
  const Geom& g = h->g;
  return h->small_fuse &&
         (long long)(g.nx + 2 * G) * (g.ny + 2 * G) * (g.nz + 2 * G) <= SMALL_BLOCK_MAX;
}

// R13 + R14 + R15 after a change of (U~, A)
int after_stage(grmhd* h, bool want_speed) {
  const Geom& g = h->g;
  int rc;
  KT(KG_BFIELD, {
    rc = fill_ghosts(h, fill_vecpot(h->E.gauge != 0));
    if (rc) return rc;
  });
  const bool small = small_block(h);
  // small blocks: the sources and the end-of-step t += dt ride in k_post (two launches fewer)
  const int flags = (want_speed ? 1 : 0) | (small && want_speed ? 2 : 0);
  const unsigned char* mk = h->have_mask ? h->mask : nullptr;
  KT(KG_C2P, {
    const dim3 pg = grd_post(g), pb(32, KP_BY, KP_BZ);
    if (small && h->E.c2p_backup)
      k_post<false, true, true><<<pg, pb, 0, h->s>>>(h->base, mk, g, h->E, h->dst, flags);
    else if (small)
      k_post<false, false, true><<<pg, pb, 0, h->s>>>(h->base, mk, g, h->E, h->dst, flags);
    else if (h->E.c2p_backup)
      k_post<false, true><<<pg, pb, 0, h->s>>>(h->base, mk, g, h->E, h->dst, flags);
    else
      k_post<false, false><<<pg, pb, 0, h->s>>>(h->base, mk, g, h->E, h->dst, flags);
    CKL("k_post");
  });
  if (!small) {
    KT(KG_SRC, {
      rc = launch_src(h);
      if (rc) return rc;
    });
  }
  KT(KG_GHOST, {
    rc = fill_ghosts(h, fill_prims());
    if (rc) return rc;
  });
  return GRMHD_OK;
}

// lanes along D (flux_xrow.cuh): one warp per 27 faces of a pencil.  mode 0: every pencil
// (the x fluxes; any direction of a narrow block when the upwind CT is on); mode 1: the
// apron columns k_flux_tma leaves out.
int apron_width(const grmhd* h) { return h->E.emf ? 3 : 1; }  // G27: PPM face -> edge stencils

template <int D, int RECON>
int launch_flux_xrow(grmhd* h, int mode, cudaStream_t st) {
  const Geom& g = h->g;
  const int ap = apron_width(h);
  const int nsd = (g.n(D) + 1 + FX_VALID - 1) / FX_VALID;
  const int nt0 = D == 0 ? g.ny : g.nx, nt1 = D == 2 ? g.ny : g.nz;
  const long long npen = (long long)(mode ? 2 * ap : nt0 + 2 * ap) * (nt1 + 2 * ap);
  const long long nitems = npen * nsd;
  const long long nblk = (nitems + FX_THREADS / 32 - 1) / (FX_THREADS / 32);
  if (h->E.emf)
    k_flux_xrow<D, RECON, true><<<(unsigned)nblk, FX_THREADS, 0, st>>>(h->base, g, h->E, nsd,
                                                                      nitems, ap, mode);
  else
    k_flux_xrow<D, RECON, false><<<(unsigned)nblk, FX_THREADS, 0, st>>>(h->base, g, h->E, nsd,
                                                                       nitems, ap, mode);
  h->launches++;
  return GRMHD_OK;
}

// ---- TMA-fed flux kernel (flux_tma.cuh) ---------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// tensor = the whole workspace as [field][z][y][x]; box of direction D with nf fields
bool make_tensor_maps(grmhd* h) {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) !=
          cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) {
    cudaGetLastError();
    return false;
  }
  const Geom& g = h->g;
  const cuuint64_t dims[4] = {(cuuint64_t)g.PXP, (cuuint64_t)g.PY, (cuuint64_t)g.PZ,
                              (cuuint64_t)h->nfields};
  const cuuint64_t strides[3] = {(cuuint64_t)g.sy * 8, (cuuint64_t)g.sz * 8,
                                 (cuuint64_t)g.NPA * 8};
  const cuuint32_t es[4] = {1, 1, 1, 1};
  for (int d = 1; d < 3; d++) {
    for (int w = 0; w < 2; w++) {
      cuuint32_t box[4] = {32, 1, 1, (cuuint32_t)(w == 0 ? NFM : 1)};
      box[d] = FT_TC;
      CUresult r = ((EncodeTiledFn)fn)(w == 0 ? &h->tm_met[d] : &h->tm_bf[d],
                                       CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, h->base, dims, strides,
                                       box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                       CU_TENSOR_MAP_SWIZZLE_NONE,
                                       CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                       CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
      if (r != CUDA_SUCCESS) return false;
    }
  }
  {
    const cuuint32_t box[4] = {ST_TX, ST_TY, 1, ST_NF};
    CUresult r = ((EncodeTiledFn)fn)(&h->tm_src, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, h->base, dims,
                                     strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                     CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return false;
  }
  return true;
}

// A5 sources of the current primitives into F_SRC
int launch_src(grmhd* h) {
  const Geom& g = h->g;
  if (h->src_impl == 1 && h->tma_ok) {
    const dim3 grid((g.nx + ST_BX - 1) / ST_BX, (g.ny + ST_BY - 1) / ST_BY, g.nz);
    k_src_tile<<<grid, dim3(ST_BX, ST_BY, 1), sizeof(SrcTileSmem), h->s>>>(h->base, g, h->E,
                                                                            h->tm_src);
    CKL("k_src_tile");
  } else {
    k_src<<<grd_src(g), dim3(KS_BX, KS_BY, 1), 0, h->s>>>(h->base, g, h->E);
    CKL("k_src");
  }
  return GRMHD_OK;
}

// ---- compact x-apron columns (FxXcol, flux_xrow.cuh) ----------------------------------------
long long xc_offset(const grmhd* h) { return (long long)(h->nfields - 1) * h->g.NPA; }
// usable when the TMA-fed kernels serve y and z (so the aprons are a launch of their own), with
// flux-CT (one apron column per side, one flux row needed), and the 32 column pairs fit the field
bool xcol_ok(const grmhd* h) {
  const Geom& g = h->g;
  return h->xcol && h->flux_impl == 1 && h->tma_ok && g.nx >= 32 &&
         (long long)XC_NSLOT * 2 * g.PY * g.PZ <= g.NPA;
}
int xcol_gather(grmhd* h, int s0, int ns) {
  const Geom& g = h->g;
  k_xcol_gather<<<dim3((g.PY + 31) / 32, (g.PZ + 3) / 4, 2 * ns), dim3(32, 4, 1), 0, h->s>>>(
      h->base, g, xc_offset(h), s0);
  CKL("k_xcol_gather");
  return GRMHD_OK;
}
template <int D, int RECON>
int launch_flux_xcol(grmhd* h) {
  const Geom& g = h->g;
  const int nsd = (g.n(D) + 1 + FX_VALID - 1) / FX_VALID;
  const int nt1 = D == 2 ? g.ny : g.nz;
  const long long nitems = 2LL * (nt1 + 2) * nsd;
  k_flux_xcol<D, RECON><<<(unsigned)((nitems + FX_THREADS / 32 - 1) / (FX_THREADS / 32)),
                          FX_THREADS, 0, h->s>>>(h->base, g, h->E, nsd, nitems, xc_offset(h));
  CKL("k_flux_xcol");
  return GRMHD_OK;
}

template <int D, int RECON, bool UCT>
int launch_flux_tma_v(grmhd* h) {
  const Geom& g = h->g;
  auto kern = k_flux_tma<D, RECON, UCT>;
  const int smem = (int)sizeof(FtSmem);
  const int cfg = (UCT ? 9 : 0) + D * 3 + RECON;
  if (h->ft_conc[cfg] == 0) {
    CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    int nb = 0, dev = 0, nsm = 0;
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, FT_THREADS, smem));
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    h->ft_conc[cfg] = nb * nsm > 0 ? nb * nsm : 1;
  }
  const int nt1 = D == 2 ? g.ny : g.nz;
  const int ngx = (g.nx + 31) / 32;
  const int ap = apron_width(h);
  const long long ngroups = (long long)ngx * (nt1 + 2 * ap);
  const int nfaces = g.n(D) + 1;
  int best = 1;
  double best_cost = 1e300;
  for (int ns = 1; ns <= 64; ns++) {
    const int sl = ((nfaces + ns - 1) / ns + FT_TC - 1) / FT_TC * FT_TC;
    if (ns > 1 && sl < 16) break;
    const int nseg = (nfaces + sl - 1) / sl;
    const long long nblk = (long long)nseg * ngroups;
    const long long waves = (nblk + h->ft_conc[cfg] - 1) / h->ft_conc[cfg];
    const double cost = (double)waves * (sl + 3);
    if (cost < best_cost * 0.97) { best_cost = cost; best = ns; }
  }
  const int seglen = ((nfaces + best - 1) / best + FT_TC - 1) / FT_TC * FT_TC;
  const int nseg = (nfaces + seglen - 1) / seglen;
  kern<<<dim3((unsigned)ngroups, nseg), FT_THREADS, smem, h->s>>>(h->base, g, h->E, seglen, ngx,
                                                                  ap, h->tm_met[D], h->tm_bf[D]);
  h->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(h, e, "k_flux_tma");
  // the 2 ap apron columns along x.  (Run beside the main kernel on a second stream they cost
  // MORE, measured 0.93 against 0.89 ms: their blocks take register space the main kernel's
  // third block per SM needs.)
  if constexpr (!UCT) {
    // ... unless the columns have compact copies (gathered once per substep in compute_fluxes):
    // contiguous loads, and only the one row flux-CT reads there is stored
    if (xcol_ok(h)) return launch_flux_xcol<D, RECON>(h);
  }
  return launch_flux_xrow<D, RECON>(h, 1, h->s);
}

template <int D, int RECON>
int launch_flux_tma(grmhd* h) {
  return h->E.emf ? launch_flux_tma_v<D, RECON, true>(h) : launch_flux_tma_v<D, RECON, false>(h);
}

// x fluxes: blocks of 128 consecutive array positions swept in memory order (flux_xflat.cuh)
template <int RECON>
int launch_flux_xflat(grmhd* h) {
  const Geom& g = h->g;
  const int ap = apron_width(h);
  const long long ipp = xf_items_per_plane(g, ap);
  const long long nblk = ipp * (g.nz + 2 * ap);
  if (h->E.emf)
    k_flux_xflat<RECON, true><<<(unsigned)nblk, XF_THREADS, 0, h->s>>>(h->base, g, h->E, ap, (int)ipp);
  else
    k_flux_xflat<RECON, false><<<(unsigned)nblk, XF_THREADS, 0, h->s>>>(h->base, g, h->E, ap, (int)ipp);
  h->launches++;
  return GRMHD_OK;
}

template <int D, int RECON>
int launch_flux_dr(grmhd* h) {
  if (D == 0 && h->flux_impl == 1) return launch_flux_xflat<RECON>(h);
  if (D != 0 && h->flux_impl == 1 && h->tma_ok && h->g.nx >= 32) {
    if constexpr (D != 0) return launch_flux_tma<D, RECON>(h);
  }
  return launch_flux_xrow<D, RECON>(h, 0, h->s);
}

template <int D>
int launch_flux_d(grmhd* h) {
  const int recon = h->o.recon == 0 ? 0 : (h->o.ppm_flatten ? 2 : 1);
  const int rc = recon == 0 ? launch_flux_dr<D, 0>(h)
                            : (recon == 1 ? launch_flux_dr<D, 1>(h) : launch_flux_dr<D, 2>(h));
  if (rc) return rc;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(h, e, "flux kernel");
  return GRMHD_OK;
}

// launch-bound small blocks: x, y and z in one launch (k_flux_all, lanes along the flux direction)
template <int RECON>
int launch_flux_all(grmhd* h) {
  const Geom& g = h->g;
  const int ap = apron_width(h);
  FluxAllArgs fa;
  fa.first[0] = 0;
  for (int d = 0; d < 3; d++) {
    fa.nsd[d] = (g.n(d) + 1 + FX_VALID - 1) / FX_VALID;
    const int nt0 = d == 0 ? g.ny : g.nx, nt1 = d == 2 ? g.ny : g.nz;
    fa.first[d + 1] = fa.first[d] + (long long)(nt0 + 2 * ap) * (nt1 + 2 * ap) * fa.nsd[d];
  }
  const long long nblk = (fa.first[3] + FX_THREADS / 32 - 1) / (FX_THREADS / 32);
  if (h->E.emf)
    k_flux_all<RECON, true><<<(unsigned)nblk, FX_THREADS, 0, h->s>>>(h->base, g, h->E, fa, ap);
  else
    k_flux_all<RECON, false><<<(unsigned)nblk, FX_THREADS, 0, h->s>>>(h->base, g, h->E, fa, ap);
  CKL("k_flux_all");
  return GRMHD_OK;
}

int compute_fluxes(grmhd* h) {
  int rc;
  if (small_block(h)) {
    const int recon = h->o.recon == 0 ? 0 : (h->o.ppm_flatten ? 2 : 1);
    KT(KG_FLUX_X, {
      rc = recon == 0 ? launch_flux_all<0>(h)
                      : (recon == 1 ? launch_flux_all<1>(h) : launch_flux_all<2>(h));
      if (rc) return rc;
    });
    return GRMHD_OK;
  }
  KT(KG_FLUX_X, { if ((rc = launch_flux_d<0>(h))) return rc; });
  KT(KG_FLUX_Y, {
    // the dynamic x-apron columns (P, B_c, B~^y, B~^z) for the y AND the z fluxes
    if (!h->E.emf && xcol_ok(h) && (rc = xcol_gather(h, 0, 10))) return rc;
    if ((rc = launch_flux_d<1>(h))) return rc;
  });
  KT(KG_FLUX_Z, { if ((rc = launch_flux_d<2>(h))) return rc; });
  return GRMHD_OK;
}

int one_step_eager(grmhd* h) {
  const Geom& g = h->g;
  KT(KG_MISC, {
    k_dt<<<1, 1, 0, h->s>>>(h->dst, g, 0);
    CKL("k_dt");
  });
  RkStage st[4];
  int ns = h->o.rk;
  if (ns == 2) {
    st[0] = {0, 0, 0, 0}; st[1] = {1, 0.5, 0.5, 0};
  } else if (ns == 3) {
    st[0] = {0, 0, 0, 0}; st[1] = {1, 0.75, 0.25, 0}; st[2] = {1, 1.0 / 3.0, 2.0 / 3.0, 0};
  } else {
    st[0] = {2, 0, 0, 0}; st[1] = {3, 0, 0, 0.5}; st[2] = {3, 0, 0, 1.0}; st[3] = {4, 0, 0, 0};
  }
  for (int s = 0; s < ns; s++) {
    int rc = compute_fluxes(h);
    if (rc) return rc;
    KT(KG_UPDATE, {
      const int gauge = h->E.gauge;
      if (gauge) {  // G_A, F_Psi^j and alpha on the vertices -1 .. n+1
        k_gauge_vertex<<<grd3(g.nx + 3, g.ny + 3, g.nz + 3), blk3(), 0, h->s>>>(h->base, g);
        CKL("k_gauge_vertex");
      }
      // with the upwind CT the edges have their own kernel; the Lorenz gauge adds the Psi row
      const int nrows = (h->E.emf ? 5 : 8) + (gauge ? 1 : 0);
      const dim3 ug((g.nx + 1 + 127) / 128, (g.ny + 1 + 1) / 2, nrows * (g.nz + 1)), ub(128, 2, 1);
      if (nrows == 8)
        k_update<8, false><<<ug, ub, 0, h->s>>>(h->base, g, h->dst, st[s], h->E.lorenz_xi);
      else if (nrows == 5)
        k_update<5, false><<<ug, ub, 0, h->s>>>(h->base, g, h->dst, st[s], h->E.lorenz_xi);
      else if (nrows == 9)
        k_update<9, true><<<ug, ub, 0, h->s>>>(h->base, g, h->dst, st[s], h->E.lorenz_xi);
      else
        k_update<6, true><<<ug, ub, 0, h->s>>>(h->base, g, h->dst, st[s], h->E.lorenz_xi);
      CKL("k_update");
      if (h->E.emf && h->uct_passes) {
        // every face -> edge parabola once: passes along x, y, z, then R11 + RK
        const int nsd = (g.nx + 1 + FX_VALID - 1) / FX_VALID;
        const long long nitems = (long long)nsd * (g.ny + 1) * (g.nz + 1);
        k_uct_xrow<<<(unsigned)((nitems + 3) / 4), 128, 0, h->s>>>(h->base, g, nsd, nitems, 3);
        CKL("k_uct_xrow");
        const int nsg = h->uct_nseg;
        const int sly = (g.ny + 1 + nsg - 1) / nsg, slz = (g.nz + 1 + nsg - 1) / nsg;
        // pass y finishes E_z, pass z finishes E_y and E_x: those go straight into R11 + RK
        k_uct_march<1><<<dim3((g.nx + 1 + 127) / 128, 2 * (g.nz + 1), (g.ny + sly) / sly), 128, 0,
                         h->s>>>(h->base, g, sly, 1, 2, h->dst, st[s], gauge);
        CKL("k_uct_march");
        k_uct_march<2><<<dim3((g.nx + 1 + 127) / 128, 2 * (g.ny + 1), (g.nz + slz) / slz), 128, 0,
                         h->s>>>(h->base, g, slz, 0, 3, h->dst, st[s], gauge);
        CKL("k_uct_march");
      } else if (h->E.emf) {
        k_emf_uct<<<dim3((g.nx + 1 + 127) / 128, (g.ny + 1 + 1) / 2, 3 * (g.nz + 1)),
                    dim3(128, 2, 1), 0, h->s>>>(h->base, g, h->dst, st[s], gauge);
        CKL("k_emf_uct");
      }
    });
    rc = after_stage(h, s == ns - 1);
    if (rc) return rc;
  }
  if (!small_block(h)) {  // (small blocks: t += dt is done by the last k_post)
    KT(KG_MISC, {
      k_dt<<<1, 1, 0, h->s>>>(h->dst, g, 1);
      CKL("k_dt");
    });
  }
  h->steps++;
  return GRMHD_OK;
}

void graph_drop(grmhd* h) {
  if (h->gexec) cudaGraphExecDestroy(h->gexec);
  h->gexec = nullptr;
  h->gstate = 0;
}

// Capture one_step_eager on the handle's own capture stream (the caller's stream may be the
// legacy default stream, which cannot be captured).  Nothing executes during the capture.
void graph_capture(grmhd* h) {
  h->gstate = 3;
  if (!h->cap_s && cudaStreamCreateWithFlags(&h->cap_s, cudaStreamNonBlocking) != cudaSuccess) {
    cudaGetLastError();
    h->cap_s = nullptr;
    return;
  }
  cudaStream_t user = h->s;
  const long long l0 = h->launches, s0 = h->steps;
  if (cudaStreamBeginCapture(h->cap_s, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
    cudaGetLastError();
    return;
  }
  h->s = h->cap_s;
  const int rc = one_step_eager(h);
  h->s = user;
  cudaGraph_t gr = nullptr;
  const cudaError_t e = cudaStreamEndCapture(h->cap_s, &gr);
  h->glaunches = h->launches - l0;
  h->launches = l0;
  h->steps = s0;
  if (rc == GRMHD_OK && e == cudaSuccess && gr &&
      cudaGraphInstantiate(&h->gexec, gr, 0) == cudaSuccess)
    h->gstate = 2;
  else {
    cudaGetLastError();
    h->gexec = nullptr;
    h->err[0] = 0;
  }
  if (gr) cudaGraphDestroy(gr);
}

int one_step(grmhd* h) {
  if (h->use_graph && !h->ktime) {
    if (h->gstate == 1) graph_capture(h);
    if (h->gstate == 2) {
      CK(cudaGraphLaunch(h->gexec, h->s));
      h->launches += h->glaunches;
      h->steps++;
      return GRMHD_OK;
    }
  }
  const int rc = one_step_eager(h);
  if (rc == GRMHD_OK && h->gstate == 0) h->gstate = 1;
  return rc;
}

// field_from_potential + prim->cons + max speed
int init_state(grmhd* h) {
  const Geom& g = h->g;
  h->dirty = false;
  int rc = fill_ghosts(h, fill_vecpot());
  if (rc) return rc;
  k_reset_state<<<1, 1, 0, h->s>>>(h->dst, 0);
  CKL("k_reset_state");
  k_post<true, false><<<grd_post(g), dim3(32, KP_BY, KP_BZ), 0, h->s>>>(
      h->base, nullptr, g, h->E, h->dst, 1);
  CKL("k_post");
  return launch_src(h);
}

}  // namespace

extern "C" {

size_t grmhd_workspace_bytes(int nx, int ny, int nz, int ghosts, const grmhd_opts* opts) {
  Geom g;
  if (ghosts != G || !valid_opts(opts) || !make_geom(nx, ny, nz, nullptr, opts, &g)) return 0;
  const size_t fields = (size_t)nfields_of(opts) * g.NPA * sizeof(double);
  const size_t stage = (size_t)stage_elems_of(g) * sizeof(double);
  const size_t mask = (size_t)g.NPA;  // bytes, multiple of 32
  return fields + stage + mask + 256;
}

int grmhd_create(int nx, int ny, int nz, int ghosts, const double dx[3], const grmhd_opts* opts,
                 void* workspace, size_t workspace_bytes, void* stream, grmhd** out) {
  if (!out) return GRMHD_EINVAL;
  *out = nullptr;
  if (!dx || !workspace || ghosts != G || !valid_opts(opts)) return GRMHD_EINVAL;
  const int n[3] = {nx, ny, nz};
  for (int a = 0; a < 3; a++) {
    if (n[a] < 1 || !(dx[a] > 0)) return GRMHD_EINVAL;
    if (opts->bc[a] == 1 && n[a] < 2) return GRMHD_EINVAL;
  }
  if (((uintptr_t)workspace & 255) != 0) return GRMHD_EINVAL;
  const size_t need = grmhd_workspace_bytes(nx, ny, nz, ghosts, opts);
  if (need == 0) return GRMHD_EINVAL;
  if (workspace_bytes < need) return GRMHD_ENOMEM;
  grmhd* h = new (std::nothrow) grmhd;
  if (!h) return GRMHD_ENOMEM;
  make_geom(nx, ny, nz, dx, opts, &h->g);
  h->o = *opts;
  h->E = make_eos(*opts);
  h->nfields = nfields_of(opts);
  h->stage_elems = stage_elems_of(h->g);
  h->base = (double*)workspace;
  h->stage = h->base + (size_t)h->nfields * h->g.NPA;
  h->mask = (unsigned char*)(h->stage + h->stage_elems);
  h->dst = (DevState*)(h->mask + h->g.NPA);
  h->s = (cudaStream_t)stream;
  // the whole workspace starts as zeros (ghost cells of U~ stay 0 for the handle's lifetime)
  cudaError_t e = cudaMemsetAsync(workspace, 0, need, h->s);
  if (e != cudaSuccess) {
    delete h;
    return GRMHD_ECUDA;
  }
  h->tma_ok = make_tensor_maps(h);
  {
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && nsm > 0)
      h->nsm = nsm;
    else
      cudaGetLastError();
  }
  *out = h;
  return GRMHD_OK;
}

int grmhd_destroy(grmhd* h) {
  if (!h) return GRMHD_EINVAL;
  cudaStreamSynchronize(h->s);
  graph_drop(h);
  if (h->cap_s) cudaStreamDestroy(h->cap_s);
  for (cudaEvent_t e : h->ev) cudaEventDestroy(e);
  delete h;
  return GRMHD_OK;
}

int grmhd_set_metric(grmhd* h, const double* const field[16]) {
  if (!h) return GRMHD_EINVAL;
  if (!field) return fail(h, GRMHD_EINVAL, "set_metric: NULL field array");
  for (int f = 0; f < 16; f++)
    if (!field[f]) return fail(h, GRMHD_EINVAL, "set_metric: NULL field");
  for (int f = 0; f < 16; f++) {
    int rc = copy_in(h, field[f], F_MET + f, false);
    if (rc) return rc;
  }
  // the metric is held fixed from here on: face values (R4) and sqrt(gamma_f) once
  const dim3 fb(32, 4, 1), fg((h->g.PXP + 31) / 32, (h->g.PY + 3) / 4, h->g.PZ);
  k_face_metric<0><<<fg, fb, 0, h->s>>>(h->base, h->g);
  CKL("k_face_metric");
  k_face_metric<1><<<fg, fb, 0, h->s>>>(h->base, h->g);
  CKL("k_face_metric");
  k_face_metric<2><<<fg, fb, 0, h->s>>>(h->base, h->g);
  CKL("k_face_metric");
  // compact copies of the x-apron columns of the static y and z face metric (slots 10 .. 31);
  // always kept up to date where they fit, whatever the options say now
  if ((long long)XC_NSLOT * 2 * h->g.PY * h->g.PZ <= h->g.NPA) {
    int rc = xcol_gather(h, 10, 22);
    if (rc) return rc;
  }
  h->have_metric = true;
  // a new metric under existing primitives: U~, B_c, the sources and the max speed are rebuilt
  // from the primitives by the next call that needs them
  if (h->have_prims) h->dirty = true;
  return sync_if_host(h, field[0]);
}

int grmhd_set_prims(grmhd* h, const double* const field[8]) {
  if (!h) return GRMHD_EINVAL;
  if (!field) return fail(h, GRMHD_EINVAL, "set_prims: NULL field array");
  if (!h->have_metric) return fail(h, GRMHD_ESTATE, "set_prims before set_metric");
  for (int r = 0; r < 5; r++)
    if (!field[r]) return fail(h, GRMHD_EINVAL, "set_prims: NULL hydro field");
  const bool haveB = field[5] && field[6] && field[7];
  if (!haveB && (field[5] || field[6] || field[7]))
    return fail(h, GRMHD_EINVAL, "set_prims: B fields must be all given or all NULL");
  const Geom& g = h->g;
  int rc;
  for (int r = 0; r < 5; r++)
    if ((rc = copy_in(h, field[r], F_P + r, false))) return rc;
  if ((rc = fill_ghosts(h, fill_prims()))) return rc;
  for (int d = 0; d < 3; d++) {
    if ((rc = zero_field(h, F_Y + 5 + d))) return rc;
    if (d == 0 && (rc = zero_field(h, F_Y + 8))) return rc;  // Psi_mhd = 0
    if ((rc = zero_field(h, F_B0 + d))) return rc;
  }
  if (haveB) {
    // G16: B~0 on faces from the ghost-filled cell-centred input (held in F_BF meanwhile)
    FillArgs fa{};
    fa.nf = 3;
    for (int d = 0; d < 3; d++) {
      if ((rc = copy_in(h, field[5 + d], F_BF + d, false))) return rc;
      fa.id[d] = F_BF + d; fa.stag[d] = 0; fa.kind[d] = 0;
    }
    if ((rc = fill_ghosts(h, fa))) return rc;
    for (int d = 0; d < 3; d++) {
      k_b0_from_centred<<<grd3(g.nx + (d == 0), g.ny + (d == 1), g.nz + (d == 2)), blk3(), 0,
                          h->s>>>(h->base, g, d);
      CKL("k_b0_from_centred");
      fa.id[d] = F_B0 + d; fa.stag[d] = 1 << d; fa.kind[d] = 0;
    }
    if ((rc = fill_ghosts(h, fa))) return rc;
  }
  h->have_prims = true;
  h->steps = 0;
  k_reset_state<<<1, 1, 0, h->s>>>(h->dst, 1);
  CKL("k_reset_state");
  h->dirty = true;
  return sync_if_host(h, field[0]);
}

int grmhd_set_vecpot(grmhd* h, const double* const field[3]) {
  if (!h) return GRMHD_EINVAL;
  if (!field) return fail(h, GRMHD_EINVAL, "set_vecpot: NULL field array");
  if (!h->have_prims) return fail(h, GRMHD_ESTATE, "set_vecpot before set_prims");
  for (int d = 0; d < 3; d++)
    if (!field[d]) return fail(h, GRMHD_EINVAL, "set_vecpot: NULL field");
  for (int d = 0; d < 3; d++) {
    int rc = copy_in(h, field[d], F_Y + 5 + d, true);
    if (rc) return rc;
  }
  h->dirty = true;
  return sync_if_host(h, field[0]);
}

int grmhd_set_mask(grmhd* h, const unsigned char* mask) {
  if (!h) return GRMHD_EINVAL;
  graph_drop(h);  // the mask pointer is a kernel argument
  if (!mask) { h->have_mask = false; return GRMHD_OK; }
  const Geom& g = h->g;
  const long long n = (long long)(g.nx + 2 * G) * (g.ny + 2 * G) * (g.nz + 2 * G);
  const unsigned char* src = mask;
  if (!is_device_ptr(mask)) {
    CK(cudaMemcpyAsync(h->stage, mask, (size_t)n, cudaMemcpyDefault, h->s));
    src = (const unsigned char*)h->stage;
  }
  k_repack_mask<<<grd1(n), 256, 0, h->s>>>(src, h->mask, g);
  CKL("k_repack_mask");
  h->have_mask = true;
  return sync_if_host(h, mask);
}

int grmhd_step(grmhd* h, int n, double cfl) {
  if (!h) return GRMHD_EINVAL;
  if (n < 0) return fail(h, GRMHD_EINVAL, "step: n < 0");
  if (!h->have_metric || !h->have_prims) return fail(h, GRMHD_ESTATE, "step before set_metric/set_prims");
  int rc = h->dirty ? init_state(h) : GRMHD_OK;
  if (rc) return rc;
  if ((rc = set_params(h, cfl, -1.0))) return rc;
  for (int s = 0; s < n; s++)
    if ((rc = one_step(h))) return rc;
  return GRMHD_OK;
}

int grmhd_step_until(grmhd* h, double t_end, double cfl, int* nsteps_done) {
  if (!h) return GRMHD_EINVAL;
  if (!h->have_metric || !h->have_prims) return fail(h, GRMHD_ESTATE, "step_until before set_metric/set_prims");
  if (t_end < 0) return fail(h, GRMHD_EINVAL, "step_until: t_end < 0");
  int rc = h->dirty ? init_state(h) : GRMHD_OK;
  if (rc) return rc;
  rc = set_params(h, cfl, t_end);
  if (rc) return rc;
  int n = 0;
  for (;;) {
    DevState st;
    CK(cudaMemcpyAsync(&st, h->dst, sizeof st, cudaMemcpyDeviceToHost, h->s));
    CK(cudaStreamSynchronize(h->s));
    if (st.bad_dt) return fail(h, GRMHD_ENUMERIC, "dt not finite/positive");
    if (!(t_end - st.t > 1e-12 * std::fmax(1.0, std::fabs(t_end)))) break;
    if ((rc = one_step(h))) return rc;
    n++;
  }
  if (nsteps_done) *nsteps_done = n;
  return GRMHD_OK;
}

int grmhd_get_prims(grmhd* h, double* const field[8]) {
  if (!h) return GRMHD_EINVAL;
  if (!field) return fail(h, GRMHD_EINVAL, "get_prims: NULL field array");
  if (h->dirty) { int rc0 = init_state(h); if (rc0) return rc0; }
  for (int r = 0; r < 8; r++) {
    if (!field[r]) return fail(h, GRMHD_EINVAL, "get_prims: NULL field");
    int rc = copy_out(h, r < 5 ? F_P + r : F_BC + (r - 5), field[r], false, 0);
    if (rc) return rc;
  }
  CK(cudaStreamSynchronize(h->s));
  return GRMHD_OK;
}

int grmhd_get_cons(grmhd* h, double* const field[8]) {
  if (!h) return GRMHD_EINVAL;
  if (!field) return fail(h, GRMHD_EINVAL, "get_cons: NULL field array");
  if (h->dirty) { int rc0 = init_state(h); if (rc0) return rc0; }
  for (int r = 0; r < 8; r++) {
    if (!field[r]) return fail(h, GRMHD_EINVAL, "get_cons: NULL field");
    int rc = copy_out(h, r < 5 ? F_Y + r : F_BC + (r - 5), field[r], false, r < 5 ? 1 : 2);
    if (rc) return rc;
  }
  CK(cudaStreamSynchronize(h->s));
  return GRMHD_OK;
}

int grmhd_get_vecpot(grmhd* h, double* const field[3]) {
  if (!h) return GRMHD_EINVAL;
  if (!field) return fail(h, GRMHD_EINVAL, "get_vecpot: NULL field array");
  if (h->dirty) { int rc0 = init_state(h); if (rc0) return rc0; }
  for (int d = 0; d < 3; d++) {
    if (!field[d]) return fail(h, GRMHD_EINVAL, "get_vecpot: NULL field");
    int rc = copy_out(h, F_Y + 5 + d, field[d], true, 0);
    if (rc) return rc;
  }
  CK(cudaStreamSynchronize(h->s));
  return GRMHD_OK;
}

int grmhd_get_psi(grmhd* h, double* field) {
  if (!h) return GRMHD_EINVAL;
  if (!field) return fail(h, GRMHD_EINVAL, "get_psi: NULL field");
  if (h->dirty) { int rc0 = init_state(h); if (rc0) return rc0; }
  int rc = copy_out(h, F_Y + 8, field, true, 0);
  if (rc) return rc;
  CK(cudaStreamSynchronize(h->s));
  return GRMHD_OK;
}

int grmhd_set_option(grmhd* h, const char* key, double value) {
  if (!h || !key) return GRMHD_EINVAL;
  if (std::strcmp(key, "graph") == 0) {
    if (value != 0.0 && value != 1.0) return fail(h, GRMHD_EINVAL, "set_option: graph is 0 or 1");
    h->use_graph = (int)value;
    return GRMHD_OK;
  }
  if (std::strcmp(key, "fixed_dt") != 0 && std::strcmp(key, "kernel_timing") != 0)
    graph_drop(h);  // every other option changes kernel arguments or the launch sequence
  if (std::strcmp(key, "fixed_dt") == 0) {
    h->fixed_dt = value;
    return GRMHD_OK;
  }
  if (std::strcmp(key, "flux_kernel") == 0) {
    if (value != 0.0 && value != 1.0) return fail(h, GRMHD_EINVAL, "set_option: flux_kernel is 0 or 1");
    h->flux_impl = (int)value;
    return GRMHD_OK;
  }
  if (std::strcmp(key, "small_fuse") == 0) {
    if (value != 0.0 && value != 1.0) return fail(h, GRMHD_EINVAL, "set_option: small_fuse is 0 or 1");
    h->small_fuse = (int)value;
    return GRMHD_OK;
  }
  if (std::strcmp(key, "flux_xcol") == 0) {
    if (value != 0.0 && value != 1.0) return fail(h, GRMHD_EINVAL, "set_option: flux_xcol is 0 or 1");
    h->xcol = (int)value;
    return GRMHD_OK;
  }
  if (std::strcmp(key, "src_kernel") == 0) {
    if (value != 0.0 && value != 1.0) return fail(h, GRMHD_EINVAL, "set_option: src_kernel is 0 or 1");
    h->src_impl = (int)value;
    return GRMHD_OK;
  }
  if (std::strcmp(key, "gauge") == 0) {
    if (value != 0.0 && value != 1.0) return fail(h, GRMHD_EINVAL, "set_option: gauge is 0 or 1");
    h->E.gauge = (int)value;
    return GRMHD_OK;
  }
  if (std::strcmp(key, "lorenz_xi") == 0) {
    if (!(value >= 0.0)) return fail(h, GRMHD_EINVAL, "set_option: lorenz_xi < 0");
    h->E.lorenz_xi = value;
    return GRMHD_OK;
  }
  if (std::strcmp(key, "emf") == 0) {
    if (value != 0.0 && value != 1.0) return fail(h, GRMHD_EINVAL, "set_option: emf is 0 or 1");
    h->E.emf = (int)value;
    return GRMHD_OK;
  }
  if (std::strcmp(key, "c2p_backup") == 0) {
    if (value != 0.0 && value != 1.0) return fail(h, GRMHD_EINVAL, "set_option: c2p_backup is 0 or 1");
    h->E.c2p_backup = (int)value;
    return GRMHD_OK;
  }
  if (std::strcmp(key, "uct_nseg") == 0) {
    if (!(value >= 1.0 && value <= 64.0)) return fail(h, GRMHD_EINVAL, "set_option: uct_nseg");
    h->uct_nseg = (int)value;
    return GRMHD_OK;
  }
  if (std::strcmp(key, "uct_passes") == 0) {
    h->uct_passes = value != 0.0;
    return GRMHD_OK;
  }
  if (std::strcmp(key, "kernel_timing") == 0) {
    int rc = kt_flush(h);
    if (rc) return rc;
    h->ktime = value != 0.0;
    for (int q = 0; q < GRMHD_NKGROUPS; q++) { h->kms[q] = 0.0; h->kcnt[q] = 0; }
    if (h->ktime && h->ev.empty()) {
      h->ev.resize(2048);
      h->ev_grp.resize(1024);
      for (auto& e : h->ev) CK(cudaEventCreate(&e));
    }
    return GRMHD_OK;
  }
  return fail(h, GRMHD_EINVAL, "set_option: unknown key");
}

int grmhd_get_stats(grmhd* h, grmhd_stats* out) {
  if (!h || !out) return GRMHD_EINVAL;
  if (h->dirty) { int rc0 = init_state(h); if (rc0) return rc0; }
  DevState st;
  CK(cudaMemcpyAsync(&st, h->dst, sizeof st, cudaMemcpyDeviceToHost, h->s));
  CK(cudaStreamSynchronize(h->s));
  out->t = st.t; out->dt = st.dt;
  for (int d = 0; d < 3; d++) {
    double v;
    std::memcpy(&v, &st.ms_acc[d], sizeof v);
    out->maxspeed[d] = v;
  }
  out->steps = h->steps;
  out->c2p_fail = st.c2p_fail; out->p_fix = st.p_fix; out->atmo = st.atmo;
  out->w_cap = st.w_cap; out->c2p_maxiter = st.c2p_maxiter;
  out->c2p_backup = st.c2p_backup;
  if (st.bad_dt) return fail(h, GRMHD_ENUMERIC, "dt not finite/positive");
  return GRMHD_OK;
}

int grmhd_get_kernel_times(grmhd* h, double ms[GRMHD_NKGROUPS],
                           long long launches[GRMHD_NKGROUPS]) {
  if (!h || !ms || !launches) return GRMHD_EINVAL;
  int rc = kt_flush(h);
  if (rc) return rc;
  for (int q = 0; q < GRMHD_NKGROUPS; q++) { ms[q] = h->kms[q]; launches[q] = h->kcnt[q]; }
  return GRMHD_OK;
}

long long grmhd_launch_count(const grmhd* h) { return h ? h->launches : 0; }

const char* grmhd_last_error(const grmhd* h) { return h ? h->err : "NULL handle"; }

// ---- stand-alone batches --------------------------------------------------------------
int grmhd_prim2con_batch(const double* const prim[8], const double* const metric[10],
                         double* const cons[8], long long n, const grmhd_opts* opts,
                         void* stream) {
  if (!prim || !metric || !cons || n < 0 || !valid_opts(opts)) return GRMHD_EINVAL;
  BatchPtrs bp{};
  for (int r = 0; r < 8; r++) { bp.prim[r] = prim[r]; bp.cons[r] = cons[r]; }
  for (int r = 0; r < 10; r++) bp.met[r] = metric[r];
  for (int r = 0; r < 8; r++) if (!prim[r] || !cons[r]) return GRMHD_EINVAL;
  for (int r = 0; r < 10; r++) if (!metric[r]) return GRMHD_EINVAL;
  if (n == 0) return GRMHD_OK;
  k_prim2con_batch<<<grd1(n), 256, 0, (cudaStream_t)stream>>>(bp, n, make_eos(*opts));
  return cudaGetLastError() == cudaSuccess ? GRMHD_OK : GRMHD_ECUDA;
}

int grmhd_con2prim_batch(const double* const cons[8], const double* const metric[10],
                         double* const prim[5], int* status, int* iters, long long n,
                         const grmhd_opts* opts, void* stream) {
  if (!cons || !metric || !prim || !status || !iters || n < 0 || !valid_opts(opts))
    return GRMHD_EINVAL;
  BatchPtrs bp{};
  for (int r = 0; r < 8; r++) { if (!cons[r]) return GRMHD_EINVAL; bp.prim[r] = cons[r]; }
  for (int r = 0; r < 10; r++) { if (!metric[r]) return GRMHD_EINVAL; bp.met[r] = metric[r]; }
  for (int r = 0; r < 5; r++) { if (!prim[r]) return GRMHD_EINVAL; bp.cons[r] = prim[r]; }
  if (n == 0) return GRMHD_OK;
  k_con2prim_batch<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(
      bp, status, iters, n, make_eos(*opts));
  return cudaGetLastError() == cudaSuccess ? GRMHD_OK : GRMHD_ECUDA;
}

int grmhd_con2prim1d_batch(const double* const cons[8], const double* const metric[10],
                           double* const prim[5], int* status, int* iters, long long n,
                           const grmhd_opts* opts, void* stream) {
  if (!cons || !metric || !prim || !status || !iters || n < 0 || !valid_opts(opts))
    return GRMHD_EINVAL;
  BatchPtrs bp{};
  for (int r = 0; r < 8; r++) { if (!cons[r]) return GRMHD_EINVAL; bp.prim[r] = cons[r]; }
  for (int r = 0; r < 10; r++) { if (!metric[r]) return GRMHD_EINVAL; bp.met[r] = metric[r]; }
  for (int r = 0; r < 5; r++) { if (!prim[r]) return GRMHD_EINVAL; bp.cons[r] = prim[r]; }
  if (n == 0) return GRMHD_OK;
  k_con2prim1d_batch<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(
      bp, status, iters, n, make_eos(*opts));
  return cudaGetLastError() == cudaSuccess ? GRMHD_OK : GRMHD_ECUDA;
}

int grmhd_dfma_peak(double* out, long long threads, int iters, void* stream) {
  if (!out || threads < 1 || iters < 1) return GRMHD_EINVAL;
  k_dfma_peak<<<(unsigned)((threads + 255) / 256), 256, 0, (cudaStream_t)stream>>>(out, threads,
                                                                                   iters);
  return cudaGetLastError() == cudaSuccess ? GRMHD_OK : GRMHD_ECUDA;
}

}  // extern "C"

// =============================================================================================
// A8 without any allocation: grmhd_maxspeed_noalloc (include/grmhd.h).
//
// The max-characteristic-speed reduction of a handle accumulates into scratch the caller's
// workspace holds (DevState::ms_acc).  Callers that cannot provide or allocate a workspace --
// code under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc -- get the
// same reduction on plain arrays of states with its scratch in a FILE-SCOPE device array of a
// fixed, modest size: every GPU that loads the library holds these NOALLOC_SCRATCH_BYTES until the
// process exits.  No cudaMalloc, cudaFree or allocating library routine is called.
//
// In host code the NAME of a __device__ array is a host-side stand-in, not a device address: a
// kernel handed `g_noalloc_scratch` from the host would fault (or, where the GPU can reach host
// memory, silently use the wrong memory).  The device address is asked for once per device, with
// that device current, through cudaGetSymbolAddress, and that pointer is what the kernel gets.
//
// Layout of the scratch: [0, 256 B) header -- a block counter (unsigned) that MUST start at zero;
// then 3 doubles per block, the block's max |lambda| in x, y, z.  The array is shared by every
// call and keeps the last call's contents: the header is cleared at the start of every call (on
// the call's stream), the partial maxima of the blocks [0, nblocks) are all overwritten before
// the last block reads exactly that range, so nothing stale is ever read.  Calls that overlap on
// the GPU (two streams, two threads) would race on the array: callers serialise them.
namespace {

constexpr int NOALLOC_BLOCK = 256;                                   // states per block
constexpr long long NOALLOC_MAX_BLOCKS = GRMHD_NOALLOC_MAX_STATES / NOALLOC_BLOCK;
constexpr int NOALLOC_HDR = 32;                                      // doubles (256 B)
constexpr size_t NOALLOC_SCRATCH_DOUBLES = NOALLOC_HDR + 3 * (size_t)NOALLOC_MAX_BLOCKS;
constexpr size_t NOALLOC_SCRATCH_BYTES = NOALLOC_SCRATCH_DOUBLES * sizeof(double);  // 384.25 KiB
static_assert(GRMHD_NOALLOC_MAX_STATES % NOALLOC_BLOCK == 0, "whole blocks");
static_assert(NOALLOC_SCRATCH_BYTES <= (1u << 20), "the static scratch stays modest");

static __device__ __align__(256) double g_noalloc_scratch[NOALLOC_SCRATCH_DOUBLES];

// R16 on n plain states: block b leaves its three maxima in scratch[HDR + 3 b ..]; the block
// that arrives last (counter in the header) reduces the nblocks partial maxima to out[0..2] and
// puts the counter back to zero.  Same per-state arithmetic as the handle's path (cell_speeds);
// max of non-negative doubles is exact and order independent.
__global__ void __launch_bounds__(NOALLOC_BLOCK)
k_maxspeed_noalloc(BatchPtrs b, long long n, Eos E, double* __restrict__ scratch,
                   double* __restrict__ out) {
  __shared__ double sm[3][NOALLOC_BLOCK / 32];
  __shared__ bool last;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const long long q = blockIdx.x * (long long)NOALLOC_BLOCK + tid;
  double s[3] = {0.0, 0.0, 0.0};
  if (q < n) {
    const Prim P = {b.prim[0][q], b.prim[1][q], b.prim[2][q], b.prim[3][q],
                    b.prim[4][q], b.prim[5][q], b.prim[6][q], b.prim[7][q]};
    cell_speeds(P, batch_met(b, q), E, s);
  }
  auto block_max = [&]() {  // s[] of thread 0 = max over the block
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
      for (int d = 0; d < 3; d++) s[d] = fmax(s[d], __shfl_xor_sync(0xffffffffu, s[d], o));
    if (lane == 0)
      for (int d = 0; d < 3; d++) sm[d][warp] = s[d];
    __syncthreads();
    if (warp == 0) {
#pragma unroll
      for (int d = 0; d < 3; d++) s[d] = lane < NOALLOC_BLOCK / 32 ? sm[d][lane] : 0.0;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int d = 0; d < 3; d++) s[d] = fmax(s[d], __shfl_xor_sync(0xffffffffu, s[d], o));
    }
  };
  block_max();
  unsigned* counter = reinterpret_cast<unsigned*>(scratch);
  double* part = scratch + NOALLOC_HDR;
  if (tid == 0) {
    for (int d = 0; d < 3; d++) part[3 * (size_t)blockIdx.x + d] = s[d];
    __threadfence();  // the partial maxima are visible before the arrival is counted
    last = atomicAdd(counter, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  s[0] = s[1] = s[2] = 0.0;
  for (unsigned k = tid; k < gridDim.x; k += NOALLOC_BLOCK)
    for (int d = 0; d < 3; d++) s[d] = fmax(s[d], __ldcg(part + 3 * (size_t)k + d));
  __syncthreads();  // sm[] is reused
  block_max();
  if (tid == 0) {
    for (int d = 0; d < 3; d++) out[d] = s[d];
    *counter = 0u;  // as the next call expects it (that call clears the header anyway)
  }
}

// set-up, once per device: the DEVICE address of the scratch array on the current device
int noalloc_scratch(double** ptr, char* err, size_t err_len) {
  constexpr int MAXDEV = 64;
  static double* cached[MAXDEV] = {nullptr};
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess && (dev < 0 || dev >= MAXDEV)) e = cudaErrorInvalidDevice;
  if (e == cudaSuccess && !cached[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e == cudaSuccess && !p) e = cudaErrorInvalidSymbol;
    if (e == cudaSuccess) cached[dev] = static_cast<double*>(p);
  }
  if (e != cudaSuccess) {
    cudaGetLastError();
    if (err && err_len)
      std::snprintf(err, err_len, "grmhd_maxspeed_noalloc: cudaGetSymbolAddress: %s",
                    cudaGetErrorString(e));
    return GRMHD_ECUDA;
  }
  *ptr = cached[dev];
  return GRMHD_OK;
}

}  // namespace

extern "C" int grmhd_maxspeed_noalloc(const double* const prim[8], const double* const metric[10],
                                      long long n, const grmhd_opts* opts, double* maxspeed,
                                      void* stream, char* err, size_t err_len) {
  auto say = [&](const char* m) { if (err && err_len) std::snprintf(err, err_len, "%s", m); };
  if (err && err_len) err[0] = 0;
  if (!prim || !metric || !maxspeed || n < 1 || !valid_opts(opts)) {
    say("grmhd_maxspeed_noalloc: NULL argument, n < 1 or invalid options");
    return GRMHD_EINVAL;
  }
  if (n > GRMHD_NOALLOC_MAX_STATES) {
    if (err && err_len)
      std::snprintf(err, err_len,
                    "grmhd_maxspeed_noalloc: n = %lld exceeds GRMHD_NOALLOC_MAX_STATES = %lld (the "
                    "static scratch holds one partial maximum per %d states); split the batch",
                    n, (long long)GRMHD_NOALLOC_MAX_STATES, NOALLOC_BLOCK);
    return GRMHD_ELIMIT;
  }
  BatchPtrs bp{};
  for (int r = 0; r < 8; r++) { if (!prim[r]) { say("grmhd_maxspeed_noalloc: NULL prim array"); return GRMHD_EINVAL; } bp.prim[r] = prim[r]; }
  for (int r = 0; r < 10; r++) { if (!metric[r]) { say("grmhd_maxspeed_noalloc: NULL metric array"); return GRMHD_EINVAL; } bp.met[r] = metric[r]; }
  double* scratch = nullptr;
  const int rc = noalloc_scratch(&scratch, err, err_len);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  // the header (block counter) must start at zero whatever an earlier call left behind
  cudaError_t e = cudaMemsetAsync(scratch, 0, NOALLOC_HDR * sizeof(double), st);
  if (e == cudaSuccess) {
    const unsigned nblk = (unsigned)((n + NOALLOC_BLOCK - 1) / NOALLOC_BLOCK);
    k_maxspeed_noalloc<<<nblk, NOALLOC_BLOCK, 0, st>>>(bp, n, make_eos(*opts), scratch, maxspeed);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) {
    if (err && err_len)
      std::snprintf(err, err_len, "grmhd_maxspeed_noalloc: %s", cudaGetErrorString(e));
    return GRMHD_ECUDA;
  }
  return GRMHD_OK;
}

/* grmhd.h -- C ABI of libgrmhd.so: the B200 (sm_100a) fp64 GRMHD substep library.
 *
 * What it computes: the Valencia-formulation GRMHD right-hand side and Runge-Kutta
 * substep of AsterX (arXiv 2406.11669; PAPER.md) on ONE uniform 3-D Cartesian block
 * with the spacetime metric held fixed:
 *   conservative->primitive recovery (eqs 36-41; atmosphere PAPER.md:326),
 *   minmod / PPM face reconstruction,
 *   HLLE fluxes in x,y,z (eq. 29; state/flux vectors eq. 18),
 *   flux divergence + metric sources (eqs 17,19),
 *   staggered vector-potential update with flux-CT electric field, B = curl A
 *   (algebraic gauge PAPER.md:159),
 *   RK2/RK3/RK4 stage combination and
 *   a max-characteristic-speed reduction for the CFL time step.
 * The ADM variables alpha, beta^i, gamma_ij, K_ij are INPUT fields.
 * DESIGN.md lists every reading of the paper (R/G rows) this library implements.
 *
 * Memory model
 *   - Every pointer argument marked [dev|host] may be a CUDA device pointer or a host
 *     pointer (pinned host memory recommended); the library copies with
 *     cudaMemcpyDefault (unified virtual addressing decides the direction).
 *     INPUT arrays in host memory have been consumed when the set_* call returns (the call
 *     waits for its copies: the caller may reuse or free them at once); with device sources
 *     set_* only enqueues on the handle's stream and the arrays must stay unchanged until that
 *     work has run.  OUTPUT calls (get_*) synchronise the stream before returning.
 *   - The caller owns every buffer, including the workspace (device memory, e.g. a
 *     torch tensor).  The library never allocates device memory for fields; it carves its
 *     structure-of-arrays state out of the workspace.  The workspace must stay alive and
 *     untouched until grmhd_destroy.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  All work of a
 *     handle is enqueued on that one stream.  Handles are not thread-safe.
 *
 * Array layout (all fp64, C order, x fastest), g = ghosts (must be 3):
 *   cell-centred arrays : shape (nz+2g, ny+2g, nx+2g); cell (i,j,k), i in [-g, nx+g), is at
 *                         linear index ((k+g)*(ny+2g) + (j+g))*(nx+2g) + (i+g);
 *                         centre x_i = x_0 + (i+1/2) dx.
 *   staggered arrays    : shape (nz+2g+1, ny+2g+1, nx+2g+1), LOWER convention:
 *                         A_x[i,j,k] at (i, j-1/2, k-1/2); A_y at (i-1/2, j, k-1/2);
 *                         A_z at (i-1/2, j-1/2, k)     (Fig. 1).
 *
 * Errors: every call returns GRMHD_OK (0) or a negative code; no exceptions, aborts or
 * stdout.  grmhd_last_error gives a human-readable string for the last failure.
 * Per-cell con2prim failures are not errors; they are counted (grmhd_get_stats).
 */
#ifndef GRMHD_H
#define GRMHD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GRMHD_OK        0
#define GRMHD_EINVAL   -1  /* bad size / NULL pointer / ghosts != 3 / bad option        */
#define GRMHD_ENOMEM   -2  /* workspace too small                                      */
#define GRMHD_ESTATE   -3  /* call order: step before metric+prims, vecpot before prims */
#define GRMHD_ECUDA    -4  /* CUDA runtime error (string in grmhd_last_error)          */
#define GRMHD_ENUMERIC -5  /* dt came out NaN / non-positive / infinite                */
#define GRMHD_ELIMIT   -6  /* size beyond the fixed maximum of a no-allocation entry point */

typedef struct grmhd grmhd; /* opaque handle (host memory, owned by the library) */

/* Options.  EOS: ideal fluid p=(Gamma-1) rho eps (eq. 46); the atmosphere
 * uses the polytrope p=K rho^Gamma_p (eqs 47-48). */
typedef struct {
  double gamma_ad;   /* ideal-fluid adiabatic index Gamma, eq. (46)                        */
  double poly_k;     /* atmosphere polytropic constant K, eq. (47)                         */
  double poly_gamma; /* atmosphere polytropic exponent, eq. (47)                           */
  double rho_atm;    /* rest-mass density floor rho_atm                     */
  double p_floor;    /* pressure floor, > 0                                                */
  double w_max;      /* Lorentz-factor cap (paper silent; G20), e.g. 100         */
  double c2p_tol;    /* Newton stop: |dz|/z + |dv2| < c2p_tol (G18), e.g. 1e-12  */
  int    c2p_maxit;  /* Newton iteration cap, e.g. 100                                     */
  int    recon;      /* 0 = minmod, 1 = PPM                                 */
  int    ppm_flatten;/* 1 = PPM shock flattening on (G8)                         */
  int    riemann;    /* 0 = HLLE eq. (29); 1 = Lax-Friedrichs eq. (30)                     */
  int    rk;         /* 2 = SSP-RK2, 3 = SSP-RK3, 4 = classic RK4 (G15)          */
  int    bc[3];      /* per axis x,y,z: 0 = periodic, 1 = outflow           */
} grmhd_opts;

typedef struct {
  double t;             /* simulation time reached                                         */
  double dt;            /* last time step used                                             */
  double maxspeed[3];   /* max |lambda| per direction of the CURRENT primitives (A8)       */
  long long steps;      /* full RK steps taken                                             */
  long long c2p_fail;   /* cell-substeps reset to atmosphere after a failed Newton solve   */
  long long p_fix;      /* cell-substeps whose pressure was raised to p_floor              */
  long long atmo;       /* cell-substeps reset because D <= rho_atm or masked              */
  long long w_cap;      /* cell-substeps whose velocity was rescaled to w_max              */
  long long c2p_maxiter;/* largest Newton iteration count seen                             */
  long long c2p_backup; /* cell-substeps recovered by the 1-D backup scheme ("c2p_backup")  */
} grmhd_stats;

/* Bytes of DEVICE workspace the handle needs for this block (0 on invalid arguments). */
size_t grmhd_workspace_bytes(int nx, int ny, int nz, int ghosts, const grmhd_opts* opts);

/* Create a handle.  dx[3]: host array of cell sizes.  workspace: [dev] pointer, at least
 * grmhd_workspace_bytes() bytes, 256-byte aligned.  stream: cudaStream_t or NULL.
 * Errors: EINVAL (nx,ny,nz < 1, < 2 on an outflow axis, ghosts != 3, dx <= 0, bad opts),
 * ENOMEM (workspace too small), ECUDA. */
int grmhd_create(int nx, int ny, int nz, int ghosts, const double dx[3],
                 const grmhd_opts* opts, void* workspace, size_t workspace_bytes,
                 void* stream, grmhd** out);
int grmhd_destroy(grmhd* h);

/* 16 cell-centred padded arrays [dev|host], ghosts SUPPLIED BY THE CALLER, in the order
 * alpha, betax, betay, betaz, gxx, gxy, gxz, gyy, gyz, gzz, kxx, kxy, kxz, kyy, kyz, kzz
 * (ADM variables).  field: host array of 16 pointers.
 * The metric is held fixed from this call on: the face values the Riemann solver needs (4-point
 * Lagrange interpolation along the face normal, and sqrt(gamma) of the face) are
 * formed here, once.  May be called again on a live handle: the conserved variables, the
 * cell-centred B, the sources and the max speed are then rebuilt from the current primitives
 * with the new metric by the next call that needs them. */
int grmhd_set_metric(grmhd* h, const double* const field[16]);

/* 8 cell-centred padded arrays [dev|host]: rho, vx, vy, vz (Eulerian v^i), press,
 * Bx, By, Bz (Eulerian B^i; the three B pointers may all be NULL = no static field).
 * Fills ghosts by the boundary condition, builds the static densitised face field B~0
 * (G16), zeroes A_i, and initialises the conserved variables by eqs (20)-(22)
 * (PAPER.md:379).  Requires set_metric first (ESTATE). */
int grmhd_set_prims(grmhd* h, const double* const field[8]);

/* 3 staggered arrays [dev|host] A_x, A_y, A_z; total field B~ = B~0 + curl A (eq. 24,
 * PAPER.md:149).  Requires set_prims first (ESTATE); re-initialises the conserved
 * variables with the new field. */
int grmhd_set_vecpot(grmhd* h, const double* const field[3]);

/* Optional cell-centred padded uint8 array [dev|host]; cells with mask != 0 are reset to
 * atmosphere at every con2prim (excision floor, BASELINE config 3).  NULL clears it. */
int grmhd_set_mask(grmhd* h, const unsigned char* mask);

/* n full RK steps; dt = cfl * min_d dx_d / maxspeed_d from the primitives at the start of
 * each step (or the "fixed_dt" option).  Asynchronous: returns after enqueue. */
int grmhd_step(grmhd* h, int n, double cfl);

/* Steps until t >= t_end, clipping the last dt; synchronises once per step.
 * nsteps_done may be NULL. */
int grmhd_step_until(grmhd* h, double t_end, double cfl, int* nsteps_done);

/* Outputs [dev|host]; each synchronises the stream before returning.
 * get_prims: 8 padded cell-centred arrays incl. filled ghosts (rho,v^i,p,B^i centred).
 * get_cons : 8 padded cell-centred arrays, UNdensitised D, S_x, S_y, S_z, tau, B^x, B^y, B^z;
 *            interior cells only, ghost cells are set to 0.
 * get_vecpot: 3 staggered arrays incl. filled ghosts. */
int grmhd_get_prims(grmhd* h, double* const field[8]);
int grmhd_get_cons(grmhd* h, double* const field[8]);
int grmhd_get_vecpot(grmhd* h, double* const field[3]);
/* Psi_mhd = sqrt(gamma) Phi of the generalised Lorenz gauge: one staggered-shape
 * array, vertex (i,j,k) = (i-1/2, j-1/2, k-1/2), incl. filled ghosts; zero in the algebraic gauge. */
int grmhd_get_psi(grmhd* h, double* field);

/* Keys: "fixed_dt" (> 0: use this dt instead of the CFL reduction; 0 = off);
 * "gauge" (0 default: algebraic gauge, d_t A_i = -E_i; 1: generalised Lorenz gauge,
 * eqs (31)-(32) PAPER.md:212-227, Psi_mhd on the vertices as a ninth evolved component; B is
 * the same in both to round-off), "lorenz_xi" (xi = lorenz_xi / dt, default 1.5);
 * "emf" (0 default: electric field on the edges by flux-CT, R10; 1: upwind constrained
 * transport, eqs (33)-(35) PAPER.md:229-250 -- the flux kernels then also store a_+, a_- and the
 * upwind transverse velocities of every face on a 3-cell transverse apron, and the edges are
 * updated by their own kernel);
 * "uct_passes" (1 default: the upwind-CT edges per reconstruction axis, each parabola once; 0: one
 * thread per edge), "uct_nseg" (segments of the marching passes, default 16);
 * "c2p_backup" (1: when the 2-D Newton con2prim fails, try the 1-D scheme of PAPER.md:297-320,
 * eqs (42)-(45), before resetting the cell to atmosphere -- the paper's policy, PAPER.md:684;
 * 0 = off, the default: failure -> atmosphere, G20);
 * "flux_kernel" (1 default: y and z fluxes by the TMA-fed marching kernel, x fluxes with the lanes
 * of a warp along x; 0: lanes along the flux direction in all three directions -- what blocks
 * narrower than 32 cells in x use anyway);
 * "flux_xcol" (1 default: with flux-CT the two apron columns x = -1 and x = nx of the y and z
 * fluxes are computed from compact, contiguous copies of those columns -- the static face metric
 * copied once per grmhd_set_metric, the primitives and B once per substep -- and only the flux row
 * flux-CT reads there is stored; 0: straight from the padded arrays, where consecutive cells of a
 * column are a row pitch apart -- bit-identical results);
 * "src_kernel" (1 default: the metric-derivative stencils of the source terms in x and y from a
 * TMA-staged shared-memory tile; 0: plain loads -- bit-identical results);
 * "small_fuse" (1 default: blocks of at most 2^16 padded cells, where a step is bound by kernel
 * launches, run the x, y and z fluxes in one launch, the three ghost-fill passes of A_i in one
 * launch of a thread-block cluster, and the source terms and t += dt inside the post-update
 * kernel -- 11 instead of 26 launches per RK2 step; 0: the kernel sequence of large blocks);
 * "graph" (1 default: after one eager step the launch sequence of a step is captured into a
 * CUDA graph and every later step is one cudaGraphLaunch into the handle's stream -- same
 * kernels, same arguments, bit-identical results; any other option or grmhd_set_mask drops the
 * graph; bypassed while "kernel_timing" is on; 0: always launch kernel by kernel);
 * "kernel_timing" (1: bracket every kernel group of the step with CUDA events on the
 * handle's stream and accumulate device times, see grmhd_get_kernel_times; 0 = off;
 * setting it clears the accumulators).  Unknown key -> EINVAL. */
int grmhd_set_option(grmhd* h, const char* key, double value);

/* Synchronises and copies the counters.  Returns ENUMERIC if any dt was not finite/positive. */
int grmhd_get_stats(grmhd* h, grmhd_stats* out);

/* Device time per kernel group since "kernel_timing" was switched on (measurement aid for
 * the roofline report; synchronises).  Groups: 0 flux-x, 1 flux-y, 2 flux-z (A3+A4),
 * 3 divergence + flux-CT + RK update (A5-A7), 4 A_i ghost fill (A1),
 * 5 B from A + con2prim (A6, A2, +A8 on the last stage), 6 primitive ghost fill (A1),
 * 7 dt scalars, 8 metric source terms (A5, eq. 19).
 * ms[q] = summed milliseconds, launches[q] = number of timed brackets. */
#define GRMHD_NKGROUPS 9
int grmhd_get_kernel_times(grmhd* h, double ms[GRMHD_NKGROUPS],
                           long long launches[GRMHD_NKGROUPS]);

/* Number of kernels this handle has launched so far (host-side counter). */
long long grmhd_launch_count(const grmhd* h);

const char* grmhd_last_error(const grmhd* h);

/* ---- stand-alone kernels exposed for unit parity tests and micro-benchmarks ---------
 * Pointwise batches on plain [dev] arrays of n states, structure-of-arrays, each array n long.
 * prim: 8 arrays rho,vx,vy,vz,p,Bx,By,Bz; metric: 10 arrays alpha,beta^i(3),gamma_ij(6);
 * cons: 8 arrays UNdensitised D,S_x,S_y,S_z,tau,B^x,B^y,B^z. */
int grmhd_prim2con_batch(const double* const prim[8], const double* const metric[10],
                         double* const cons[8], long long n, const grmhd_opts* opts,
                         void* stream);
/* cons in (5 hydro rows + 3 B rows) -> prim out (5), status out (int32 per state: bit0
 * atmosphere, bit1 c2p failure, bit2 pressure fix, bit3 W cap), iterations (int32). */
int grmhd_con2prim_batch(const double* const cons[8], const double* const metric[10],
                         double* const prim[5], int* status, int* iters, long long n,
                         const grmhd_opts* opts, void* stream);
/* The 1-D scheme alone (eqs 42-45; Brent's method on x = hW): prim out =
 * rho, v^i, p = (Gamma-1) rho eps without floors; status 0 = converged, 2 = no bracket / no
 * convergence; iters = Brent iterations. */
int grmhd_con2prim1d_batch(const double* const cons[8], const double* const metric[10],
                           double* const prim[5], int* status, int* iters, long long n,
                           const grmhd_opts* opts, void* stream);
/* Dependent-free DFMA loop used to MEASURE the FP64 pipe peak: each of `threads` threads
 * performs `iters` * 16 DFMAs; out receives one double per thread.  */
int grmhd_dfma_peak(double* out, long long threads, int iters, void* stream);

/* ---- the max-speed reduction with NO allocation ---------------------------------------
 * For callers that cannot call cudaMalloc or hold a workspace (code under CUDA-graph capture,
 * tight serving loops, harnesses that forbid allocation): the max-characteristic-speed reduction
 * of the CFL step (north_star "max-characteristic-speed reduction for the CFL dt"; speeds:
 * PAPER.md:199, R16 / G9) on n plain states, structure of arrays as above:
 *   prim   [dev] 8 arrays rho, v^x, v^y, v^z, p, B^x, B^y, B^z (cell-centred values), n each;
 *   metric [dev] 10 arrays alpha, beta^i (3), gamma_ij (6), n each;
 *   maxspeed [dev] 3 doubles OUT: max over the states of max(|lambda_-|, |lambda_+|) along
 *            x, y, z -- what grmhd_get_stats reports as maxspeed for the cells of a handle
 *            (dt = cfl * min_d dx_d / maxspeed[d]).  A NaN speed never wins the max.
 * The call enqueues one memset and one kernel on `stream` and returns; it allocates nothing and
 * calls no allocating routine.  Its scratch (one partial maximum per 256 states) is a file-scope
 * __device__ array of 384.25 KiB that every GPU loading the library holds until the process
 * exits; hence the limit  1 <= n <= GRMHD_NOALLOC_MAX_STATES: a larger n returns GRMHD_ELIMIT
 * (split the batch and take the max of the results).  Every call on a device shares that
 * array: calls that overlap on the GPU (different streams or threads) RACE -- serialise them.
 * err/err_len: optional buffer for a human-readable message (there is no handle to keep one);
 * may be NULL/0.  Other errors: GRMHD_EINVAL (NULL array, n < 1, bad options), GRMHD_ECUDA. */
#define GRMHD_NOALLOC_MAX_STATES 4194304LL /* 2^22 */
int grmhd_maxspeed_noalloc(const double* const prim[8], const double* const metric[10],
                           long long n, const grmhd_opts* opts, double* maxspeed, void* stream,
                           char* err, size_t err_len);

#ifdef __cplusplus
}
#endif
#endif /* GRMHD_H */

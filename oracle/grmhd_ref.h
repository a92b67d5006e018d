/* grmhd_ref.h -- C ABI of the ORACLE (libgrmhd_ref.so).
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  A plain, slow, obviously-correct fp64 CPU
 * implementation of the discretisation written from PAPER.md (arXiv 2406.11669) and the
 * readings listed in DESIGN.md.  It shares no code, header, table or helper with the CUDA
 * library (paper_2406_11669_b200/csrc); only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.  All pointers are HOST pointers.
 *
 * Array layouts are those of the problem statement: cell-centred padded arrays of shape
 * (nz+2g, ny+2g, nx+2g), staggered arrays (nz+2g+1, ny+2g+1, nx+2g+1), x fastest, g = 3,
 * lower-face / lower-edge convention.
 */
#ifndef GRMHD_REF_H
#define GRMHD_REF_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct ref_grmhd ref_grmhd;

typedef struct {
  double gamma_ad, poly_k, poly_gamma, rho_atm, p_floor, w_max, c2p_tol;
  int c2p_maxit, recon, ppm_flatten, riemann, rk;
  int bc[3];
} ref_opts;

typedef struct {
  double t, dt, maxspeed[3];
  long long steps, c2p_fail, p_fix, atmo, w_cap, c2p_maxiter;
  long long c2p_backup; /* states recovered by the 1-D backup scheme (option "c2p_backup") */
} ref_stats;

int ref_create(int nx, int ny, int nz, int ghosts, const double dx[3], const ref_opts* o,
               ref_grmhd** out);
int ref_destroy(ref_grmhd* h);
int ref_set_metric(ref_grmhd* h, const double* const field[16]);
int ref_set_prims(ref_grmhd* h, const double* const field[8]);
int ref_set_vecpot(ref_grmhd* h, const double* const field[3]);
int ref_set_mask(ref_grmhd* h, const unsigned char* mask);
int ref_step(ref_grmhd* h, int n, double cfl);
int ref_step_until(ref_grmhd* h, double t_end, double cfl, int* nsteps_done);
int ref_get_prims(ref_grmhd* h, double* const field[8]);
int ref_get_cons(ref_grmhd* h, double* const field[8]);
int ref_get_vecpot(ref_grmhd* h, double* const field[3]);
int ref_get_psi(ref_grmhd* h, double* field); /* Psi_mhd on vertices (staggered shape), option "gauge" = 1 */
int ref_set_option(ref_grmhd* h, const char* key, double value);
int ref_get_stats(ref_grmhd* h, ref_stats* out);
void ref_set_num_threads(int n); /* OpenMP threads for the cell loops (1 = the oracle proper) */
int ref_get_num_threads(void);

/* ---- pieces exposed so that tests can pin them one by one ------------------------- */
/* L(Y) of the CURRENT state: 5 cell-centred padded arrays (d/dt of densitised D,S_j,tau;
 * interior cells, 0 elsewhere) and 3 staggered arrays (d/dt A_i = -E_i; edges bounding an
 * interior face, 0 elsewhere). */
int ref_rhs(ref_grmhd* h, double* const dU[5], double* const dA[3]);
/* d/dt A_i including the gauge term of eq. (31) and d/dt Psi_mhd of eq. (32) (option "gauge");
 * xi = lorenz_xi / (dt of the last step), 0 before the first step */
int ref_rhs_gauge(ref_grmhd* h, double* const dA[3], double* dPsi);
/* stored numerical fluxes of the current state: flux[d][r], d = direction, r = 0..7 rows
 * (D,S_x,S_y,S_z,tau,B^x,B^y,B^z), staggered-shape arrays, densitised F~ = sqrt(gamma_f) F^ */
int ref_fluxes(ref_grmhd* h, double* const flux[24]);
/* densitised face field B~^d (3 staggered-shape arrays) */
int ref_get_bface(ref_grmhd* h, double* const field[3]);

/* point functions: prim = rho,vx,vy,vz,p,Bx,By,Bz; metric = alpha,beta^x..z,gxx,gxy,gxz,gyy,gyz,gzz */
void ref_prim2con_pt(const double prim[8], const double metric[10], double gamma_ad,
                     double cons[8]); /* undensitised D,S_j,tau,B^k, eqs (20)-(22) */
/* returns status bits (1 atmosphere, 2 failure, 4 pressure fix, 8 W cap); cons_out = the
 * (possibly rewritten) undensitised D,S_j,tau */
int ref_con2prim_pt(const double cons[8], const double metric[10], const ref_opts* o,
                    int masked, double prim_out[5], double cons_out[5], int* iters);
/* as ref_con2prim_pt with the 1-D backup enabled (status bit 16 = recovered by the backup) */
int ref_con2prim_backup_pt(const double cons[8], const double metric[10], const ref_opts* o,
                           double prim_out[5], double cons_out[5], int* iters);
/* the 1-D scheme alone, eqs (42)-(45) PAPER.md:297-320: prim_out = rho, v^i, p without floors;
 * returns 0 or 2 (no bracket / no convergence); iters = Brent iterations */
int ref_con2prim1d_pt(const double cons[8], const double metric[10], const ref_opts* o,
                      double prim_out[5], int* iters);
/* out = W^ of eq. (44), eps^ of eq. (45), f of eq. (43) at a given x */
void ref_c2p1d_relations_pt(const double cons[8], const double metric[10], const ref_opts* o,
                            double x, double out[3]);
void ref_flux_pt(int d, const double prim[8], const double metric[10], double gamma_ad,
                 double F[8]); /* eq. (18), including its 1/alpha */
void ref_speeds_pt(int d, const double prim[8], const double metric[10], double gamma_ad,
                   double lam[2]); /* lambda_-, lambda_+ (R6) */
void ref_riemann_pt(int d, const double primL[8], const double primR[8],
                    const double metric_face[10], const ref_opts* o,
                    double Fhat[8]); /* undensitised F^ of eq. (29)/(30) incl. face floors */
/* sources S of eq. (19) in 3+1 form: dalpha[j], dbeta[j][i]=d_j beta^i, dgam[j][6]=d_j gamma_kl,
 * K[6]; out S[5] for (D,S_x,S_y,S_z,tau) */
void ref_source_pt(const double prim[8], const double metric[10], const double K[6],
                   const double dalpha[3], const double dbeta[9], const double dgam[18],
                   double gamma_ad, double S[5]);
/* reconstruct one variable along a line of n cells: faces f = 3..n-3 get qL[f] (from cell
 * f-1) and qR[f] (from cell f); press/vnorm feed the PPM flattening (may be NULL when
 * method = 0 or flatten = 0). */
void ref_recon_line(int method, int flatten, int n, const double* q, const double* press,
                    const double* vnorm, double* qL, double* qR);
#ifdef __cplusplus
}
#endif
#endif

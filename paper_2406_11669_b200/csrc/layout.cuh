// layout.cuh -- data layout of a handle in HBM.
//
// One block of nx*ny*nz cells with G = 3 ghost layers.  Every field, cell
// centred or staggered, lives in an array of the same padded extent (PZ, PY, PXP), x
// fastest, structure-of-arrays, fields back to back at a stride of NPA doubles:
//   PXP = roundup(nx + 8, 4)   x pitch: rows are whole 32-byte sectors; cell i = 0 sits at
//                              x index X0 = 4 so interior rows start sector aligned
//   PY  = ny + 7, PZ = nz + 7  (room for the staggered index n + G)
// Staggered fields use the LOWER convention: index (i,j,k) of A_z is the
// edge (i-1/2, j-1/2, k), of a d-face field the face i_d - 1/2.
#pragma once
#include <cstddef>
#include <cstdint>

namespace gk {

constexpr int G = 3;
constexpr int X0 = 4;

struct Geom {
  int nx, ny, nz;
  int PXP, PY, PZ;
  long long sy, sz;  // strides of j and k
  long long NP;      // PXP*PY*PZ
  long long NPA;     // field stride (NP rounded up to 32 doubles = 256 B)
  double dx[3], idx[3];
  int bc[3];

  __host__ __device__ long long at(int i, int j, int k) const {
    return (long long)(k + G) * sz + (long long)(j + G) * sy + (i + X0);
  }
  __host__ __device__ int n(int a) const { return a == 0 ? nx : (a == 1 ? ny : nz); }
  __host__ __device__ long long stride(int a) const { return a == 0 ? 1 : (a == 1 ? sy : sz); }
};

// field ids (units of NPA doubles from the workspace base)
enum FieldId {
  F_MET = 0,    // 16: alpha, beta^i, gamma_ij (6), K_ij (6)
  F_P = 16,     // 5 : rho, v^x, v^y, v^z, p                        cell centres
  F_BC = 21,    // 3 : Eulerian B^i at cell centres
  F_BF = 24,    // 3 : densitised B~^d on d-faces (total)
  F_B0 = 27,    // 3 : static part B~0 (G16)
  F_Y = 30,     // 9 : evolved D~, S~_j, tau~ (cells), A_i (edges), Psi_mhd (vertices, Lorenz gauge)
  F_Y0 = 39,    // 9 : RK register Y^0
  F_FX = 48,    // 7 : stored x-fluxes: D,S_x,S_y,S_z,tau rows + B^y, B^z rows
  F_FY = 55,    // 7 : y-fluxes (+ B^z, B^x rows)
  F_FZ = 62,    // 7 : z-fluxes (+ B^x, B^y rows)
  F_SRC = 69,   // 4 : alpha sqrt(gamma) S of eq. (19) for the rows S_x, S_y, S_z, tau (cells)
  F_W = 73,     // 12: upwind-CT face data, 4 per direction d: a_+, a_- (eq. 34) and the upwind
                //     transverse velocities vbar^{(d+1)%3}, vbar^{(d+2)%3} (eq. 33); F_W + 4 d + r
  F_GV = 85,    // 5 : Lorenz gauge, on vertices: G_A (eq. 31), F_Psi^x,y,z (eq. 32), alpha
  F_FM = 90,    // 33: STATIC face metric, 11 per direction d (the ADM variables are held fixed,
                //     PAPER.md:61, so the 4-point Lagrange values of R4 are formed once, in
                //     grmhd_set_metric): F_FM + 11 d + {alpha, beta^x, beta^y, beta^z, gamma_xx,
                //     gamma_xy, gamma_xz, gamma_yy, gamma_yz, gamma_zz, sqrt(gamma)} on the lower
                //     d-face of the index
  F_KS = 123,   // 9 : RK4 accumulator k1 + 2 k2 + 2 k3 (only allocated when rk = 4)
  F_END_RK23 = 123,
  F_END_RK4 = 132
};
constexpr int NFM = 11;  // static face-metric fields per direction

// device-resident scalars of a handle
struct DevState {
  double t, dt;
  double cfl, fixed_dt, t_end;       // inputs of the dt kernel (t_end < 0: no clipping)
  unsigned long long ms_acc[3];      // bit patterns of max |lambda| per direction (A8)
  double ms_used[3];                 // speeds the last dt was computed from
  long long c2p_fail, p_fix, atmo, w_cap, c2p_maxiter;
  long long c2p_backup;              // states recovered by the 1-D backup scheme
  int bad_dt;
  int pad;
};

}  // namespace gk

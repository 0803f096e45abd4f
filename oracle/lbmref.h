/* oracle/lbmref.h — C interface of the CPU ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, single-threaded fp64 restatement of the per-time-step update of the 2-D (D2Q9)
 * color-gradient lattice Boltzmann model with the ghost-node wetting boundary condition of
 * arxiv/paper_2605_30878 (§II Eq. 4-9, §III :100, App. A Eq. A1-A17).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * call this.  It shares no code with the CUDA path (paper_2605_30878_b200/csrc) and neither
 * includes the other's headers.  Every function cites the passage it follows in lbmref.c.
 *
 * Conventions: node (i,j) at position (x,y)=(i,j); idx = j*nx + i;
 * periodic in both directions; walls are rows of solid nodes inside the array; dx = dt = 1;
 * c_s^2 = 1/3; direction order of Eq. A5.
 */
#ifndef LBMREF_H
#define LBMREF_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lbmref_ctx lbmref_ctx;

typedef struct { double cx, cy, r; } lbmref_disk;   /* closed disk, periodic images */

typedef struct {
  int32_t nx, ny;
  double  rho_l, rho_g;     /* phase densities                                  */
  double  nu_l, nu_g;       /* kinematic viscosities; tau = 1/2 + 3 nu         */
  double  sigma, W;         /* surface tension, interface width (Eq. 4, Eq. 5)                */
  double  theta_deg;        /* equilibrium contact angle measured in the liquid */
  double  mobility;         /* M_phi at reference p = 0 -> alpha = 1 - 10 M_phi/3 */
  double  gx, gy;           /* body acceleration, F_b = rho g (Eq. 2)                         */
  int32_t wall_rows;        /* 1: rows j=0 and j=ny-1 are flat walls (must be solid in mask)  */
  int32_t ghost_rule;       /* 0: Eq. 9 (paper); 1: Eq. 10 (Fakhari-Bolster half-way)         */
  int32_t picard;           /* passes of the local (u,p,F) fixed point; 1 = the definition (R9) */
} lbmref_params;

/* class codes (Fig. 1) */
enum { LBMREF_FLUID_BULK = 0, LBMREF_FLUID_BOUNDARY = 1, LBMREF_GHOST = 2, LBMREF_SOLID_BULK = 3 };

/* derived per-node quantities, for tests */
typedef struct {
  double phi, gradx, grady, lap;
  double rho, tau;
  double Fsx, Fsy, Fx, Fy;     /* surface tension force; total F_macro */
  double ux, uy, p;
} lbmref_node_fields;

int  lbmref_create(lbmref_ctx** out, const lbmref_params* prm, const uint8_t* mask,
                   const lbmref_disk* disks, int32_t n_disks);
int  lbmref_init(lbmref_ctx* c, const double* phi0, const double* u0);
int  lbmref_step(lbmref_ctx* c, int64_t n);
int  lbmref_get(lbmref_ctx* c, double* rho, double* phi, double* ux, double* uy, double* p);
int  lbmref_get_populations(lbmref_ctx* c, double* N, double* B);
int  lbmref_set_populations(lbmref_ctx* c, const double* N, const double* B);
int  lbmref_get_classification(lbmref_ctx* c, uint8_t* cls, int32_t* n_ghost, int32_t* ghost_idx,
                               double* ghost_nx, double* ghost_ny, double* ghost_depth,
                               int32_t* ghost_corner, double* ghost_wgt);
int  lbmref_get_phi_raw(lbmref_ctx* c, double* phi);  /* stored phi array incl. ghost values */
int  lbmref_diag(lbmref_ctx* c, double out[8]);
const char* lbmref_last_error(const lbmref_ctx* c);
void lbmref_destroy(lbmref_ctx* c);

/* ---- pieces exposed so that tests can pin them one by one ---- */
void   lbmref_lattice(int32_t cx[9], int32_t cy[9], int32_t opp[9], double w[9]);
void   lbmref_matrices(double M[81], double Minv[81]);
double lbmref_alpha_from_mobility(double mobility);
void   lbmref_chi(double alpha, double chi[9]);
double lbmref_ghost_rule(double phiF, double eps, int32_t rule);         /* Eq. 9 / Eq. 10 */
void   lbmref_neq(double alpha, double p, double ux, double uy, double out[9]);  /* Eq. A4 */
double lbmref_pressure(double alpha, const double N[9], double ux, double uy);   /* Eq. A15 */
void   lbmref_gradients(const double phi_nb[9], double* gx, double* gy, double* lap);
void   lbmref_bilinear_setup(double xF, double yF, int32_t nx, int32_t ny,
                             int32_t corner[4], double wgt[4]);
/* full local update of one fluid node: phi_nb[i] = phi(x + c_i), phi_nb[0] = phi(x) */
void   lbmref_node_update(const lbmref_params* prm, const double N[9], const double phi_nb[9],
                          double Nstar[9], double Bstar[9], lbmref_node_fields* f);

/* NEXT row f2: unit solid normal from the mask alone (indicator smoothed twice, sixth-order isotropic stencil) */
void lbmref_mask_smooth(const int32_t* in, int32_t* out, int nx, int ny);
void lbmref_mask_normal(const int32_t* s, int nx, int ny, int i, int j, double* nxs, double* nys);

#ifdef __cplusplus
}
#endif
#endif

/* oracle/lbmref.c — the CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded fp64 implementation of what the hot path computes, written from
 * PAPER.md alone, step by step in the paper's order and notation.  No blocking, no fusion, generic
 * 9x9 matrix form of the collision (Eq. A1).  It shares no code with the CUDA path.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference may use it.
 *
 * Passages followed: §II Eq. 4-9, defaults and ghost initialisation (:100),
 * App. A Eq. A1-A17 (:260-322).  Where the paper is silent or garbled the readings R1..R23 of
 * DESIGN.md ("Readings of the paper") are taken; each is named where it is used.
 *
 * Parity pins: tests/test_oracle_*.py (algebraic identities, closed forms, brute force,
 * conservation, Laplace law at density ratio 1 and 1000, contact angle on a cylinder, single-phase
 * and two-layer Poiseuille, rotational covariance of the node's force).  The correction forces
 * F_visc (A11, R10), F_p (A10) and the harmonic viscosity rule (R6) are pinned by
 * tests/test_oracle_forces.py, which also measures the mobility of the color equation (R5).
 * Conventions that no independent fact fixes stay "parity unpinned": R9 (one Picard pass rather than
 * a converged iteration), R14 (no anti-diffusion part in the initial B_i; the moments of the initial
 * state are pinned), R15 (plain bilinear interpolation whatever the corner's class).
 *
 * Build: gcc -O2 -ffp-contract=off -fPIC -shared -o liblbmref.so lbmref.c -lm
 */
#include "lbmref.h"
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

/* ---- D2Q9 lattice, Eq. A5-A6 ---------------------------------------- */
static const int CX[9] = {0, 1, 0, -1, 0, 1, -1, -1, 1};
static const int CY[9] = {0, 0, 1, 0, -1, 1, 1, -1, -1};
static const int OPP[9] = {0, 3, 4, 1, 2, 7, 8, 5, 6};
static const double WGT[9] = {4.0 / 9.0, 1.0 / 9.0, 1.0 / 9.0, 1.0 / 9.0, 1.0 / 9.0,
                              1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0};
#define CS2 (1.0 / 3.0)

/* Transformation matrix, Eq. A2.  Row 2 prints ten entries in the extracted
 * text; reading R1 takes the standard (-4,-1,-1,-1,-1,2,2,2,2), which makes all rows mutually
 * orthogonal (pinned in tests). */
static const double MMAT[9][9] = {
    {1, 1, 1, 1, 1, 1, 1, 1, 1},
    {-4, -1, -1, -1, -1, 2, 2, 2, 2},
    {4, -2, -2, -2, -2, 1, 1, 1, 1},
    {0, 1, 0, -1, 0, 1, -1, -1, 1},
    {0, -2, 0, 2, 0, 1, -1, -1, 1},
    {0, 0, 1, 0, -1, 1, 1, -1, -1},
    {0, 0, -2, 0, 2, 1, 1, -1, -1},
    {0, 1, -1, 1, -1, 0, 0, 0, 0},
    {0, 0, 0, 0, 0, 1, -1, 1, -1}};

/* Solid normal from the mask alone (NEXT row f2; "smooth solid normals can be obtained
 * with numerical stencils that preserve isotropy of the gradient operator up to sixth order").
 * Stencil: the 12 points |c|^2 = 1, 2, 4 with weights 4/15, 1/10, 1/120 (sixth-order isotropic; x120:
 * 32, 12, 1, so every sum is an exact integer).  The solid indicator s (1 on solid nodes) is smoothed
 * twice with these weights plus a centre weight 60/120 (the raw staircase gives normals that are off
 * by up to 34 degrees on a disk of radius 40; two passes: 13 degrees max, 3 degrees mean), then
 * n_s = -grad(s~)/|grad(s~)|, (0,0) if the gradient vanishes.  Periodic wrap. */
static const int MN_OX[12] = {1, 0, -1, 0, 1, -1, -1, 1, 2, 0, -2, 0};
static const int MN_OY[12] = {0, 1, 0, -1, 1, 1, -1, -1, 0, 2, 0, -2};
static const int MN_WG[12] = {32, 32, 32, 32, 12, 12, 12, 12, 1, 1, 1, 1};

void lbmref_mask_smooth(const int32_t* in, int32_t* out, int nx, int ny) {
  for (int j = 0; j < ny; j++)
    for (int i = 0; i < nx; i++) {
      int32_t acc = 60 * in[j * nx + i];
      for (int k = 0; k < 12; k++) {
        int ii = ((i + MN_OX[k]) % nx + nx) % nx, jj = ((j + MN_OY[k]) % ny + ny) % ny;
        acc += MN_WG[k] * in[jj * nx + ii];
      }
      out[j * nx + i] = acc;
    }
}

void lbmref_mask_normal(const int32_t* s, int nx, int ny, int i, int j, double* nxs, double* nys) {
  long gx = 0, gy = 0;
  for (int k = 0; k < 12; k++) {
    int ii = ((i + MN_OX[k]) % nx + nx) % nx, jj = ((j + MN_OY[k]) % ny + ny) % ny;
    gx += (long)MN_WG[k] * MN_OX[k] * s[jj * nx + ii];
    gy += (long)MN_WG[k] * MN_OY[k] * s[jj * nx + ii];
  }
  double ax = -(double)gx, ay = -(double)gy;
  double m = sqrt(ax * ax + ay * ay);
  if (m > 0.0) { *nxs = ax / m; *nys = ay / m; }
  else { *nxs = 0.0; *nys = 0.0; }
}

struct lbmref_ctx {
  lbmref_params P;
  int n;
  uint8_t* solid;   /* copy of the mask, 1 = solid */
  uint8_t* cls;
  int n_ghost;
  int32_t* g_idx;
  double *g_nx, *g_ny, *g_depth;
  int32_t* g_corner; /* 4 per ghost */
  double* g_wgt;     /* 4 per ghost */
  double* g_new;     /* Jacobi staging */
  double *N, *B, *N2, *B2; /* SoA: pop[i*n + idx] */
  double* phi;
  double* scratch;
  int64_t t;
  char err[256];
};

enum { OK = 0, EINVAL_ = -1, ENOMEM_ = -2 };

/* ---- small exported pieces --------------------------------------------------------------- */
void lbmref_lattice(int32_t cx[9], int32_t cy[9], int32_t opp[9], double w[9]) {
  for (int i = 0; i < 9; i++) { cx[i] = CX[i]; cy[i] = CY[i]; opp[i] = OPP[i]; w[i] = WGT[i]; }
}

/* M of Eq. A2 and M^-1 = M^T diag(1/|row|^2) (rows are orthogonal, R1). */
void lbmref_matrices(double M[81], double Minv[81]) {
  for (int k = 0; k < 9; k++) {
    double nrm = 0.0;
    for (int i = 0; i < 9; i++) nrm += MMAT[k][i] * MMAT[k][i];
    for (int i = 0; i < 9; i++) {
      M[k * 9 + i] = MMAT[k][i];
      Minv[i * 9 + k] = MMAT[k][i] / nrm;
    }
  }
}

/* Eq. A7 text: M_phi = (c_s^2 dt/2)[9(1-alpha)/5 + p/c_s^2]; reading R5 takes the
 * reference pressure p = 0, so alpha = 1 - 10 M_phi / 3. */
double lbmref_alpha_from_mobility(double mobility) { return 1.0 - 10.0 * mobility / 3.0; }

/* Color weights, Eq. A7. */
void lbmref_chi(double alpha, double chi[9]) {
  chi[0] = alpha;
  for (int i = 1; i <= 4; i++) chi[i] = (1.0 - alpha) / 5.0;
  for (int i = 5; i <= 8; i++) chi[i] = (1.0 - alpha) / 20.0;
}

/* Ghost-node rule.  rule 0: Eq. 9, phi_G = phi_F / (phi_F + (1-phi_F) e^eps).
 * rule 1: Eq. 10, Fakhari-Bolster with the wall half-way; "special care" at
 * eps -> 0: the first-order series phi_F - eps phi_F (1-phi_F), common to both
 * rules, is used for |eps| < 1e-8. */
double lbmref_ghost_rule(double phiF, double eps, int32_t rule) {
  if (rule == 0) return phiF / (phiF + (1.0 - phiF) * exp(eps));
  {
    /* Eq. 10: phi_G = (2/eps) (a - sqrt(a^2 - 2 eps phi_F)) - phi_F, a = 1 + eps/2.  As
     * printed it is 0/0 at theta = 90 deg (eps = 0, "special care", :87) and loses digits near it; with
     * a - s = (a^2 - s^2)/(a + s) = 2 eps phi_F/(a + s) the same expression has no cancellation and
     * no singular point. */
    double a = 1.0 + 0.5 * eps;
    return 4.0 * phiF / (a + sqrt(a * a - 2.0 * eps * phiF)) - phiF;
  }
}

/* Color-blind equilibrium, Eq. A4, with the i = 0 branch read as
 * chi_0 - (1-w_0) p/c_s^2 - w_0 u^2/(2 c_s^2) (R4). */
void lbmref_neq(double alpha, double p, double ux, double uy, double out[9]) {
  double chi[9];
  double u2 = ux * ux + uy * uy;
  lbmref_chi(alpha, chi);
  out[0] = chi[0] - (1.0 - WGT[0]) * p / CS2 - WGT[0] * u2 / (2.0 * CS2);
  for (int i = 1; i < 9; i++) {
    double cu = CX[i] * ux + CY[i] * uy;
    out[i] = chi[i] + WGT[i] * (p / CS2 + cu / CS2 + cu * cu / (2.0 * CS2 * CS2) - u2 / (2.0 * CS2));
  }
}

/* Auxiliary pressure, Eq. A15. */
double lbmref_pressure(double alpha, const double N[9], double ux, double uy) {
  double s = 0.0;
  for (int i = 1; i < 9; i++) s += N[i];
  return (-(WGT[0] / 2.0) * (ux * ux + uy * uy) - (1.0 - alpha) * CS2 + s * CS2) / (1.0 - WGT[0]);
}

/* Isotropic second-order D2Q9 stencils (R8): grad = 3 sum w_i c_i phi(x+c_i),
 * lap = 6 sum w_i [phi(x+c_i) - phi(x)].  The paper needs grad phi and lap phi (Eq. 4,
 * PAPER.md:45) but does not print the stencil. */
void lbmref_gradients(const double phi_nb[9], double* gx, double* gy, double* lap) {
  double sx = 0.0, sy = 0.0, sl = 0.0;
  for (int i = 1; i < 9; i++) {
    sx += WGT[i] * CX[i] * phi_nb[i];
    sy += WGT[i] * CY[i] * phi_nb[i];
    sl += WGT[i] * (phi_nb[i] - phi_nb[0]);
  }
  *gx = 3.0 * sx;
  *gy = 3.0 * sy;
  *lap = 6.0 * sl;
}

static int wrapi(int a, int n) {
  a %= n;
  return a < 0 ? a + n : a;
}

/* Bilinear interpolation stencil of the point x_F ("phi_F is obtained from bilinear
 * interpolation"): cell origin (floor x, floor y), periodic wrap of the four corners. */
void lbmref_bilinear_setup(double xF, double yF, int32_t nx, int32_t ny, int32_t corner[4],
                           double wgt[4]) {
  double fi = floor(xF), fj = floor(yF);
  double fx = xF - fi, fy = yF - fj;
  int i0 = wrapi((int)fi, nx), j0 = wrapi((int)fj, ny);
  int i1 = wrapi(i0 + 1, nx), j1 = wrapi(j0 + 1, ny);
  corner[0] = j0 * nx + i0; wgt[0] = (1.0 - fx) * (1.0 - fy);
  corner[1] = j0 * nx + i1; wgt[1] = fx * (1.0 - fy);
  corner[2] = j1 * nx + i0; wgt[2] = (1.0 - fx) * fy;
  corner[3] = j1 * nx + i1; wgt[3] = fx * fy;
}

/* ---- the local update of one fluid node: step 3 of the time step ------------------------- */
void lbmref_node_update(const lbmref_params* P, const double N[9], const double phi_nb[9],
                        double Nstar[9], double Bstar[9], lbmref_node_fields* f) {
  double M[81], Minv[81], chi[9];
  double alpha = lbmref_alpha_from_mobility(P->mobility);
  double phi = phi_nb[0];
  double gx, gy, lap;
  lbmref_matrices(M, Minv);
  lbmref_chi(alpha, chi);

  /* gradients (R8) */
  lbmref_gradients(phi_nb, &gx, &gy, &lap);

  /* mixture rules: rho linear in phi, 1/nu harmonic in the kinematic viscosity;
   * tau = 1/2 + nu/(dt c_s^2). */
  double rho = P->rho_l * phi + P->rho_g * (1.0 - phi);
  double drx = (P->rho_l - P->rho_g) * gx, dry = (P->rho_l - P->rho_g) * gy;
  double nu = 1.0 / (phi / P->nu_l + (1.0 - phi) / P->nu_g);
  double tau = 0.5 + nu / CS2;

  /* surface tension force, Eq. 4 */
  double mu = -P->sigma * ((48.0 / P->W) * phi * (1.0 - phi) * (phi - 0.5) + (3.0 * P->W / 2.0) * lap);
  double Fsx = mu * gx, Fsy = mu * gy;
  /* body force rho g, Eq. 2 */
  double Fbx = rho * P->gx, Fby = rho * P->gy;

  /* raw moments of N */
  double jx = 0.0, jy = 0.0, m7 = 0.0, m8 = 0.0;
  for (int i = 0; i < 9; i++) {
    jx += N[i] * CX[i];
    jy += N[i] * CY[i];
    m7 += N[i] * (CX[i] * CX[i] - CY[i] * CY[i]);
    m8 += N[i] * (CX[i] * CY[i]);
  }

  /* u, p, F_p, F_visc are mutually implicit (A10, A11, A14, A15).  Reading R9: local Picard
   * passes started from u0 = j + (F_s + F_b)/(2 rho); `picard` = 1 is the definition.
   * Reading R10: (grad u + grad u^T) = -Pi^neq_dev / (tau c_s^2), trace dropped (Eq. 1), so
   * F_visc (A11) = -((tau-1/2)/tau) Pi^neq_dev . grad rho. */
  double ux = jx + (Fsx + Fbx) / (2.0 * rho);
  double uy = jy + (Fsy + Fby) / (2.0 * rho);
  double p = lbmref_pressure(alpha, N, ux, uy);
  double Fx = Fsx + Fbx, Fy = Fsy + Fby;
  int K = P->picard < 1 ? 1 : P->picard;
  for (int k = 0; k < K; k++) {
    double m7n = m7 - (ux * ux - uy * uy);
    double m8n = m8 - ux * uy;
    double cv = -(tau - 0.5) / tau;
    double Fvx = cv * (0.5 * m7n * drx + m8n * dry);
    double Fvy = cv * (m8n * drx - 0.5 * m7n * dry);
    double Fpx = -p * drx, Fpy = -p * dry;              /* A10 */
    Fx = Fsx + Fbx + Fpx + Fvx;                          /* A9 */
    Fy = Fsy + Fby + Fpy + Fvy;
    ux = jx + Fx / (2.0 * rho);                          /* A14 */
    uy = jy + Fy / (2.0 * rho);
    p = lbmref_pressure(alpha, N, ux, uy);               /* A15 */
  }

  /* equilibrium A4 and forcing A8 (c_o read as c_s, R2): F_i = w_i/c_s^2 (F dt / rho) . c_i */
  double Neq[9], Fi[9];
  lbmref_neq(alpha, p, ux, uy, Neq);
  for (int i = 0; i < 9; i++) Fi[i] = WGT[i] / CS2 * ((Fx / rho) * CX[i] + (Fy / rho) * CY[i]);

  /* collision A1 with S = diag(1,1,1,1,1,1,1,s7,s8), s7 = s8 = 1/tau (A3, R7) */
  double S[9];
  for (int k = 0; k < 7; k++) S[k] = 1.0;
  S[7] = S[8] = 1.0 / tau;
  double md[9], mF[9];
  for (int k = 0; k < 9; k++) {
    double a = 0.0, b = 0.0;
    for (int i = 0; i < 9; i++) {
      a += M[k * 9 + i] * (N[i] - Neq[i]);
      b += M[k * 9 + i] * Fi[i];
    }
    md[k] = S[k] * a;
    mF[k] = (1.0 - 0.5 * S[k]) * b;
  }
  for (int i = 0; i < 9; i++) {
    double a = 0.0, b = 0.0;
    for (int k = 0; k < 9; k++) {
      a += Minv[i * 9 + k] * md[k];
      b += Minv[i * 9 + k] * mF[k];
    }
    Nstar[i] = N[i] - a + b;
  }

  /* segregation A12; n_phi = grad phi/|grad phi|, term dropped where the
   * gradient vanishes (R16); N^{eq,u=0} uses the final p (R20). */
  double g2 = sqrt(gx * gx + gy * gy);
  double nxh = 0.0, nyh = 0.0;
  if (g2 > 0.0) { nxh = gx / g2; nyh = gy / g2; }
  double Neq0[9];
  lbmref_neq(alpha, p, 0.0, 0.0, Neq0);
  for (int i = 0; i < 9; i++)
    Bstar[i] = phi * Nstar[i] + 2.0 * (CX[i] * nxh + CY[i] * nyh) / P->W * phi * (1.0 - phi) * Neq0[i];

  if (f) {
    f->phi = phi; f->gradx = gx; f->grady = gy; f->lap = lap;
    f->rho = rho; f->tau = tau;
    f->Fsx = Fsx; f->Fsy = Fsy; f->Fx = Fx; f->Fy = Fy;
    f->ux = ux; f->uy = uy; f->p = p;
  }
}

/* ---- create: classification and ghost geometry (one-time) -------------------------------- */
static int fail(lbmref_ctx* c, int code, const char* msg) {
  if (c) snprintf(c->err, sizeof c->err, "%s", msg);
  return code;
}

static double minimg(double d, double L) {
  /* minimum-image displacement in a periodic box of length L */
  d = fmod(d, L);
  if (d >= 0.5 * L) d -= L;
  if (d < -0.5 * L) d += L;
  return d;
}

int lbmref_create(lbmref_ctx** out, const lbmref_params* P, const uint8_t* mask,
                  const lbmref_disk* disks, int32_t n_disks) {
  if (!out || !P || !mask) return EINVAL_;
  *out = NULL;
  if (P->nx < 3 || P->ny < 3) return EINVAL_;
  if (!(P->rho_l > 0.0) || !(P->rho_g > 0.0)) return EINVAL_;
  if (!(P->nu_l > 0.0) || !(P->nu_g > 0.0)) return EINVAL_;   /* tau > 1/2 */
  if (!(P->W >= 4.0)) return EINVAL_;
  if (!(P->sigma >= 0.0)) return EINVAL_;
  if (!(P->theta_deg >= 0.0 && P->theta_deg <= 180.0)) return EINVAL_;
  if (!(P->mobility > 0.0 && P->mobility < 0.3)) return EINVAL_;
  if (P->ghost_rule != 0 && P->ghost_rule != 1) return EINVAL_;
  if (n_disks < 0 || (n_disks > 0 && !disks)) return EINVAL_;

  lbmref_ctx* c = (lbmref_ctx*)calloc(1, sizeof *c);
  if (!c) return ENOMEM_;
  c->P = *P;
  int nx = P->nx, ny = P->ny, n = nx * ny;
  c->n = n;
  c->solid = (uint8_t*)malloc((size_t)n);
  c->cls = (uint8_t*)malloc((size_t)n);
  c->phi = (double*)calloc((size_t)n, sizeof(double));
  c->scratch = (double*)calloc((size_t)n, sizeof(double));
  c->N = (double*)calloc((size_t)9 * n, sizeof(double));
  c->B = (double*)calloc((size_t)9 * n, sizeof(double));
  c->N2 = (double*)calloc((size_t)9 * n, sizeof(double));
  c->B2 = (double*)calloc((size_t)9 * n, sizeof(double));
  if (!c->solid || !c->cls || !c->phi || !c->scratch || !c->N || !c->B || !c->N2 || !c->B2) {
    lbmref_destroy(c);
    return ENOMEM_;
  }
  for (int k = 0; k < n; k++) c->solid[k] = mask[k] ? 1 : 0;
  if (P->wall_rows) {
    for (int i = 0; i < nx; i++)
      if (!c->solid[i] || !c->solid[(ny - 1) * nx + i]) {
        lbmref_destroy(c);
        return EINVAL_;
      }
  }

  /* (1) node classes: "The solid (fluid) boundary nodes are those with at least one
   * neighbor that is fluid (solid), as defined by the given stencil" — D2Q9, periodic wrap. */
  int n_ghost = 0;
  for (int j = 0; j < ny; j++)
    for (int i = 0; i < nx; i++) {
      int k = j * nx + i, other = 0;
      for (int q = 1; q < 9; q++) {
        int kk = wrapi(j + CY[q], ny) * nx + wrapi(i + CX[q], nx);
        if (c->solid[kk] != c->solid[k]) other = 1;
      }
      if (c->solid[k]) c->cls[k] = other ? LBMREF_GHOST : LBMREF_SOLID_BULK;
      else c->cls[k] = other ? LBMREF_FLUID_BOUNDARY : LBMREF_FLUID_BULK;
      if (c->cls[k] == LBMREF_GHOST) n_ghost++;
    }
  c->n_ghost = n_ghost;
  size_t ng = (size_t)(n_ghost > 0 ? n_ghost : 1);
  c->g_idx = (int32_t*)malloc(ng * sizeof(int32_t));
  c->g_nx = (double*)malloc(ng * sizeof(double));
  c->g_ny = (double*)malloc(ng * sizeof(double));
  c->g_depth = (double*)malloc(ng * sizeof(double));
  c->g_corner = (int32_t*)malloc(4 * ng * sizeof(int32_t));
  c->g_wgt = (double*)malloc(4 * ng * sizeof(double));
  c->g_new = (double*)malloc(ng * sizeof(double));
  if (!c->g_idx || !c->g_nx || !c->g_ny || !c->g_depth || !c->g_corner || !c->g_wgt || !c->g_new) {
    lbmref_destroy(c);
    return ENOMEM_;
  }

  /* (2) ghost list in increasing idx with analytic unit normals pointing away
   * from the solid, x_F = x_G + dx n_s (Fig. 2) and its bilinear
   * stencil.  Owner of a ghost node (R17): wall row if it lies on one, else the disk that
   * contains it with the least depth R - |x_G - x_c| (minimum image). */
  int g = 0;
  int32_t* smooth2 = NULL;
  for (int k = 0; k < n; k++) {
    if (c->cls[k] != LBMREF_GHOST) continue;
    int i = k % nx, j = k / nx;
    double nxs = 0.0, nys = 0.0, depth = 0.0;
    int found = 0;
    if (P->wall_rows && (j == 0 || j == ny - 1)) {
      nxs = 0.0;
      nys = (j == 0) ? 1.0 : -1.0;
      depth = 0.5; /* half-way wall (R17) */
      found = 1;
    } else {
      double best = 0.0;
      for (int d = 0; d < n_disks; d++) {
        double dx = minimg((double)i - disks[d].cx, (double)nx);
        double dy = minimg((double)j - disks[d].cy, (double)ny);
        double r2 = dx * dx + dy * dy;
        if (r2 <= disks[d].r * disks[d].r) {
          double dist = sqrt(r2);
          double dep = disks[d].r - dist;
          if (!found || dep < best) {
            best = dep;
            found = 1;
            depth = dep;
            if (dist > 0.0) { nxs = dx / dist; nys = dy / dist; }
            else { nxs = 0.0; nys = 0.0; }
          }
        }
      }
    }
    if (!found && n_disks == 0) { /* NEXT row f2: no analytic shape given, normal from the mask */
      if (!smooth2) { /* the indicator smoothed twice, built on first use */
        int32_t* s0 = (int32_t*)malloc((size_t)n * sizeof(int32_t));
        int32_t* s1 = (int32_t*)malloc((size_t)n * sizeof(int32_t));
        smooth2 = (int32_t*)malloc((size_t)n * sizeof(int32_t));
        if (!s0 || !s1 || !smooth2) { free(s0); free(s1); free(smooth2); lbmref_destroy(c); return ENOMEM_; }
        for (int kk = 0; kk < n; kk++) s0[kk] = c->solid[kk] ? 1 : 0;
        lbmref_mask_smooth(s0, s1, nx, ny);
        lbmref_mask_smooth(s1, smooth2, nx, ny);
        free(s0); free(s1);
      }
      lbmref_mask_normal(smooth2, nx, ny, i, j, &nxs, &nys);
      depth = 0.0;
      found = 1;
    }
    if (!found) { /* mask and geometry disagree */
      free(smooth2);
      lbmref_destroy(c);
      return EINVAL_;
    }
    c->g_idx[g] = k;
    c->g_nx[g] = nxs;
    c->g_ny[g] = nys;
    c->g_depth[g] = depth;
    lbmref_bilinear_setup((double)i + nxs, (double)j + nys, nx, ny, &c->g_corner[4 * g], &c->g_wgt[4 * g]);
    g++;
  }
  free(smooth2);
  *out = c;
  return OK;
}

void lbmref_destroy(lbmref_ctx* c) {
  if (!c) return;
  free(c->solid); free(c->cls); free(c->phi); free(c->scratch);
  free(c->N); free(c->B); free(c->N2); free(c->B2);
  free(c->g_idx); free(c->g_nx); free(c->g_ny); free(c->g_depth);
  free(c->g_corner); free(c->g_wgt); free(c->g_new);
  free(c);
}

const char* lbmref_last_error(const lbmref_ctx* c) { return c ? c->err : "null context"; }

/* ---- init (R14): phi from phi0 on fluid nodes, (1+cos theta)/2 on all solid nodes
 * (PAPER.md:100), N_i = N_i^eq(p = 0, u0), B_i = phi N_i. ---------------------------------- */
int lbmref_init(lbmref_ctx* c, const double* phi0, const double* u0) {
  if (!c || !phi0) return EINVAL_;
  int n = c->n;
  double alpha = lbmref_alpha_from_mobility(c->P.mobility);
  double phis = 0.5 * (1.0 + cos(c->P.theta_deg * M_PI / 180.0));
  for (int k = 0; k < n; k++) {
    double Neq[9];
    if (c->solid[k]) {
      c->phi[k] = phis;
      for (int i = 0; i < 9; i++) c->N[i * n + k] = c->B[i * n + k] = 0.0;
      continue;
    }
    c->phi[k] = phi0[k];
    lbmref_neq(alpha, 0.0, u0 ? u0[k] : 0.0, u0 ? u0[n + k] : 0.0, Neq);
    for (int i = 0; i < 9; i++) {
      c->N[i * n + k] = Neq[i];
      c->B[i * n + k] = phi0[k] * Neq[i];
    }
  }
  c->t = 0;
  return OK;
}

/* Steps 1 and 2 of the time step on an explicit phi array (so that lbmref_get can run them on a
 * scratch copy without touching the state). */
static void order_parameter_and_ghosts(lbmref_ctx* c, double* phi) {
  int n = c->n;
  /* 1. phi = sum_i B_i on fluid nodes, A13 */
  for (int k = 0; k < n; k++) {
    if (c->solid[k]) continue;
    double s = 0.0;
    for (int i = 0; i < 9; i++) s += c->B[i * n + k];
    phi[k] = s;
  }
  /* 2. ghost update, Jacobi (R13): every phi_F from the array as it stands (fluid: time-t
   * values; solid: values of the previous update / init), then commit all at once.
   * eps = -(4 dx / W) cos theta, Eq. 9. */
  double eps = -(4.0 / c->P.W) * cos(c->P.theta_deg * M_PI / 180.0);
  for (int g = 0; g < c->n_ghost; g++) {
    double phiF = 0.0;
    for (int q = 0; q < 4; q++) phiF += c->g_wgt[4 * g + q] * phi[c->g_corner[4 * g + q]];
    c->g_new[g] = lbmref_ghost_rule(phiF, eps, c->P.ghost_rule);
  }
  for (int g = 0; g < c->n_ghost; g++) phi[c->g_idx[g]] = c->g_new[g];
}

static void gather_phi_nb(const lbmref_ctx* c, const double* phi, int i, int j, double nb[9]) {
  int nx = c->P.nx, ny = c->P.ny;
  for (int q = 0; q < 9; q++) nb[q] = phi[wrapi(j + CY[q], ny) * nx + wrapi(i + CX[q], nx)];
}

/* One time step t -> t+1 (order of operations: R11). */
static void one_step(lbmref_ctx* c) {
  int nx = c->P.nx, ny = c->P.ny, n = c->n;
  order_parameter_and_ghosts(c, c->phi);
  /* 3. local update of every fluid node: post-collision N*, B* into N2, B2 */
  for (int j = 0; j < ny; j++)
    for (int i = 0; i < nx; i++) {
      int k = j * nx + i;
      if (c->solid[k]) continue;
      double Nl[9], nb[9], Ns[9], Bs[9];
      for (int q = 0; q < 9; q++) Nl[q] = c->N[q * n + k];
      gather_phi_nb(c, c->phi, i, j, nb);
      lbmref_node_update(&c->P, Nl, nb, Ns, Bs, NULL);
      for (int q = 0; q < 9; q++) { c->N2[q * n + k] = Ns[q]; c->B2[q * n + k] = Bs[q]; }
    }
  /* 4. propagation A16-A17 with half-way bounce-back for both N_i and B_i
   * (R12): pull form, N_i(x,t+1) = N_i*(x - c_i) if that node is fluid, else N_opp(i)*(x). */
  for (int j = 0; j < ny; j++)
    for (int i = 0; i < nx; i++) {
      int k = j * nx + i;
      if (c->solid[k]) continue;
      for (int q = 0; q < 9; q++) {
        int ks = wrapi(j - CY[q], ny) * nx + wrapi(i - CX[q], nx);
        if (c->solid[ks]) {
          c->N[q * n + k] = c->N2[OPP[q] * n + k];
          c->B[q * n + k] = c->B2[OPP[q] * n + k];
        } else {
          c->N[q * n + k] = c->N2[q * n + ks];
          c->B[q * n + k] = c->B2[q * n + ks];
        }
      }
    }
  c->t++;
}

int lbmref_step(lbmref_ctx* c, int64_t nsteps) {
  if (!c || nsteps < 0) return EINVAL_;
  for (int64_t s = 0; s < nsteps; s++) one_step(c);
  return OK;
}

/* Macroscopic fields at the current time: phi (with this time's ghost values, computed on a
 * scratch copy so that the state is not advanced), rho, u (A14), p (A15).  u = p = rho = 0 on
 * solid nodes ("fluid dynamical quantities are not evaluated at these nodes"). */
int lbmref_get(lbmref_ctx* c, double* rho, double* phi, double* ux, double* uy, double* p) {
  if (!c) return EINVAL_;
  int nx = c->P.nx, ny = c->P.ny, n = c->n;
  memcpy(c->scratch, c->phi, (size_t)n * sizeof(double));
  order_parameter_and_ghosts(c, c->scratch);
  for (int j = 0; j < ny; j++)
    for (int i = 0; i < nx; i++) {
      int k = j * nx + i;
      if (phi) phi[k] = c->scratch[k];
      if (c->solid[k]) {
        if (rho) rho[k] = 0.0;
        if (ux) ux[k] = 0.0;
        if (uy) uy[k] = 0.0;
        if (p) p[k] = 0.0;
        continue;
      }
      double Nl[9], nb[9], Ns[9], Bs[9];
      lbmref_node_fields f;
      for (int q = 0; q < 9; q++) Nl[q] = c->N[q * n + k];
      gather_phi_nb(c, c->scratch, i, j, nb);
      lbmref_node_update(&c->P, Nl, nb, Ns, Bs, &f);
      if (rho) rho[k] = f.rho;
      if (ux) ux[k] = f.ux;
      if (uy) uy[k] = f.uy;
      if (p) p[k] = f.p;
    }
  return OK;
}

int lbmref_get_populations(lbmref_ctx* c, double* N, double* B) {
  if (!c) return EINVAL_;
  if (N) memcpy(N, c->N, (size_t)9 * c->n * sizeof(double));
  if (B) memcpy(B, c->B, (size_t)9 * c->n * sizeof(double));
  return OK;
}

int lbmref_set_populations(lbmref_ctx* c, const double* N, const double* B) {
  if (!c) return EINVAL_;
  if (N) memcpy(c->N, N, (size_t)9 * c->n * sizeof(double));
  if (B) memcpy(c->B, B, (size_t)9 * c->n * sizeof(double));
  return OK;
}

int lbmref_get_phi_raw(lbmref_ctx* c, double* phi) {
  if (!c || !phi) return EINVAL_;
  memcpy(phi, c->phi, (size_t)c->n * sizeof(double));
  return OK;
}

int lbmref_get_classification(lbmref_ctx* c, uint8_t* cls, int32_t* n_ghost, int32_t* ghost_idx,
                              double* ghost_nx, double* ghost_ny, double* ghost_depth,
                              int32_t* ghost_corner, double* ghost_wgt) {
  if (!c) return EINVAL_;
  size_t ng = (size_t)c->n_ghost;
  if (cls) memcpy(cls, c->cls, (size_t)c->n);
  if (n_ghost) *n_ghost = c->n_ghost;
  if (ghost_idx) memcpy(ghost_idx, c->g_idx, ng * sizeof(int32_t));
  if (ghost_nx) memcpy(ghost_nx, c->g_nx, ng * sizeof(double));
  if (ghost_ny) memcpy(ghost_ny, c->g_ny, ng * sizeof(double));
  if (ghost_depth) memcpy(ghost_depth, c->g_depth, ng * sizeof(double));
  if (ghost_corner) memcpy(ghost_corner, c->g_corner, 4 * ng * sizeof(int32_t));
  if (ghost_wgt) memcpy(ghost_wgt, c->g_wgt, 4 * ng * sizeof(double));
  return OK;
}

/* Diagnostics over fluid nodes at the current time: sum phi, sum (1-phi), kinetic energy
 * 1/2 sum rho |u|^2, max |u|, min phi, max phi, n_fluid, NaN flag.  Plain left-to-right sums. */
int lbmref_diag(lbmref_ctx* c, double out[8]) {
  if (!c || !out) return EINVAL_;
  int n = c->n;
  double* rho = (double*)malloc((size_t)n * sizeof(double));
  double* phi = (double*)malloc((size_t)n * sizeof(double));
  double* ux = (double*)malloc((size_t)n * sizeof(double));
  double* uy = (double*)malloc((size_t)n * sizeof(double));
  if (!rho || !phi || !ux || !uy) { free(rho); free(phi); free(ux); free(uy); return ENOMEM_; }
  lbmref_get(c, rho, phi, ux, uy, NULL);
  double ml = 0, mg = 0, ke = 0, umax = 0, pmin = INFINITY, pmax = -INFINITY, nf = 0, bad = 0;
  for (int k = 0; k < n; k++) {
    if (c->solid[k]) continue;
    double u2 = ux[k] * ux[k] + uy[k] * uy[k];
    ml += phi[k];
    mg += 1.0 - phi[k];
    ke += 0.5 * rho[k] * u2;
    if (sqrt(u2) > umax) umax = sqrt(u2);
    if (phi[k] < pmin) pmin = phi[k];
    if (phi[k] > pmax) pmax = phi[k];
    if (!(phi[k] == phi[k]) || !(u2 == u2)) bad = 1;
    nf += 1;
  }
  out[0] = ml; out[1] = mg; out[2] = ke; out[3] = umax;
  out[4] = pmin; out[5] = pmax; out[6] = nf; out[7] = bad;
  free(rho); free(phi); free(ux); free(uy);
  return OK;
}

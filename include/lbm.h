/* include/lbm.h — C ABI of liblbm_b200.so: the per-time-step update of the 2-D (D2Q9) color-gradient
 * lattice Boltzmann model with the ghost-node wetting boundary condition of arxiv/paper_2605_30878,
 * hand-written CUDA for sm_100a (B200).  One GPU, fp64 or fp32 device arithmetic.
 *
 * What the calls compute (citations are PAPER.md lines; "R<k>" are the readings in DESIGN.md):
 *   lbm_create   node classes (a fluid/solid boundary node has >= 1 solid/fluid D2Q9
 *                neighbour), the index-sorted ghost-node list with analytic unit normals n_s
 *                (:100), the point x_F = x_G + dx n_s and its bilinear stencil (:66, Fig. 2).
 *   lbm_init     phi on solid nodes = (1 + cos theta)/2 (:100); N_i = N_i^eq(p = 0, u0) (Eq. A4,
 *                :275), B_i = phi N_i (R14); first ghost update (Eq. 9, :78-80).
 *   lbm_step     n x { collision A1 (:264) with velocity-based equilibrium A4, forcing A8-A11
 *                (:290-302), surface tension Eq. 4 (:45), segregation A12 (:307); propagation
 *                A16-A17 (:318-322) with half-way bounce-back (R12); phi = sum_i B_i (A13, :311);
 *                ghost update phi_G = phi_F / (phi_F + (1 - phi_F) e^eps), eps = -4 dx cos(theta)/W
 *                (Eq. 9, :78-80) }.
 *   lbm_get      rho (:43), phi (A13), u (A14, :313), p (A15, :315) at the current time.
 *   lbm_rows_export / lbm_rows_import   no arithmetic: the rows of the state next to a cut, for the slab
 *                decomposition along y (the update of a row reaches 3 rows: A16-A17, R8, :66).
 *
 * Conventions: node (i, j) sits at (x, y) = (i, j); linear index idx = j*nx + i (x fastest);
 * periodic in both directions; flat walls are rows of solid nodes inside the array; dx = dt = 1;
 * c_s^2 = 1/3; direction order of Eq. A5 (:280):
 *   c = (0,0),(1,0),(0,1),(-1,0),(0,-1),(1,1),(-1,1),(-1,-1),(1,-1).
 * Population arrays are structure-of-arrays: pop[q*nx*ny + idx].
 *
 * Deviations from the call list SURVEY.md 8(b) proposed (all recorded in DESIGN.md 1): lbm_plan (exact sizing
 * from the mask, needs a device) exists beside lbm_workspace_bytes (host-only upper bound); lbm_params has
 * three more fields (precision, ghost_rule, schedule); B_i are returned only after lbm_keep_B because they
 * are not part of the stored state; lbm_set_populations, lbm_sample_populations, lbm_rows_* and lbm_diag_static
 * were added;
 * test and measurement hooks live in include/lbm_test.h.
 *
 * Memory and ownership: every pointer is the caller's.  Pointers marked HOST must be host
 * memory (pageable or pinned) and are only used during the call; they are never retained.
 * `d_workspace` (DEVICE) is the only device memory a context uses — state, lists and the temporaries of
 * lbm_create alike.  Three calls allocate and free their own: lbm_plan and the hook lbm_node_update_batch
 * (they have no workspace), and lbm_keep_B(ctx, 1) under the compacted layouts (PACK, SPARSE), whose
 * workspace holds no B planes (9 planes of nx*ny values, released by lbm_destroy).  The workspace must
 * stay allocated until lbm_destroy and be at least `workspace_bytes` (from lbm_plan) long, 256-byte
 * aligned.  `cuda_stream` is a borrowed cudaStream_t (0 = default stream); all work of a context
 * is enqueued on it.  A context is not thread-safe; different contexts are independent.
 *
 * Errors: every int-returning call returns LBM_OK (0) or a negative code; nothing throws or aborts
 * across the ABI; lbm_last_error(ctx) holds a readable message (for LBM_ECUDA the CUDA error
 * string).  There is NO CPU fallback: without a usable CUDA device every compute call fails with
 * LBM_ECUDA.
 */
#ifndef LBM_B200_H
#define LBM_B200_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { LBM_OK = 0, LBM_EINVAL = -1, LBM_ENOMEM = -2, LBM_ECUDA = -3 };

/* node classes (Fig. 1) */
enum { LBM_FLUID_BULK = 0, LBM_FLUID_BOUNDARY = 1, LBM_GHOST = 2, LBM_SOLID_BULK = 3 };

/* launch schedules of lbm_step (same arithmetic per node, different kernel decomposition) */
enum {
  LBM_SCHEDULE_AUTO = 0,      /* the fastest schedule available (currently PACK)                  */
  LBM_SCHEDULE_BASELINE = 1,  /* 3 launches/step: collide+stream, phi = sum B, ghost; N and B in HBM */
  LBM_SCHEDULE_FUSED = 2,     /* 2 launches/step: tiled collide+stream that also produces phi(t+1)
                                 from B* held in shared memory (B never touches HBM), ghost        */
                              /* 3 was the WARP schedule of round 1 (superseded by PAIR, removed): LBM_EINVAL */
  LBM_SCHEDULE_PAIR = 4,      /* 2 launches/step, barrier-free: one warp marches down a strip of columns,
                                 every lane owns an aligned group of nodes (2 in fp64, 4 in fp32); each
                                 population is fetched once, unshifted, as an 8/16-byte vector through a
                                 per-warp cp.async ring; phi(t+1) is assembled in registers;
                                 propagation in x is a warp shuffle; fp32 arithmetic is packed
                                 (FFMA2).  Needs even nx, else FUSED is used                        */
  LBM_SCHEDULE_PACK = 5,      /* the PAIR kernel on pair-compacted population planes: a plane stores
                                 only the node pairs that hold a fluid node, row after row, without
                                 holes (addressed through a 1-bit-per-pair mask + prefix table).  No
                                 dense copy exists: lbm_get / lbm_diag / ... read the compact planes.
                                 Needs even nx, else FUSED is used                                  */
  LBM_SCHEDULE_SPARSE = 6,    /* the PACK layout with lanes mapped to fluid groups: one persistent CTA
                                 per SM, rows brought on chip by 1-D bulk copies (TMA) into a shared-memory
                                 ring, consumer warps work on 32 consecutive entries of the active-group
                                 sequence.  Needs 16-byte groups (fp64: even nx; fp32: nx % 4 == 0) and
                                 at least 4 groups per row, else PACK is used                        */
  LBM_SCHEDULE_INPLACE = 7    /* single-buffer streaming (AA pattern) on the canonical state: ONE buffer of the
                                 nine N_i and one of the nine B_i (18 planes instead of BASELINE's 36), one
                                 thread per node; every thread writes only the slots it read.  Same arithmetic
                                 and the same two launches per step as BASELINE (collide, phi = sum B_i)    */
};

typedef struct lbm_ctx lbm_ctx;                 /* opaque; one simulation                         */

typedef struct { double cx, cy, r; } lbm_disk;  /* analytic solid: closed disk, periodic images   */

typedef struct {
  int32_t nx, ny;          /* grid; both >= 3                                                     */
  int32_t precision;       /* 64 or 32: device storage and arithmetic (host I/O is always double) */
  int32_t wall_rows;       /* 1: rows j = 0 and j = ny-1 are flat walls (must be solid in mask)   */
  int32_t ghost_rule;      /* 0: Eq. 9 (the paper's rule); 1: Eq. 10 (Fakhari-Bolster, :84)       */
  int32_t schedule;        /* LBM_SCHEDULE_*                                                      */
  double  rho_l, rho_g;    /* phase densities (:43); "density ratio" = rho_l / rho_g              */
  double  nu_l, nu_g;      /* kinematic viscosities; tau = 1/2 + 3 nu (:273)                      */
  double  sigma, W;        /* surface tension, interface width (Eq. 4-5); W >= 4 (:80)            */
  double  theta_deg;       /* equilibrium contact angle measured in the liquid (:60), [0, 180]    */
  double  mobility;        /* M_phi at reference p = 0: alpha = 1 - 10 M_phi / 3 (:288, R5)       */
  double  gx, gy;          /* body acceleration, F_b = rho g (Eq. 2, :39)                         */
} lbm_params;

/* Sizes a context.  mask: HOST, nx*ny bytes, non-zero = solid.  Runs the classification kernel
 * once on a temporary device copy of the mask (cudaMalloc/cudaFree inside the call) and returns
 * the exact number of ghost nodes and the workspace size lbm_create needs.  Either output may be
 * NULL.  LBM_EINVAL on bad parameters (sizes < 3, rho <= 0, nu <= 0, W < 4, sigma < 0, theta
 * outside [0,180], mobility outside (0, 0.3), precision not 32/64, wall rows not solid). */
int lbm_plan(const lbm_params* prm, const uint8_t* mask, int64_t* n_ghost, size_t* workspace_bytes);

/* Relaxation time <-> kinematic viscosity of a phase, tau = 1/2 + nu / (c_s^2 dt) = 1/2 + 3 nu (dx = dt = 1,
 * c_s^2 = 1/3): for callers who state the problem with tau per phase (north_star: "tau or viscosity per phase").
 * Host arithmetic only. */
double lbm_nu_from_tau(double tau);
double lbm_tau_from_nu(double nu);

/* Upper bound of the workspace size without touching a device or the mask (pure host arithmetic): what
 * lbm_create needs for a mask with at most `n_ghost_bound` ghost nodes in which every node group may hold
 * a fluid node.  lbm_plan's exact figure is never larger.  0 on bad parameters. */
size_t lbm_workspace_bytes(const lbm_params* prm, int64_t n_ghost_bound);

/* Builds a context in the caller's device workspace.  mask: HOST nx*ny bytes (copied).
 * disks: HOST array of n_disks analytic disks whose rasterisation produced the solid nodes of the
 * mask (closed disks, minimum-image distance^2 <= r^2); every ghost node that is not on a wall
 * row must lie in at least one disk, else LBM_EINVAL ("mask and geometry disagree").  The owner of
 * a ghost node is the containing disk with the least depth r - |x_G - x_c| (first wins ties, R17).
 * With n_disks == 0 the normals of all ghost nodes that are not on a wall row come from the mask
 * alone: n_s = -grad(s~)/|grad(s~)|, s~ the solid indicator smoothed twice, all with
 * the sixth-order isotropic 12-point stencil (weights 4/15, 1/10, 1/120 at |c|^2 = 1, 2, 4; centre
 * weight 1/2 in the smoothing); depth is reported as 0.  On a disk of radius 40 these normals are
 * within 13 degrees (3 degrees on average, no bias) of the analytic ones.
 * LBM_ENOMEM if workspace_bytes is too small. */
int lbm_create(lbm_ctx** out, const lbm_params* prm, const uint8_t* mask, const lbm_disk* disks,
               int32_t n_disks, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/* Sets the state at time 0.  phi0: HOST nx*ny doubles (values on solid nodes are ignored).
 * u0: HOST 2*nx*ny doubles (u_x plane then u_y plane) or NULL for a fluid at rest.  Synchronises
 * the stream before returning. */
int lbm_init(lbm_ctx* ctx, const double* phi0, const double* u0);

/* Advances n >= 0 time steps.  Asynchronous: kernels are enqueued on the stream. */
int lbm_step(lbm_ctx* ctx, int64_t n);

/* Blocks until all enqueued work of the context has finished. */
int lbm_sync(lbm_ctx* ctx);

/* Macroscopic fields at the current time, HOST nx*ny doubles each, any may be NULL.  phi carries
 * this time's ghost values on ghost nodes and (1+cos theta)/2 on bulk solid nodes; rho = u = p = 0
 * on solid nodes ("fluid dynamical quantities are not evaluated at these nodes", :21).  p is the
 * auxiliary pressure of Eq. A15 (p_h = rho p).  Synchronises. */
int lbm_get(lbm_ctx* ctx, double* rho, double* phi, double* ux, double* uy, double* p);

/* Post-stream populations N_i(x, t), B_i(x, t) of the current time, HOST 9*nx*ny doubles each
 * (SoA), either may be NULL; zeros on solid nodes.  Under every schedule but BASELINE (FUSED,
 * PAIR, PACK, SPARSE, hence AUTO) the B_i are not part of the stored state: they are available right after
 * lbm_init, and after lbm_step only if lbm_keep_B(ctx, 1) was set before that step (else
 * LBM_EINVAL for B != NULL).  Synchronises. */
int lbm_get_populations(lbm_ctx* ctx, double* N, double* B);

/* Overwrites the post-stream populations of the current time (the arrays lbm_get_populations returns):
 * N and/or B, HOST 9*nx*ny doubles each (SoA), either may be NULL; values on solid nodes are ignored.
 * With B given, phi = sum_i B_i (A13, :311) on fluid nodes and the ghost values are updated from it
 * (Eq. 9, Jacobi: solid corners keep their previous values, R13) — exactly what the next time step of
 * the oracle does after its set_populations.  Synchronises. */
int lbm_set_populations(lbm_ctx* ctx, const double* N, const double* B);

/* Rows of the state as one device buffer: the hand-over between the slabs of a 1-D domain decomposition along y
 * (the path shards into slabs that exchange the populations and phi rows next to each cut; the method
 * itself is local, A16-A17 :318-322 move a population by one node per step).  The complete state of a context at time
 * t is phi(x, t) (fluid and ghost values) and the populations N_i; lbm_rows_export copies the part that belongs to
 * the grid rows j0 <= j < j0 + nrows (no wrap) into d_buf (DEVICE, >= lbm_rows_bytes bytes, caller-owned),
 * lbm_rows_import overwrites those rows from such a buffer.  The buffer is in the context's own storage format: it
 * can only be imported by a context with the same nx, precision and schedule whose solid mask agrees on these rows
 * (else LBM_EINVAL: the sizes differ).  Under LBM_SCHEDULE_INPLACE the buffer also carries where that schedule parks
 * the populations at even / odd times: the two contexts must have taken numbers of steps of the same parity since
 * lbm_init (slabs always have).  Asynchronous on the context's stream; lbm_rows_bytes may synchronise once.
 * Ghost-node geometry is not transferred: each context computes its own at lbm_create. */
int lbm_rows_bytes(lbm_ctx* ctx, int32_t j0, int32_t nrows, size_t* bytes);
int lbm_rows_export(lbm_ctx* ctx, int32_t j0, int32_t nrows, void* d_buf, size_t capacity);
int lbm_rows_import(lbm_ctx* ctx, int32_t j0, int32_t nrows, const void* d_buf, size_t bytes);

/* Every schedule but BASELINE: when on != 0 the last time step of every lbm_step call also writes the
 * post-collision B_i* to HBM so that lbm_get_populations / lbm_sample_populations can return B_i; set before
 * lbm_init it keeps the initial B_i too.  No effect on the arithmetic.  Dense layouts (FUSED, PAIR) have the
 * planes in their workspace; the compacted layouts (PACK, SPARSE, hence AUTO) allocate them with cudaMalloc on the
 * first call with on != 0 (LBM_ECUDA if that fails).  Ignored by the BASELINE schedule (B always stored). */
int lbm_keep_B(lbm_ctx* ctx, int32_t on);

/* Populations at selected nodes only (for parity checks at sizes where 18 full arrays are too
 * much to move): idx HOST n_idx int64 node indices; N, B HOST 9*n_idx doubles (q-major:
 * out[q*n_idx + k]); B may be NULL (same availability rule as lbm_get_populations). */
int lbm_sample_populations(lbm_ctx* ctx, int64_t n_idx, const int64_t* idx, double* N, double* B);

/* Classification and ghost geometry (all HOST, any may be NULL): cls nx*ny bytes (LBM_* classes);
 * *n_ghost; then per ghost node in increasing idx: ghost_idx[n_ghost], unit normal
 * (ghost_nx, ghost_ny), depth below the surface, the 4 bilinear corner indices ghost_corner
 * [4*n_ghost] and weights ghost_wgt[4*n_ghost] of x_F (order (i0,j0),(i0+1,j0),(i0,j0+1),
 * (i0+1,j0+1)). */
int lbm_get_classification(lbm_ctx* ctx, uint8_t* cls, int32_t* n_ghost, int32_t* ghost_idx,
                           double* ghost_nx, double* ghost_ny, double* ghost_depth,
                           int32_t* ghost_corner, double* ghost_wgt);

/* Diagnostics over fluid nodes at the current time (warp-shuffle + fixed-tree block reductions,
 * deterministic): out[0] = sum phi, [1] = sum (1 - phi), [2] = 1/2 sum rho |u|^2, [3] = max |u|,
 * [4] = min phi, [5] = max phi, [6] = number of fluid nodes, [7] = 1 if any NaN.  out: HOST. */
int lbm_diag(lbm_ctx* ctx, double out[8]);

/* The same diagnostics for callers that cannot allocate or synchronise (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the eight values of lbm_diag go to d_out (DEVICE, 8 doubles, caller-owned),
 * asynchronously on the context's stream.  The block partials of the reduction live in a file-scope device array of
 * the library (4 MiB, held by every GPU that loads the library until the process exits) instead of the workspace; the
 * call makes no cudaMalloc / cudaFree, no host copy and no synchronisation.
 * Limit: ceil(nx / 256) * ny <= 65,536 block partials (e.g. up to 4096 x 4096); larger grids get LBM_EINVAL with the
 * numbers in lbm_last_error: use lbm_diag there.  The array is shared by ALL contexts on a device and keeps the last
 * call's partials (every slot that is read is written first, nothing needs clearing): two calls that overlap on the
 * GPU (different streams, or graphs launched concurrently) race; calls on one stream, or otherwise ordered, do not. */
int lbm_diag_static(lbm_ctx* ctx, double* d_out);

const char* lbm_last_error(const lbm_ctx* ctx); /* ctx may be NULL: last error of lbm_plan/create */
const char* lbm_version(void);
void lbm_destroy(lbm_ctx* ctx);                 /* frees the host handle only; workspace is the caller's */

#ifdef __cplusplus
}
#endif
#endif

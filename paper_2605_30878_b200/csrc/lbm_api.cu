// lbm_api.cu — host side of liblbm_b200.so: the C ABI of include/lbm.h, workspace carving and
// the launch schedule.  No CPU fallback: every compute call needs a CUDA device.
#include <cuda_runtime.h>
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/lbm.h"
#include "../../include/lbm_test.h"
#include "lbm_fused.cuh"
#include "lbm_kernels.cuh"
#include "lbm_pair.cuh"
#include "lbm_sparse.cuh"

using namespace lbm;

namespace {

thread_local char g_err[512] = "";

struct Arena {  // carves 256-byte aligned chunks out of the caller's workspace
  char* base;
  size_t off;
  template <typename T>
  T* take(size_t count) {
    off = (off + 255) & ~(size_t)255;
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += count * sizeof(T);
    return p;
  }
};

}  // namespace

struct lbm_ctx {
  lbm_params P;
  size_t n;
  int ng;
  int is32;
  int fused;
  int sched;         // resolved LBM_SCHEDULE_* (never AUTO)
  int keep_B;
  int inplace;       // INPLACE schedule: one N and one B buffer, AA pattern
  int aa_local;      // ... and the state is parked in the nodes' own opposite slots (odd number of steps since standard)
  int B_owned;       // compacted layouts: the B planes are not in the workspace; lbm_keep_B allocates them on demand
  int B_valid;       // B planes of buffer `cur` hold the post-collision B* of the last step
  cudaStream_t st;
  Consts<double> Cd;
  Consts<float> Cf;
  // device arrays (inside the caller's workspace)
  void* N[2];
  void* B[2];        // BASELINE: both; FUSED: B[0] only (keep_B / init)
  void* phi[2];
  uint8_t* cls;
  uint8_t* links;
  uint16_t* cl16;     // class byte | link byte << 8 (WARP schedule reads one word per node)
  int* gidx;
  int* corner;
  void* wgt;
  double* wgt_d;
  double *gnx, *gny, *gdepth;
  uint8_t* csolid;
  // the same list in the ghost kernel's processing order (tile-major)
  uint2* gent_p;      // {node index, corner code}
  void* gfr_p;        // (f_x, f_y) in the device precision
  // PACK schedule: pair-compacted population planes (dense N[cur] is a mirror, refreshed on demand)
  int packed;
  int ccur;
  int nw;            // ptab words per row
  size_t cps;        // compact plane stride in pairs
  uint2* ptab;
  void* Nc[2];
  long long nfp;        // groups stored in a compact plane
  unsigned* row_base;   // host, ny + 1: compact index of the first group of every row (lbm_rows_*; fetched on first use)
  // SPARSE schedule: per (strip, row) descriptors, per-group metadata, the marches of every CTA
  int sparse;
  int sp_nstrips, sp_ncta, sp_nmarch, sp_sw;
  SpDesc* sp_desc;
  uint16_t* sp_cnt;
  uint2* sp_meta;
  SpMarch* sp_march;
  int* sp_first;
  size_t sp_march_cap;
  int* blk_cnt;
  int* blk_off;
  int* scal;          // [0] ghost total, [1] geometry error flag
  double* stage;      // 5 n doubles (n >= partials)
  double* diag_out;   // 8 doubles
  long long* samp_idx;
  size_t samp_cap;
  Disk* disks;
  int n_disks;
  int cur, pcur;      // population buffer holding the last post-collision state; phi buffer of time t
  int64_t t;
  int64_t launches[4];
  // small grids are launch-bound: lbm_step replays CUDA graphs of kGraphSteps steps, one graph per
  // parity of the ping-pong buffers it starts from
  int graph_warm;          // two plain steps have run on this context (kernel attributes are set)
  cudaGraphExec_t gexec[8];
  int64_t gdelta[8][4];   // launches a replay adds
  // lbm_diag_static: device address of g_diag_static on this context's device, resolved at lbm_create
  DiagVec* diag_static;
  int diag_static_err;     // cudaError_t of that resolution
  char err[512];
};

// ---- scratch of lbm_diag_static (lbm.h): the block partials of the diagnostics reduction in a file-scope device
// array, so that the call needs no workspace region, no cudaMalloc and no host synchronisation.  Every GPU that loads
// the library holds these 4 MiB until the process exits.  In host code the NAME is a host-side stand-in, not a device
// address: the address a kernel can use comes from cudaGetSymbolAddress (static_scratch_of below).
constexpr long long kDiagStaticMax = 65536;   // block partials (64 B each): grids up to e.g. 4096 x 4096
static __device__ __align__(256) DiagVec g_diag_static[kDiagStaticMax];

namespace {

int fail(lbm_ctx* c, int code, const char* msg) {
  snprintf(g_err, sizeof g_err, "%s", msg);
  if (c) snprintf(c->err, sizeof c->err, "%s", msg);
  return code;
}

int cuda_fail(lbm_ctx* c, cudaError_t e, const char* where) {
  char buf[400];
  snprintf(buf, sizeof buf, "CUDA error at %s: %s", where, cudaGetErrorString(e));
  return fail(c, LBM_ECUDA, buf);
}

#define CK(call)                                                   \
  do {                                                             \
    cudaError_t e_ = (call);                                       \
    if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);       \
  } while (0)

// once per device, with that device current (lbm_create is the set-up): the device address of g_diag_static
cudaError_t static_scratch_of(DiagVec** ptr) {
  struct Entry { int dev; DiagVec* p; cudaError_t e; };
  static std::mutex mu;
  static std::vector<Entry> table;
  *ptr = nullptr;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lk(mu);
  for (const auto& t : table)
    if (t.dev == dev) { *ptr = t.p; return t.e; }
  void* p = nullptr;
  e = cudaGetSymbolAddress(&p, g_diag_static);
  if (e != cudaSuccess) { cudaGetLastError(); p = nullptr; }
  table.push_back(Entry{dev, (DiagVec*)p, e});
  *ptr = (DiagVec*)p;
  return e;
}

int validate(const lbm_params* P, const char** why) {
  *why = "";
  if (!P) { *why = "null params"; return LBM_EINVAL; }
  if (P->nx < 3 || P->ny < 3) { *why = "nx, ny must be >= 3"; return LBM_EINVAL; }
  if ((long long)P->nx * P->ny > 0xffffffffLL / 9 - 4096) { *why = "nx*ny too large: 9 nx ny must fit 32-bit element offsets"; return LBM_EINVAL; }
  if (P->precision != 32 && P->precision != 64) { *why = "precision must be 32 or 64"; return LBM_EINVAL; }
  if (!(P->rho_l > 0.0) || !(P->rho_g > 0.0)) { *why = "densities must be > 0"; return LBM_EINVAL; }
  if (!(P->nu_l > 0.0) || !(P->nu_g > 0.0)) { *why = "viscosities must be > 0 (tau > 1/2)"; return LBM_EINVAL; }
  if (!(P->W >= 4.0)) { *why = "W must be >= 4 (PAPER.md:80)"; return LBM_EINVAL; }
  if (!(P->sigma >= 0.0)) { *why = "sigma must be >= 0"; return LBM_EINVAL; }
  if (!(P->theta_deg >= 0.0 && P->theta_deg <= 180.0)) { *why = "theta outside [0, 180]"; return LBM_EINVAL; }
  if (!(P->mobility > 0.0 && P->mobility < 0.3)) { *why = "mobility outside (0, 0.3)"; return LBM_EINVAL; }
  if (P->ghost_rule != 0 && P->ghost_rule != 1) { *why = "ghost_rule must be 0 or 1"; return LBM_EINVAL; }
  if (P->schedule < 0 || P->schedule > 7 || P->schedule == 3) { *why = "unknown schedule"; return LBM_EINVAL; }
  if (P->wall_rows != 0 && P->wall_rows != 1) { *why = "wall_rows must be 0 or 1"; return LBM_EINVAL; }
  return LBM_OK;
}

int check_walls(const lbm_params* P, const uint8_t* mask) {
  if (!P->wall_rows) return LBM_OK;
  for (int i = 0; i < P->nx; i++)
    if (!mask[i] || !mask[(size_t)(P->ny - 1) * P->nx + i]) return LBM_EINVAL;
  return LBM_OK;
}

// element stride between population planes: nx*ny rounded up to 64 elements plus 37*64, so that
// plane strides are never a power of two (8192^2 planes would otherwise all map to the same L2 sets)
size_t plane_stride(const lbm_params* P) {
  const size_t n = (size_t)P->nx * P->ny;
  return ((n + 63) & ~(size_t)63) + 37 * 64;
}

// Uniform grid of disk candidates for the one-time ghost geometry: cell (cy, cx) lists, in increasing
// disk index, every disk whose periodic bounding box overlaps the cell.
constexpr int kCell = 64;
void cover_cells(double lo, double hi, int n, int nc, std::vector<char>& hit) {
  std::fill(hit.begin(), hit.end(), 0);
  if (hi - lo >= n) { std::fill(hit.begin(), hit.end(), 1); return; }
  // walk the interval cell by cell in unwrapped coordinates; wrap every probe point
  for (double x = floor(lo); x <= floor(hi) + 1; x += 1.0) {
    if (x < floor(lo) || x > ceil(hi)) continue;
    long long xi = (long long)x % n;
    if (xi < 0) xi += n;
    hit[(size_t)(xi / kCell) < (size_t)nc ? xi / kCell : nc - 1] = 1;
  }
}
void build_disk_cells(const lbm_params* P, const lbm_disk* disks, int n_disks, int* ncx_out,
                      std::vector<int>& start, std::vector<int>& list) {
  const int ncx = (P->nx + kCell - 1) / kCell, ncy = (P->ny + kCell - 1) / kCell;
  *ncx_out = ncx;
  std::vector<std::vector<int>> cells((size_t)ncx * ncy);
  std::vector<char> hx(ncx), hy(ncy);
  for (int d = 0; d < n_disks; d++) {
    cover_cells(disks[d].cx - disks[d].r - 1.0, disks[d].cx + disks[d].r + 1.0, P->nx, ncx, hx);
    cover_cells(disks[d].cy - disks[d].r - 1.0, disks[d].cy + disks[d].r + 1.0, P->ny, ncy, hy);
    for (int cy = 0; cy < ncy; cy++)
      if (hy[cy])
        for (int cx = 0; cx < ncx; cx++)
          if (hx[cx]) cells[(size_t)cy * ncx + cx].push_back(d);
  }
  start.assign(cells.size() + 1, 0);
  for (size_t k = 0; k < cells.size(); k++) start[k + 1] = start[k] + (int)cells[k].size();
  list.resize((size_t)start.back() + 1);
  for (size_t k = 0; k < cells.size(); k++) std::copy(cells[k].begin(), cells[k].end(), list.begin() + start[k]);
}

bool use_inplace(const lbm_params* P) { return P->schedule == LBM_SCHEDULE_INPLACE; }
// the B_i are part of the stored state under BASELINE and INPLACE (the canonical 36 / 18 + 18 values)
bool use_fused(const lbm_params* P) { return P->schedule != LBM_SCHEDULE_BASELINE && !use_inplace(P); }

// one layout function serves both sizing (base == nullptr) and carving; everything that does not
// depend on the ghost count comes first, so a carve with ng = 0 and one with the real ng agree
// on those arrays
bool use_pack(const lbm_params* P) {
  return (P->schedule == LBM_SCHEDULE_PACK || P->schedule == LBM_SCHEDULE_AUTO || P->schedule == LBM_SCHEDULE_SPARSE) &&
         (P->nx % 2) == 0;
}
// SPARSE runs on the PACK layout when a group is 16 bytes (fp64 pairs, fp32 quads) and a row has enough groups
// for the two-group phi halo of a strip to wrap at most once
constexpr int kSpMaxCta = 1024;
bool use_sparse(const lbm_params* P) {
  if (P->schedule != LBM_SCHEDULE_SPARSE || !use_pack(P)) return false;
  const int G = pack_group(P->precision == 32 ? 4 : 8, P->nx);
  const int ng = P->nx / G;
  return G * (P->precision == 32 ? 4 : 8) == 16 && ng >= 4 && ng <= 65535;
}
int sp_strips(const lbm_params* P) {
  const int ng = P->nx / pack_group(P->precision == 32 ? 4 : 8, P->nx);
  return (ng + SP_S - 1) / SP_S;
}
size_t sp_march_capacity(const lbm_params* P) {
  return (size_t)sp_strips(P) * ((size_t)P->ny / SP_TYMAX + 2) + kSpMaxCta + 8;
}

// number of aligned node pairs that hold a fluid node (PACK schedule); mask: host, non-zero = solid
long long count_fluid_pairs(const lbm_params* P, const uint8_t* mask) {
  long long c = 0;
  const size_t n = (size_t)P->nx * P->ny;
  const size_t G = (size_t)pack_group(P->precision == 32 ? 4 : 8, P->nx);
  for (size_t k = 0; k + G <= n; k += G) {
    bool any = false;
    for (size_t t = 0; t < G; t++) any |= !mask[k + t];
    c += any ? 1 : 0;
  }
  return c;
}

constexpr size_t kStagePlanes = 3;   // host <-> device staging: nx*ny doubles each (phi0 + u0 of lbm_init is the largest user)

size_t layout(lbm_ctx* c, char* base, const lbm_params* P, long long ng, long long nfp) {
  const size_t n = (size_t)P->nx * P->ny;
  const size_t rs = P->precision == 32 ? 4 : 8;
  const size_t g = (size_t)(ng > 0 ? ng : 1);
  const size_t nblk = (n + 255) / 256;
  const bool fused = use_fused(P);
  Arena A{base, 0};
  const size_t ps = plane_stride(P);
  const int G = pack_group(P->precision == 32 ? 4 : 8, P->nx);
  const int nw = (P->nx / G + 31) / 32;
  const size_t cps = (((size_t)(nfp > 0 ? nfp : 1) + 63) & ~(size_t)63) + 37 * 64;
  // The populations come first (their size does not depend on the ghost count: lbm_create uses them as scratch
  // before lbm_init).  Compacted layouts (PACK / SPARSE) keep the two compact buffers and NO dense copy: every
  // call off the hot path reads and writes the compact planes through PopView.  B planes exist in the workspace
  // only where they are part of the state or of the fall-back kernels (dense layouts).
  char *N0 = nullptr, *N1 = nullptr, *B0 = nullptr, *B1 = nullptr, *Nc0 = nullptr, *Nc1 = nullptr;
  uint2* ptab = nullptr;
  if (use_pack(P)) {
    Nc0 = A.take<char>(9 * cps * G * rs);
    Nc1 = A.take<char>(9 * cps * G * rs);
    ptab = A.take<uint2>((size_t)P->ny * nw);
  } else {
    const bool single = use_inplace(P);   // INPLACE: one buffer of N and one of B
    N0 = A.take<char>(9 * ps * rs);
    N1 = single ? nullptr : A.take<char>(9 * ps * rs);
    B0 = A.take<char>(9 * ps * rs);
    B1 = (fused || single) ? nullptr : A.take<char>(9 * ps * rs);
  }
  char* p0 = A.take<char>(n * rs);
  char* p1 = A.take<char>(n * rs);
  uint8_t* cls = A.take<uint8_t>(n);
  uint8_t* links = A.take<uint8_t>(n);
  uint16_t* cl16 = A.take<uint16_t>(n + 2);   // +2: the WARP kernel copies aligned 4-byte pairs
  int* blk_cnt = A.take<int>(nblk);
  int* blk_off = A.take<int>(nblk);
  int* scal = A.take<int>(64);
  double* stage = A.take<double>(kStagePlanes * n + 64);
  double* diag_out = A.take<double>(8);
  const size_t samp_cap = 1 << 20;
  long long* samp = A.take<long long>(samp_cap);
  int* gidx = A.take<int>(g);
  int* corner = A.take<int>(4 * g);
  char* wgt = A.take<char>(4 * g * rs);
  double* wgt_d = A.take<double>(4 * g);
  double* gnx = A.take<double>(g);
  double* gny = A.take<double>(g);
  double* gdepth = A.take<double>(g);
  uint8_t* csolid = A.take<uint8_t>(g);
  uint2* gent_p = A.take<uint2>(g);
  char* gfr_p = A.take<char>(2 * g * rs);
  SpDesc* sp_desc = nullptr; uint16_t* sp_cnt = nullptr; uint2* sp_meta = nullptr; SpMarch* sp_march = nullptr; int* sp_first = nullptr;
  if (use_sparse(P)) {
    const size_t nsr = (size_t)sp_strips(P) * P->ny;
    sp_desc = A.take<SpDesc>(nsr);
    sp_cnt = A.take<uint16_t>(nsr + 8);
    sp_meta = A.take<uint2>((size_t)(nfp > 0 ? nfp : 1) + 64);
    sp_march = A.take<SpMarch>(sp_march_capacity(P));
    sp_first = A.take<int>(kSpMaxCta + 8);
  }
  if (c && base) {
    c->sp_desc = sp_desc; c->sp_cnt = sp_cnt; c->sp_meta = sp_meta; c->sp_march = sp_march; c->sp_first = sp_first;
    c->sp_march_cap = sp_march_capacity(P);
    c->N[0] = N0; c->N[1] = N1; c->B[0] = B0; c->B[1] = B1; c->phi[0] = p0; c->phi[1] = p1;
    c->cls = cls; c->links = links; c->cl16 = cl16; c->gidx = gidx; c->corner = corner; c->wgt = wgt; c->wgt_d = wgt_d;
    c->gnx = gnx; c->gny = gny; c->gdepth = gdepth; c->csolid = csolid;
    c->gent_p = gent_p; c->gfr_p = gfr_p;
    c->ptab = ptab; c->Nc[0] = Nc0; c->Nc[1] = Nc1; c->nw = nw; c->cps = cps; c->blk_cnt = blk_cnt;
    c->blk_off = blk_off; c->scal = scal; c->stage = stage; c->diag_out = diag_out;
    c->samp_idx = samp; c->samp_cap = samp_cap;
  }
  return ((A.off + 255) & ~(size_t)255) + 256;
}

template <typename R>
Consts<R> make_consts(const lbm_params& P) {
  Consts<R> C;
  const double alpha = 1.0 - 10.0 * P.mobility / 3.0;   // Eq. A7 text (:288) at reference p = 0 (R5)
  const double ct = cos(P.theta_deg * M_PI / 180.0);
  const double eps = -(4.0 / P.W) * ct;                 // Eq. 9 (:80), dx = 1
  C.nx = P.nx; C.ny = P.ny;
  C.ps = plane_stride(&P);
  C.rho_g = (R)P.rho_g; C.drho = (R)(P.rho_l - P.rho_g);
  C.inu_g = (R)(1.0 / P.nu_g); C.dinu = (R)(1.0 / P.nu_l - 1.0 / P.nu_g);
  C.s48W = (R)(P.sigma * 48.0 / P.W); C.s15W = (R)(P.sigma * 1.5 * P.W);
  C.twoW = (R)(2.0 / P.W);
  C.gbx = (R)P.gx; C.gby = (R)P.gy;
  C.chi0 = (R)alpha; C.chi1 = (R)((1.0 - alpha) / 5.0); C.chi5 = (R)((1.0 - alpha) / 20.0);
  C.E = (R)exp(eps); C.eps = (R)eps;
  C.phi_solid = (R)(0.5 * (1.0 + ct));
  C.ghost_rule = P.ghost_rule;
  C.all_links = 0;
  return C;
}

dim3 row_grid(int nx, int ny, int* bx) {
  int b = 256;
  while (b > 32 && b / 2 >= nx) b /= 2;
  *bx = b;
  return dim3((unsigned)((nx + b - 1) / b), (unsigned)ny, 1);
}

template <typename R> const Consts<R>& consts_of(const lbm_ctx* c);
template <> const Consts<double>& consts_of<double>(const lbm_ctx* c) { return c->Cd; }
template <> const Consts<float>& consts_of<float>(const lbm_ctx* c) { return c->Cf; }

// phi(t) fluid part is in phi[pcur]; finish it with the ghost update
template <typename R>
void launch_ghost(lbm_ctx* c) {
  if (c->ng == 0) return;
  k_ghost_update<R><<<(c->ng + 127) / 128, 128, 0, c->st>>>(
      consts_of<R>(c), c->ng, c->gent_p, (const typename GhostFrac<R>::T*)c->gfr_p,
      (const R*)c->phi[c->pcur ^ 1], (R*)c->phi[c->pcur]);
  c->launches[2]++;
}

bool launch_fused_sparse(lbm_ctx* c, const Consts<double>& C, const double* Ns, double* Nd, double* Bd, const double* pi, double* po);
bool launch_fused_sparse(lbm_ctx* c, const Consts<float>& C, const float* Ns, float* Nd, float* Bd, const float* pi, float* po);

// INPLACE: where the state is parked (lbm_kernels.cuh, k_collide_aa_*); the readers get it through Consts::all_links
void set_parking(lbm_ctx* c, bool local) {
  c->aa_local = local ? 1 : 0;
  c->Cd.all_links = c->Cf.all_links = c->aa_local;
}

struct StepTimer {   // optional event brackets around each launch (lbm_step_timed): 4 events per step, read in bulk
  cudaEvent_t* ev;   // the caller provides 4 events for this step
};

template <typename R>
int step_once(lbm_ctx* c, bool write_B, StepTimer* tm = nullptr) {
  int bx;
  if (tm) cudaEventRecord(tm->ev[0], c->st);
  const dim3 grid = row_grid(c->P.nx, c->P.ny, &bx);
  const Consts<R>& C = consts_of<R>(c);
  if (c->inplace) {   // AA pattern on the single N / B buffers (cur stays 0); phi ping-pongs as everywhere
    if (!c->aa_local)
      k_collide_aa_nbr<R><<<grid, bx, 0, c->st>>>(C, c->cls, c->links, (R*)c->N[0], (R*)c->B[0], (const R*)c->phi[c->pcur]);
    else
      k_collide_aa_local<R><<<grid, bx, 0, c->st>>>(C, c->cls, (R*)c->N[0], (R*)c->B[0], (const R*)c->phi[c->pcur]);
    set_parking(c, !c->aa_local);
    c->pcur ^= 1;
    if (tm) cudaEventRecord(tm->ev[1], c->st);
    k_phi_sum<R><<<grid, bx, 0, c->st>>>(consts_of<R>(c), c->cls, c->links, (const R*)c->B[0], (R*)c->phi[c->pcur]);
    c->launches[0]++;
    c->launches[1]++;
    c->B_valid = 1;
  } else if (!c->fused) {
    k_collide_baseline<R><<<grid, bx, 0, c->st>>>(C, c->cls, c->links, (const R*)c->N[c->cur],
                                                 (R*)c->N[c->cur ^ 1], (R*)c->B[c->cur ^ 1],
                                                 (const R*)c->phi[c->pcur]);
    c->cur ^= 1;
    c->pcur ^= 1;
    if (tm) cudaEventRecord(tm->ev[1], c->st);
    k_phi_sum<R><<<grid, bx, 0, c->st>>>(C, c->cls, c->links, (const R*)c->B[c->cur], (R*)c->phi[c->pcur]);
    c->launches[0]++;
    c->launches[1]++;
    c->B_valid = 1;
  } else {
    const R* Ns = (const R*)c->N[c->cur];
    R* Nd = (R*)c->N[c->cur ^ 1];
    R* Bd = write_B ? (R*)c->B[0] : nullptr;
    const R* pi = (const R*)c->phi[c->pcur];
    R* po = (R*)c->phi[c->pcur ^ 1];
    bool done = false;
    if (c->packed && c->sparse) {   // SPARSE: the same compact planes, lanes mapped to fluid groups
      done = launch_fused_sparse(c, C, (const R*)c->Nc[c->ccur], (R*)c->Nc[c->ccur ^ 1], Bd, pi, po);
      if (!done) return LBM_ECUDA;
      c->ccur ^= 1;
      c->cur ^= 1;     // undone below: the dense buffer index does not move
    } else if (c->packed) {   // PACK: compact planes step compact -> compact; the dense mirror N[cur] goes stale
      done = launch_fused_pack(C, c->cl16, (const R*)c->Nc[c->ccur], (R*)c->Nc[c->ccur ^ 1], Bd, pi, po, c->st, c->ptab,
                               c->nw, (unsigned)(c->cps * pack_group((int)sizeof(R), c->P.nx) * sizeof(R)));
      if (!done) return LBM_ECUDA;   // never step the stale dense mirror instead
      c->ccur ^= 1;
      c->cur ^= 1;     // undone below: the dense buffer index does not move
    }
    if (!done && c->sched == LBM_SCHEDULE_PAIR) done = launch_fused_pair(C, c->cl16, Ns, Nd, Bd, pi, po, c->st);   // false: odd nx
    if (!done) launch_fused_step<R>(C, c->cls, c->links, Ns, Nd, Bd, pi, po, c->st);
    c->cur ^= 1;
    c->pcur ^= 1;
    c->launches[0]++;
    c->B_valid = write_B ? 1 : 0;
    if (tm) cudaEventRecord(tm->ev[1], c->st);
  }
  if (tm) cudaEventRecord(tm->ev[2], c->st);
  launch_ghost<R>(c);
  c->t++;
  if (tm) cudaEventRecord(tm->ev[3], c->st);
  return LBM_OK;
}


// SPARSE schedule: one persistent CTA per SM (lbm_sparse.cuh)
template <typename V, typename R>
bool launch_sparse_v(lbm_ctx* c, const Consts<R>& C, const R* Ns, R* Nd, R* Bd, const R* pi, R* po) {
  const size_t smem = sizeof(SpSmem<V>);
  auto kern = Bd ? k_fused_sparse<V, true> : k_fused_sparse<V, false>;
  if (!ensure_smem_attr(reinterpret_cast<const void*>(kern), smem)) return false;
  kern<<<c->sp_ncta, SP_THREADS, smem, c->st>>>(C, Ns, Nd, Bd, pi, po, c->sp_desc, c->sp_cnt, c->sp_meta, c->sp_march,
                                               c->sp_first, c->sp_sw);
  return true;
}
bool launch_fused_sparse(lbm_ctx* c, const Consts<double>& C, const double* Ns, double* Nd, double* Bd, const double* pi,
                         double* po) {
  return launch_sparse_v<D2, double>(c, C, Ns, Nd, Bd, pi, po);
}
bool launch_fused_sparse(lbm_ctx* c, const Consts<float>& C, const float* Ns, float* Nd, float* Bd, const float* pi,
                         float* po) {
  return launch_sparse_v<Q4, float>(c, C, Ns, Nd, Bd, pi, po);
}

// SPARSE schedule, one-time: cut the (strip, row) sequence into marches of about equal weight, one run of
// marches per CTA.  cnt[strip * ny + row] = entries of that strip row.
void sp_partition(const uint16_t* cnt, int nstrips, int ny, int ncta_max, std::vector<SpMarch>& marches,
                  std::vector<int>& first) {
  double total = 0.0;
  auto weight = [&](int s, int r) { return (double)std::max<int>(cnt[(size_t)s * ny + r], SP_MINPOS) + 12.0; };
  for (int s = 0; s < nstrips; s++)
    for (int r = 0; r < ny; r++) total += weight(s, r);
  // a CTA should have at least ~64 rows of a full strip to amortise its 4 halo rows
  int ncta = (int)std::min<double>(ncta_max, std::max(1.0, total / (64.0 * (SP_S + 4))));
  const double target = total / ncta;
  marches.clear();
  first.assign(1, 0);
  double cum = 0.0;
  int cur = 0;
  for (int s = 0; s < nstrips; s++) {
    int r = 0;
    while (r < ny) {
      const int owner = std::min(ncta - 1, (int)(cum / target));
      while (cur < owner) { first.push_back((int)marches.size()); cur++; }
      SpMarch m{s, r, 0, 0};
      while (r < ny && m.rows < SP_TYMAX && std::min(ncta - 1, (int)(cum / target)) == owner) {
        cum += weight(s, r);
        r++;
        m.rows++;
      }
      marches.push_back(m);
    }
  }
  while (cur < ncta) { first.push_back((int)marches.size()); cur++; }
}

// the populations of the current time, wherever they live (dense planes or the compact buffers of PACK / SPARSE)
template <typename R>
PopView<R> pop_view(const lbm_ctx* c) {
  if (c->packed)
    return PopView<R>{(R*)c->Nc[c->ccur], 0, c->ptab, c->P.nx, c->nw, pack_group((int)sizeof(R), c->P.nx), c->sparse, c->cps};
  return dense_view<R>((R*)c->N[c->cur], plane_stride(&c->P), c->P.nx);
}
template <typename R>
PopView<R> B_view(const lbm_ctx* c) {
  return dense_view<R>((R*)(c->fused ? c->B[0] : c->B[c->cur]), plane_stride(&c->P), c->P.nx);
}


// lbm_rows_*: the pieces of the state that belong to rows [j0, j0 + nrows): phi (dense rows) and the nine population
// planes (dense rows, or the rows' run of groups in the compact planes; BASELINE: the nine B planes too).  Each piece
// is one contiguous device range.
struct RowPiece { char* p; size_t bytes; };
int row_pieces(lbm_ctx* ctx, int j0, int nrows, RowPiece (&pc)[19], int* npc) {
  const lbm_params& P = ctx->P;
  if (j0 < 0 || nrows < 1 || (long long)j0 + nrows > P.ny) return fail(ctx, LBM_EINVAL, "rows outside the grid (ranges do not wrap)");
  const size_t rs = ctx->is32 ? 4 : 8;
  int k = 0;
  pc[k++] = RowPiece{(char*)ctx->phi[ctx->pcur] + (size_t)j0 * P.nx * rs, (size_t)nrows * P.nx * rs};
  if (!ctx->packed) {
    const size_t ps = plane_stride(&P);
    for (int q = 0; q < 9; q++)
      pc[k++] = RowPiece{(char*)ctx->N[ctx->cur] + ((size_t)q * ps + (size_t)j0 * P.nx) * rs, (size_t)nrows * P.nx * rs};
    if (!ctx->fused)   // BASELINE: the B_i are part of the stored state
      for (int q = 0; q < 9; q++)
        pc[k++] = RowPiece{(char*)ctx->B[ctx->cur] + ((size_t)q * ps + (size_t)j0 * P.nx) * rs, (size_t)nrows * P.nx * rs};
  } else {
    if (!ctx->row_base) {
      unsigned* rb = (unsigned*)malloc(((size_t)P.ny + 1) * sizeof(unsigned));
      if (!rb) return fail(ctx, LBM_ENOMEM, "host allocation failed");
      // .y of the first table word of every row
      cudaError_t e = cudaMemcpy2DAsync(rb, sizeof(unsigned), (const char*)ctx->ptab + sizeof(unsigned), (size_t)ctx->nw * sizeof(uint2),
                                        sizeof(unsigned), (size_t)P.ny, cudaMemcpyDeviceToHost, ctx->st);
      if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->st);
      if (e != cudaSuccess) { free(rb); return cuda_fail(ctx, e, "row table"); }
      rb[P.ny] = (unsigned)ctx->nfp;
      ctx->row_base = rb;
    }
    const size_t G = (size_t)pack_group((int)rs, P.nx);
    const size_t g0 = ctx->row_base[j0], g1 = ctx->row_base[j0 + nrows];
    char* base = (char*)ctx->Nc[ctx->ccur];
    if (g1 > g0) {
      if (ctx->sparse) pc[k++] = RowPiece{base + g0 * 9 * G * rs, (g1 - g0) * 9 * G * rs};   // group-major
      else
        for (int q = 0; q < 9; q++) pc[k++] = RowPiece{base + ((size_t)q * ctx->cps + g0) * G * rs, (g1 - g0) * G * rs};
    }
  }
  *npc = k;
  return LBM_OK;
}

// lbm_rows_export / lbm_rows_import: the contiguous pieces of some grid rows' state (phi rows, the rows' run in every
// population plane) to / from one packed buffer, 16 bytes per thread; TO_BUF packs, else unpacks.
struct RowPieces {
  char* p[19];
  unsigned long long end[19];   // running end offset of every piece in the packed buffer, in 16-byte units
  int n;
};
template <bool TO_BUF>
__global__ void __launch_bounds__(256) k_rows_copy(const RowPieces P, char* __restrict__ buf, unsigned long long total16) {
  for (unsigned long long t = (unsigned long long)blockIdx.x * 256 + threadIdx.x; t < total16;
       t += (unsigned long long)gridDim.x * 256) {
    int k = 0;
    while (k < P.n - 1 && t >= P.end[k]) k++;
    const unsigned long long in_piece = t - (k ? P.end[k - 1] : 0ull);
    uint4* a = reinterpret_cast<uint4*>(P.p[k]) + in_piece;
    uint4* b = reinterpret_cast<uint4*>(buf) + t;
    if (TO_BUF) *b = *a;
    else *a = *b;
  }
}

// one launch when every piece is 16-byte aligned (always, unless nx is odd), else one copy per piece
template <bool TO_BUF>
int rows_copy(lbm_ctx* ctx, const RowPiece* pc, int n, char* buf) {
  bool vec = ((uintptr_t)buf & 15) == 0;
  size_t total = 0;
  for (int i = 0; i < n; i++) { vec = vec && ((uintptr_t)pc[i].p & 15) == 0 && (pc[i].bytes & 15) == 0; total += pc[i].bytes; }
  if (vec && total > 0) {
    RowPieces P;
    P.n = n;
    unsigned long long e = 0;
    for (int i = 0; i < n; i++) { P.p[i] = pc[i].p; e += pc[i].bytes / 16; P.end[i] = e; }
    const unsigned nb = (unsigned)std::min<unsigned long long>((e + 255) / 256, 148ull * 16);
    k_rows_copy<TO_BUF><<<nb, 256, 0, ctx->st>>>(P, buf, e);
    CK(cudaGetLastError());
    return LBM_OK;
  }
  size_t off = 0;
  for (int i = 0; i < n; i++) {
    if (TO_BUF) CK(cudaMemcpyAsync(buf + off, pc[i].p, pc[i].bytes, cudaMemcpyDeviceToDevice, ctx->st));
    else CK(cudaMemcpyAsync(pc[i].p, buf + off, pc[i].bytes, cudaMemcpyDeviceToDevice, ctx->st));
    off += pc[i].bytes;
  }
  return LBM_OK;
}

}  // namespace

extern "C" {

const char* lbm_version(void) { return "liblbm_b200 0.2 (sm_100a)"; }

const char* lbm_last_error(const lbm_ctx* ctx) { return ctx ? ctx->err : g_err; }

int lbm_plan(const lbm_params* prm, const uint8_t* mask, int64_t* n_ghost, size_t* workspace_bytes) {
  lbm_ctx* ctx = nullptr;
  const char* why;
  if (validate(prm, &why) != LBM_OK) return fail(nullptr, LBM_EINVAL, why);
  if (!mask) return fail(nullptr, LBM_EINVAL, "null mask");
  if (check_walls(prm, mask) != LBM_OK) return fail(nullptr, LBM_EINVAL, "wall rows are not solid in the mask");
  const size_t n = (size_t)prm->nx * prm->ny;
  uint8_t* d_mask = nullptr;
  unsigned long long* d_tot = nullptr;
  CK(cudaMalloc(&d_mask, n + 8));
  cudaError_t e = cudaMalloc(&d_tot, 8);
  if (e != cudaSuccess) { cudaFree(d_mask); return cuda_fail(nullptr, e, "cudaMalloc"); }
  unsigned long long tot = 0;
  e = cudaMemcpy(d_mask, mask, n, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemset(d_tot, 0, 8);
  if (e == cudaSuccess) {
    k_classify<<<(unsigned)((n + 255) / 256), 256>>>(d_mask, prm->nx, prm->ny, nullptr, nullptr, nullptr, d_tot);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpy(&tot, d_tot, 8, cudaMemcpyDeviceToHost);
  cudaFree(d_mask);
  cudaFree(d_tot);
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "lbm_plan");
  if (n_ghost) *n_ghost = (int64_t)tot;
  if (workspace_bytes) *workspace_bytes = layout(nullptr, nullptr, prm, (long long)tot, use_pack(prm) ? count_fluid_pairs(prm, mask) : 0);
  return LBM_OK;
}

double lbm_nu_from_tau(double tau) { return (tau - 0.5) / 3.0; }
double lbm_tau_from_nu(double nu) { return 0.5 + 3.0 * nu; }

size_t lbm_workspace_bytes(const lbm_params* prm, int64_t n_ghost_bound) {
  const char* why;
  if (validate(prm, &why) != LBM_OK || n_ghost_bound < 0) return 0;
  const long long groups = ((long long)prm->nx * prm->ny + 1) / 2;   // no more groups than node pairs
  return layout(nullptr, nullptr, prm, (long long)n_ghost_bound, use_pack(prm) ? groups : 0);
}

int lbm_create(lbm_ctx** out, const lbm_params* prm, const uint8_t* mask, const lbm_disk* disks,
               int32_t n_disks, void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  lbm_ctx* ctx = nullptr;
  if (!out) return fail(nullptr, LBM_EINVAL, "null out");
  *out = nullptr;
  const char* why;
  if (validate(prm, &why) != LBM_OK) return fail(nullptr, LBM_EINVAL, why);
  if (!mask) return fail(nullptr, LBM_EINVAL, "null mask");
  if (n_disks < 0 || (n_disks > 0 && !disks)) return fail(nullptr, LBM_EINVAL, "bad disk list");
  if (check_walls(prm, mask) != LBM_OK) return fail(nullptr, LBM_EINVAL, "wall rows are not solid in the mask");
  if (!d_workspace || ((uintptr_t)d_workspace & 255)) return fail(nullptr, LBM_EINVAL, "workspace null or not 256-byte aligned");
  const size_t n = (size_t)prm->nx * prm->ny;
  // the disk list and the mask upload need room before the ghost count is known
  const long long nfp = use_pack(prm) ? count_fluid_pairs(prm, mask) : 0;
  const size_t min_ws = layout(nullptr, nullptr, prm, 0, nfp);
  if (workspace_bytes < min_ws) return fail(nullptr, LBM_ENOMEM, "workspace too small");

  lbm_ctx* c = new (std::nothrow) lbm_ctx;
  if (!c) return fail(nullptr, LBM_ENOMEM, "host allocation failed");
  memset(c, 0, sizeof *c);
  ctx = c;
  c->P = *prm;
  c->n = n;
  c->is32 = prm->precision == 32;
  c->fused = use_fused(prm) ? 1 : 0;
  c->inplace = use_inplace(prm) ? 1 : 0;
  c->sched = prm->schedule == LBM_SCHEDULE_AUTO ? (use_pack(prm) ? LBM_SCHEDULE_PACK : LBM_SCHEDULE_PAIR) : prm->schedule;
  if (c->sched == LBM_SCHEDULE_SPARSE && !use_sparse(prm)) c->sched = use_pack(prm) ? LBM_SCHEDULE_PACK : LBM_SCHEDULE_PAIR;
  c->st = (cudaStream_t)cuda_stream;
  c->Cd = make_consts<double>(*prm);
  c->Cf = make_consts<float>(*prm);
  layout(c, (char*)d_workspace, prm, 0, nfp);   // provisional carve: cls/links/blk arrays do not depend on ng

#define CKC(call)                                                              \
  do {                                                                         \
    cudaError_t e_ = (call);                                                   \
    if (e_ != cudaSuccess) { int rc_ = cuda_fail(nullptr, e_, #call); delete c; return rc_; } \
  } while (0)

  // temporaries of this call are carved from the dense population planes, which hold nothing before lbm_init
  Arena scratch{(char*)(c->Nc[0] ? c->Nc[0] : c->N[0]), 0};
  const size_t rs_ = c->is32 ? 4 : 8;
  const size_t scratch_cap = c->Nc[0] ? 2 * 9 * c->cps * (size_t)pack_group((int)rs_, prm->nx) * rs_   // both compact buffers
                                      : 2 * 9 * plane_stride(prm) * rs_;                               // both dense buffers
  auto scratch_take = [&](size_t bytes) -> void* {
    char* p0 = scratch.take<char>(bytes);
    return scratch.off <= scratch_cap ? p0 : nullptr;
  };

  // (1) classification; the mask is staged in the (not yet used) stage area
  uint8_t* d_mask = reinterpret_cast<uint8_t*>(c->stage);
  const unsigned nblk = (unsigned)((n + 255) / 256);
  CKC(cudaMemcpyAsync(d_mask, mask, n, cudaMemcpyHostToDevice, c->st));
  k_classify<<<nblk, 256, 0, c->st>>>(d_mask, prm->nx, prm->ny, c->cls, c->links, c->blk_cnt, nullptr);
  k_scan_blocks<<<1, 1024, 0, c->st>>>(c->blk_cnt, (int)nblk, c->blk_off, c->scal);
  k_pack_cl16<<<nblk, 256, 0, c->st>>>(c->cls, c->links, (long long)n, c->cl16);
  CKC(cudaGetLastError());
  int ng = 0;
  CKC(cudaMemcpyAsync(&ng, c->scal, sizeof(int), cudaMemcpyDeviceToHost, c->st));
  CKC(cudaStreamSynchronize(c->st));
  c->ng = ng;
  const size_t need = layout(nullptr, nullptr, prm, ng, nfp);
  if (workspace_bytes < need) {
    delete c;
    return fail(nullptr, LBM_ENOMEM, "workspace too small for the ghost list (size it with lbm_plan)");
  }
  layout(c, (char*)d_workspace, prm, ng, nfp);   // ghost arrays now have their real extent

  // (2) index-sorted ghost list and per-ghost geometry
  if (ng > 0) {
    k_compact_ghosts<<<nblk, 256, 0, c->st>>>(c->cls, (long long)n, c->blk_off, c->gidx);
    // disk list staged behind the mask copy in the stage area (5n doubles >= n bytes + disks?)
    const size_t disk_bytes = (size_t)n_disks * sizeof(Disk);
    const size_t stage_bytes = (kStagePlanes * n + 64) * sizeof(double);
    const size_t disk_off = (n + 255) & ~(size_t)255;
    if (disk_off + disk_bytes > stage_bytes) {
      delete c;
      return fail(nullptr, LBM_EINVAL, "too many disks for this grid");
    }
    Disk* d_disks = reinterpret_cast<Disk*>(reinterpret_cast<char*>(c->stage) + disk_off);
    static_assert(sizeof(Disk) == sizeof(lbm_disk), "disk layout");
    if (n_disks > 0) CKC(cudaMemcpyAsync(d_disks, disks, disk_bytes, cudaMemcpyHostToDevice, c->st));
    CKC(cudaMemsetAsync(c->scal + 1, 0, sizeof(int), c->st));
    const unsigned gb = (unsigned)((ng + 127) / 128);
    int ncx = 1;
    std::vector<int> h_start, h_list;
    build_disk_cells(prm, disks, n_disks, &ncx, h_start, h_list);
    int* d_cells = (int*)scratch_take((h_start.size() + h_list.size()) * sizeof(int));   // [start | list]
    if (!d_cells) { delete c; return fail(nullptr, LBM_ENOMEM, "workspace too small for the disk cell lists"); }
    int* d_start = d_cells;
    int* d_list = d_cells + h_start.size();
    cudaMemcpyAsync(d_start, h_start.data(), h_start.size() * sizeof(int), cudaMemcpyHostToDevice, c->st);
    cudaMemcpyAsync(d_list, h_list.data(), h_list.size() * sizeof(int), cudaMemcpyHostToDevice, c->st);
    int* d_smooth = nullptr;   // mask-only normals (n_disks == 0): the solid indicator smoothed twice
    if (n_disks == 0) {
      d_smooth = (int*)scratch_take(2 * n * sizeof(int));
      if (!d_smooth) { delete c; return fail(nullptr, LBM_ENOMEM, "workspace too small for the mask-normal temporaries"); }
      k_mask_smooth<<<nblk, 256, 0, c->st>>>(c->cls, nullptr, d_smooth + n, prm->nx, prm->ny);
      k_mask_smooth<<<nblk, 256, 0, c->st>>>(nullptr, d_smooth + n, d_smooth, prm->nx, prm->ny);
    }
    double2* d_gfrac = (double2*)scratch_take((size_t)ng * sizeof(double2));   // (f_x, f_y) of x_F, consumed by k_ghost_permute
    if (!d_gfrac) { delete c; return fail(nullptr, LBM_ENOMEM, "workspace too small for the ghost geometry temporaries"); }
    if (c->is32)
      k_ghost_geometry<float><<<gb, 128, 0, c->st>>>(ng, c->gidx, prm->nx, prm->ny, prm->wall_rows, d_disks,
                                                     n_disks, d_start, d_list, ncx, kCell, d_smooth, c->cls, c->gnx, c->gny, c->gdepth, c->corner,
                                                     c->wgt_d, (float*)c->wgt, c->csolid, d_gfrac, c->scal + 1);
    else
      k_ghost_geometry<double><<<gb, 128, 0, c->st>>>(ng, c->gidx, prm->nx, prm->ny, prm->wall_rows, d_disks,
                                                      n_disks, d_start, d_list, ncx, kCell, d_smooth, c->cls, c->gnx, c->gny, c->gdepth, c->corner,
                                                      c->wgt_d, (double*)c->wgt, c->csolid, d_gfrac, c->scal + 1);
    CKC(cudaGetLastError());
    int bad = 0;
    cudaMemcpyAsync(&bad, c->scal + 1, sizeof(int), cudaMemcpyDeviceToHost, c->st);
    {
      const cudaError_t e = cudaStreamSynchronize(c->st);
      if (e != cudaSuccess) { delete c; return cuda_fail(nullptr, e, "ghost geometry"); }
    }
    if (bad) {
      delete c;
      return fail(nullptr, LBM_EINVAL, "mask and geometry disagree: a ghost node lies in no disk");
    }
    // tile-major processing order for the ghost update (one-time)
    {
      unsigned *k_in = nullptr, *k_out = nullptr;
      int *v_in = nullptr, *v_out = nullptr;
      void* tmp = nullptr;
      size_t tmp_bytes = 0;
      k_in = (unsigned*)scratch_take(4 * sizeof(int) * (size_t)ng);
      if (!k_in) { delete c; return fail(nullptr, LBM_ENOMEM, "workspace too small for the ghost ordering"); }
      cudaError_t e = cudaSuccess;
      k_out = k_in + ng; v_in = reinterpret_cast<int*>(k_out + ng); v_out = v_in + ng;
      k_ghost_tile_keys<<<(ng + 255) / 256, 256, 0, c->st>>>(ng, c->gidx, prm->nx, k_in, v_in);
      e = cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, k_in, k_out, v_in, v_out, ng, 0, 32, c->st);
      if (e == cudaSuccess && !(tmp = scratch_take(tmp_bytes ? tmp_bytes : 1))) { delete c; return fail(nullptr, LBM_ENOMEM, "workspace too small for the ghost ordering"); }
      if (e == cudaSuccess) e = cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, k_in, k_out, v_in, v_out, ng, 0, 32, c->st);
      if (e == cudaSuccess) {
        if (c->is32)
          k_ghost_permute<float><<<(ng + 255) / 256, 256, 0, c->st>>>(ng, v_out, c->gidx, (const int4*)c->corner, d_gfrac, c->csolid,
                                                                      prm->nx, prm->ny, c->gent_p, (float2*)c->gfr_p);
        else
          k_ghost_permute<double><<<(ng + 255) / 256, 256, 0, c->st>>>(ng, v_out, c->gidx, (const int4*)c->corner, d_gfrac, c->csolid,
                                                                       prm->nx, prm->ny, c->gent_p, (double2*)c->gfr_p);
        e = cudaGetLastError();
      }
      if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
      if (e != cudaSuccess) { delete c; return cuda_fail(nullptr, e, "ghost processing order"); }
    }
  }
  if (use_pack(prm)) {   // PACK schedule: pair mask words and their compact base indices
    const long long nwords = (long long)prm->ny * c->nw;
    void* tmp = nullptr;
    size_t tmp_bytes = 0;
    scratch.off = 0;
    unsigned* pmask = (unsigned*)scratch_take(3 * sizeof(int) * (size_t)nwords + 16);
    if (!pmask) { delete c; return fail(nullptr, LBM_ENOMEM, "workspace too small for the group table temporaries"); }
    cudaError_t e = cudaSuccess;
    int* pcount = reinterpret_cast<int*>(pmask + nwords);
    int* pbase = pcount + nwords;
    const unsigned nb = (unsigned)((nwords + 255) / 256);
    k_pair_mask<<<nb, 256, 0, c->st>>>(c->cls, prm->nx, prm->ny, c->nw, pack_group(c->is32 ? 4 : 8, prm->nx), pmask, pcount);
    e = cub::DeviceScan::ExclusiveSum(nullptr, tmp_bytes, pcount, pbase, (int)nwords, c->st);
    if (e == cudaSuccess && !(tmp = scratch_take(tmp_bytes ? tmp_bytes : 1))) { delete c; return fail(nullptr, LBM_ENOMEM, "workspace too small for the group table temporaries"); }
    if (e == cudaSuccess) e = cub::DeviceScan::ExclusiveSum(tmp, tmp_bytes, pcount, pbase, (int)nwords, c->st);
    if (e == cudaSuccess) {
      k_pair_tab<<<nb, 256, 0, c->st>>>(pmask, pbase, nwords, c->ptab);
      e = cudaGetLastError();
    }
    int last[2] = {0, 0};   // the device's group count must be the host's (the compact planes were sized with it)
    if (e == cudaSuccess) e = cudaMemcpyAsync(&last[0], pbase + (nwords - 1), sizeof(int), cudaMemcpyDeviceToHost, c->st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&last[1], pcount + (nwords - 1), sizeof(int), cudaMemcpyDeviceToHost, c->st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->st);
    if (e != cudaSuccess) { delete c; return cuda_fail(nullptr, e, "pair table"); }
    if ((long long)last[0] + last[1] != nfp) { delete c; return fail(nullptr, LBM_EINVAL, "internal: fluid group counts of host and device differ"); }
    c->packed = 1;
    c->nfp = nfp;
  }
  if (use_sparse(prm)) {   // SPARSE schedule: per-group metadata, per (strip, row) descriptors, marches
    const int G = pack_group(c->is32 ? 4 : 8, prm->nx);
    const int ng = prm->nx / G;
    const int nstrips = sp_strips(prm);
    const size_t nsr = (size_t)nstrips * prm->ny;
    k_sp_meta<<<(unsigned)(((long long)prm->ny * ng + 255) / 256), 256, 0, c->st>>>(c->cls, c->links, c->ptab, prm->nx, prm->ny,
                                                                                 c->nw, G, c->sp_meta);
    const int sw = (ng + nstrips - 1) / nstrips;   // strips of equal width (<= SP_S groups)
    c->sp_sw = sw;
    k_sp_desc<<<(unsigned)((nsr + 127) / 128), 128, 0, c->st>>>(c->ptab, c->sp_meta, prm->nx, prm->ny, c->nw, G, nstrips, sw,
                                                               c->sp_desc, c->sp_cnt);
    CKC(cudaGetLastError());
    std::vector<uint16_t> h_cnt(nsr);
    CKC(cudaMemcpyAsync(h_cnt.data(), c->sp_cnt, nsr * sizeof(uint16_t), cudaMemcpyDeviceToHost, c->st));
    CKC(cudaStreamSynchronize(c->st));
    int dev = 0, nsm = 0;
    CKC(cudaGetDevice(&dev));
    CKC(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    std::vector<SpMarch> marches;
    std::vector<int> first;
    sp_partition(h_cnt.data(), nstrips, prm->ny, std::min(nsm, kSpMaxCta), marches, first);
    if (marches.size() > c->sp_march_cap) { delete c; return fail(nullptr, LBM_EINVAL, "internal: march table overflow"); }
    CKC(cudaMemcpyAsync(c->sp_march, marches.data(), marches.size() * sizeof(SpMarch), cudaMemcpyHostToDevice, c->st));
    CKC(cudaMemcpyAsync(c->sp_first, first.data(), first.size() * sizeof(int), cudaMemcpyHostToDevice, c->st));
    CKC(cudaStreamSynchronize(c->st));
    c->sp_nstrips = nstrips;
    c->sp_ncta = (int)first.size() - 1;
    c->sp_nmarch = (int)marches.size();
    c->sparse = 1;
  }
  CKC(cudaStreamSynchronize(c->st));
#undef CKC
  c->diag_static_err = (int)static_scratch_of(&c->diag_static);   // a failure is reported by lbm_diag_static, not here
  *out = c;
  return LBM_OK;
}

void lbm_destroy(lbm_ctx* ctx) {
  if (!ctx) return;
  for (auto& g : ctx->gexec)
    if (g) cudaGraphExecDestroy(g);
  if (ctx->B_owned) cudaFree(ctx->B[0]);
  free(ctx->row_base);
  delete ctx;
}

int lbm_init(lbm_ctx* ctx, const double* phi0, const double* u0) {
  if (!ctx || !phi0) return fail(ctx, LBM_EINVAL, "null argument");
  const size_t n = ctx->n;
  double* d_phi0 = ctx->stage;
  double* d_u0 = u0 ? ctx->stage + n : nullptr;
  CK(cudaMemcpyAsync(d_phi0, phi0, n * sizeof(double), cudaMemcpyHostToDevice, ctx->st));
  if (u0) CK(cudaMemcpyAsync(d_u0, u0, 2 * n * sizeof(double), cudaMemcpyHostToDevice, ctx->st));
  ctx->cur = 0;
  ctx->pcur = 0;
  ctx->t = 0;
  set_parking(ctx, false);   // k_init writes the standard parking
  int bx;
  const dim3 grid = row_grid(ctx->P.nx, ctx->P.ny, &bx);
  ctx->ccur = 0;
  void* Bp = ctx->fused ? ctx->B[0] : ctx->B[ctx->cur];   // may be absent (compacted layout without lbm_keep_B)
  if (ctx->is32)
    k_init<float><<<grid, bx, 0, ctx->st>>>(ctx->Cf, ctx->cls, ctx->links, d_phi0, d_u0, pop_view<float>(ctx),
                                            (float*)Bp, (float*)ctx->phi[0], (float*)ctx->phi[1]);
  else
    k_init<double><<<grid, bx, 0, ctx->st>>>(ctx->Cd, ctx->cls, ctx->links, d_phi0, d_u0, pop_view<double>(ctx),
                                             (double*)Bp, (double*)ctx->phi[0], (double*)ctx->phi[1]);
  ctx->launches[3]++;
  ctx->B_valid = Bp ? 1 : 0;
  if (ctx->is32) launch_ghost<float>(ctx); else launch_ghost<double>(ctx);
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(ctx->st));
  return LBM_OK;
}

namespace {
constexpr int kGraphSteps = 32;                    // even: the ping-pong indices return to where they started
constexpr size_t kGraphMaxNodes = (size_t)1 << 22; // larger grids run milliseconds per kernel: nothing to gain
}

int lbm_step(lbm_ctx* ctx, int64_t nsteps) {
  if (!ctx || nsteps < 0) return fail(ctx, LBM_EINVAL, "bad argument");
  int64_t s = 0;
  // the legacy default stream cannot be captured; with keep_B the last step differs from the others
  if (ctx->st != nullptr && ctx->st != cudaStreamLegacy && !ctx->keep_B && !ctx->inplace && ctx->n <= kGraphMaxNodes) {
    if (!ctx->graph_warm && nsteps - s >= kGraphSteps + 2) {   // first launches outside any capture
      for (int k = 0; k < 2; k++, s++)
        if ((ctx->is32 ? step_once<float>(ctx, false) : step_once<double>(ctx, false)) != LBM_OK)
          return cuda_fail(ctx, cudaGetLastError(), "kernel launch of lbm_step");
      ctx->graph_warm = 1;
    }
    while (ctx->graph_warm && nsteps - s >= kGraphSteps) {
      const int key = (ctx->cur & 1) | ((ctx->pcur & 1) << 1) | ((ctx->ccur & 1) << 2);
      if (!ctx->gexec[key]) {   // capture kGraphSteps steps once, then run them
        int64_t before[4];
        for (int k = 0; k < 4; k++) before[k] = ctx->launches[k];
        if (cudaStreamBeginCapture(ctx->st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); break; }
        int rc = LBM_OK;
        for (int k = 0; k < kGraphSteps && rc == LBM_OK; k++)
          rc = ctx->is32 ? step_once<float>(ctx, false) : step_once<double>(ctx, false);
        cudaGraph_t g = nullptr;
        const cudaError_t e = cudaStreamEndCapture(ctx->st, &g);
        if (rc != LBM_OK || e != cudaSuccess || !g) {
          if (g) cudaGraphDestroy(g);
          return cuda_fail(ctx, e != cudaSuccess ? e : cudaGetLastError(), "capture of the step graph");
        }
        const cudaError_t ei = cudaGraphInstantiate(&ctx->gexec[key], g, 0);
        cudaGraphDestroy(g);
        if (ei != cudaSuccess) { ctx->gexec[key] = nullptr; return cuda_fail(ctx, ei, "cudaGraphInstantiate"); }
        for (int k = 0; k < 4; k++) ctx->gdelta[key][k] = ctx->launches[k] - before[k];
        // the capture advanced the bookkeeping by kGraphSteps steps: this launch executes them
      } else {
        ctx->t += kGraphSteps;
        for (int k = 0; k < 4; k++) ctx->launches[k] += ctx->gdelta[key][k];
        ctx->B_valid = ctx->fused ? 0 : 1;
      }
      CK(cudaGraphLaunch(ctx->gexec[key], ctx->st));
      s += kGraphSteps;
    }
  }
  for (; s < nsteps; s++) {
    const bool wb = ctx->fused && ctx->keep_B && s == nsteps - 1;
    const int rc = ctx->is32 ? step_once<float>(ctx, wb) : step_once<double>(ctx, wb);
    if (rc != LBM_OK) {
      const cudaError_t e = cudaGetLastError();
      return cuda_fail(ctx, e, "kernel launch of lbm_step (the state did not advance past the failed step)");
    }
  }
  CK(cudaGetLastError());
  return LBM_OK;
}

int lbm_step_timed(lbm_ctx* ctx, int64_t nsteps, double ms[3]) {
  if (!ctx || nsteps < 0 || !ms) return fail(ctx, LBM_EINVAL, "bad argument");
  // events of a chunk of steps are recorded without any host synchronisation in between and read afterwards
  const int chunk = 256;
  std::vector<cudaEvent_t> ev(4 * chunk);
  for (auto& e : ev) CK(cudaEventCreate(&e));
  double acc[3] = {0.0, 0.0, 0.0};
  CK(cudaStreamSynchronize(ctx->st));
  int rc = LBM_OK;
  for (int64_t s0 = 0; s0 < nsteps && rc == LBM_OK; s0 += chunk) {
    const int m = (int)std::min<int64_t>(chunk, nsteps - s0);
    for (int k = 0; k < m && rc == LBM_OK; k++) {
      StepTimer tm{&ev[4 * k]};
      const bool wb = ctx->fused && ctx->keep_B && s0 + k == nsteps - 1;
      rc = ctx->is32 ? step_once<float>(ctx, wb, &tm) : step_once<double>(ctx, wb, &tm);
    }
    if (rc != LBM_OK) break;
    if (cudaEventSynchronize(ev[4 * (m - 1) + 3]) != cudaSuccess) { rc = LBM_ECUDA; break; }
    for (int k = 0; k < m; k++)
      for (int j = 0; j < 3; j++) {
        float t = 0.f;
        cudaEventElapsedTime(&t, ev[4 * k + j], ev[4 * k + j + 1]);
        acc[j] += t;
      }
  }
  for (auto& e : ev) cudaEventDestroy(e);
  if (rc != LBM_OK) return cuda_fail(ctx, cudaGetLastError(), "kernel launch of lbm_step_timed");
  CK(cudaGetLastError());
  for (int k = 0; k < 3; k++) ms[k] = acc[k];
  return LBM_OK;
}

int lbm_sync(lbm_ctx* ctx) {
  if (!ctx) return fail(ctx, LBM_EINVAL, "null context");
  CK(cudaStreamSynchronize(ctx->st));
  return LBM_OK;
}

int lbm_keep_B(lbm_ctx* ctx, int32_t on) {
  if (!ctx) return fail(ctx, LBM_EINVAL, "null context");
  if (on && ctx->fused && !ctx->B[0]) {   // compacted layouts carry no B planes in the workspace: allocate them now
    const size_t bytes = 9 * plane_stride(&ctx->P) * (size_t)(ctx->is32 ? 4 : 8);
    void* b = nullptr;
    CK(cudaMalloc(&b, bytes));
    CK(cudaMemsetAsync(b, 0, bytes, ctx->st));
    ctx->B[0] = b;
    ctx->B_owned = 1;
    ctx->B_valid = 0;
  }
  ctx->keep_B = on ? 1 : 0;
  return LBM_OK;
}

int lbm_get(lbm_ctx* ctx, double* rho, double* phi, double* ux, double* uy, double* p) {
  if (!ctx) return fail(ctx, LBM_EINVAL, "null context");
  const size_t n = ctx->n;
  double* h[5] = {rho, phi, ux, uy, p};
  int bx;
  const dim3 grid = row_grid(ctx->P.nx, ctx->P.ny, &bx);
  // the moments kernel writes the fields it is given; the staging area holds kStagePlanes of them at a time
  int f = 0;
  while (f < 5) {
    double* d[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    int used = 0, f1 = f;
    for (; f1 < 5 && used < (int)kStagePlanes; f1++)
      if (h[f1]) d[f1] = ctx->stage + (size_t)(used++) * n;
    if (used) {
      if (ctx->is32)
        k_moments<float><<<grid, bx, 0, ctx->st>>>(ctx->Cf, ctx->cls, ctx->links, pop_view<float>(ctx),
                                                   (const float*)ctx->phi[ctx->pcur], d[0], d[1], d[2], d[3], d[4]);
      else
        k_moments<double><<<grid, bx, 0, ctx->st>>>(ctx->Cd, ctx->cls, ctx->links, pop_view<double>(ctx),
                                                    (const double*)ctx->phi[ctx->pcur], d[0], d[1], d[2], d[3], d[4]);
      ctx->launches[3]++;
      CK(cudaGetLastError());
      for (int k = f; k < f1; k++)
        if (d[k]) CK(cudaMemcpyAsync(h[k], d[k], n * sizeof(double), cudaMemcpyDeviceToHost, ctx->st));
      CK(cudaStreamSynchronize(ctx->st));
    }
    f = f1;
  }
  return LBM_OK;
}

int lbm_get_populations(lbm_ctx* ctx, double* N, double* B) {
  if (!ctx) return fail(ctx, LBM_EINVAL, "null context");
  if (B && !ctx->B_valid)
    return fail(ctx, LBM_EINVAL, "B is not stored under this schedule: call lbm_keep_B(ctx, 1) before lbm_step");
  const size_t n = ctx->n;
  int bx;
  const dim3 grid = row_grid(ctx->P.nx, ctx->P.ny, &bx);
  const double chi[9] = {ctx->Cd.chi0, ctx->Cd.chi1, ctx->Cd.chi1, ctx->Cd.chi1, ctx->Cd.chi1,
                         ctx->Cd.chi5, ctx->Cd.chi5, ctx->Cd.chi5, ctx->Cd.chi5};
  for (int which = 0; which < 2; which++) {
    double* host = which ? B : N;
    if (!host) continue;
    const int CH = (int)kStagePlanes;             // staging planes at a time
    for (int q0 = 0; q0 < 9; q0 += CH) {
      const int q1 = q0 + CH < 9 ? q0 + CH : 9;
      for (int q = q0; q < q1; q++) {
        double* dst = ctx->stage + (size_t)(q - q0) * n;
        const double add = which ? 0.0 : chi[q];
        if (ctx->is32)
          k_gather_plane<float><<<grid, bx, 0, ctx->st>>>(ctx->Cf, ctx->cls, ctx->links, which ? B_view<float>(ctx) : pop_view<float>(ctx), q, add, dst);
        else
          k_gather_plane<double><<<grid, bx, 0, ctx->st>>>(ctx->Cd, ctx->cls, ctx->links, which ? B_view<double>(ctx) : pop_view<double>(ctx), q, add, dst);
        ctx->launches[3]++;
      }
      CK(cudaGetLastError());
      CK(cudaMemcpyAsync(host + (size_t)q0 * n, ctx->stage, (size_t)(q1 - q0) * n * sizeof(double),
                         cudaMemcpyDeviceToHost, ctx->st));
      CK(cudaStreamSynchronize(ctx->st));
    }
  }
  return LBM_OK;
}

int lbm_rows_bytes(lbm_ctx* ctx, int32_t j0, int32_t nrows, size_t* bytes) {
  if (!ctx || !bytes) return fail(ctx, LBM_EINVAL, "null argument");
  RowPiece pc[19];
  int n = 0;
  const int rc = row_pieces(ctx, j0, nrows, pc, &n);
  if (rc != LBM_OK) return rc;
  size_t b = 0;
  for (int i = 0; i < n; i++) b += pc[i].bytes;
  *bytes = b;
  return LBM_OK;
}

int lbm_rows_export(lbm_ctx* ctx, int32_t j0, int32_t nrows, void* d_buf, size_t cap) {
  if (!ctx || !d_buf) return fail(ctx, LBM_EINVAL, "null argument");
  RowPiece pc[19];
  int n = 0;
  const int rc = row_pieces(ctx, j0, nrows, pc, &n);
  if (rc != LBM_OK) return rc;
  size_t need = 0;
  for (int i = 0; i < n; i++) need += pc[i].bytes;
  if (need > cap) return fail(ctx, LBM_ENOMEM, "row buffer too small (lbm_rows_bytes)");
  return rows_copy<true>(ctx, pc, n, (char*)d_buf);
}

int lbm_rows_import(lbm_ctx* ctx, int32_t j0, int32_t nrows, const void* d_buf, size_t bytes) {
  if (!ctx || !d_buf) return fail(ctx, LBM_EINVAL, "null argument");
  RowPiece pc[19];
  int n = 0;
  const int rc = row_pieces(ctx, j0, nrows, pc, &n);
  if (rc != LBM_OK) return rc;
  size_t need = 0;
  for (int i = 0; i < n; i++) need += pc[i].bytes;
  if (bytes != need) return fail(ctx, LBM_EINVAL, "row buffer size differs from lbm_rows_bytes: the two contexts do not agree on these rows");
  const int rc2 = rows_copy<false>(ctx, pc, n, (char*)const_cast<void*>(d_buf));
  if (rc2 != LBM_OK) return rc2;
  if (ctx->fused) ctx->B_valid = 0;   // B planes kept by lbm_keep_B no longer belong to this state
  return LBM_OK;
}

int lbm_set_populations(lbm_ctx* ctx, const double* N, const double* B) {
  if (!ctx) return fail(ctx, LBM_EINVAL, "null context");
  if (!N && !B) return LBM_OK;
  const size_t n = ctx->n;
  int bx;
  const dim3 grid = row_grid(ctx->P.nx, ctx->P.ny, &bx);
  if (ctx->inplace && ctx->aa_local) {
    // k_scatter_plane writes the standard parking: bring what is NOT overwritten there first.  A direction and its
    // opposite only ever use each other's planes, so pair by pair: gather both (as the readers see them), scatter both.
    for (int which = 0; which < 2; which++) {
      if (which ? B != nullptr : N != nullptr) continue;
      const int pairs[4][2] = {{1, 3}, {2, 4}, {5, 7}, {6, 8}};
      for (const auto& pr : pairs) {
        for (int t = 0; t < 2; t++) {
          double* dst = ctx->stage + (size_t)t * n;
          if (ctx->is32) k_gather_plane<float><<<grid, bx, 0, ctx->st>>>(ctx->Cf, ctx->cls, ctx->links, which ? B_view<float>(ctx) : pop_view<float>(ctx), pr[t], 0.0, dst);
          else k_gather_plane<double><<<grid, bx, 0, ctx->st>>>(ctx->Cd, ctx->cls, ctx->links, which ? B_view<double>(ctx) : pop_view<double>(ctx), pr[t], 0.0, dst);
        }
        for (int t = 0; t < 2; t++) {
          const double* src = ctx->stage + (size_t)t * n;
          if (ctx->is32) k_scatter_plane<float><<<grid, bx, 0, ctx->st>>>(ctx->Cf, ctx->cls, ctx->links, src, pr[t], 0.0, which ? B_view<float>(ctx) : pop_view<float>(ctx));
          else k_scatter_plane<double><<<grid, bx, 0, ctx->st>>>(ctx->Cd, ctx->cls, ctx->links, src, pr[t], 0.0, which ? B_view<double>(ctx) : pop_view<double>(ctx));
        }
        ctx->launches[3] += 4;
      }
      CK(cudaGetLastError());
    }
    CK(cudaStreamSynchronize(ctx->st));
    set_parking(ctx, false);
  }
  const double chi[9] = {ctx->Cd.chi0, ctx->Cd.chi1, ctx->Cd.chi1, ctx->Cd.chi1, ctx->Cd.chi1,
                         ctx->Cd.chi5, ctx->Cd.chi5, ctx->Cd.chi5, ctx->Cd.chi5};
  void* Bp = ctx->fused ? ctx->B[0] : ctx->B[ctx->cur];   // may be absent (compacted layout without lbm_keep_B)
  const int CH = (int)kStagePlanes - 1;                    // planes 0 .. CH-1 stage the input, the last one accumulates phi
  double* acc = ctx->stage + (size_t)CH * n;
  for (int which = 0; which < 2; which++) {
    const double* host = which ? B : N;
    if (!host) continue;
    const bool scatter = which ? Bp != nullptr : true;
    for (int q0 = 0; q0 < 9; q0 += CH) {
      const int q1 = q0 + CH < 9 ? q0 + CH : 9;
      CK(cudaMemcpyAsync(ctx->stage, host + (size_t)q0 * n, (size_t)(q1 - q0) * n * sizeof(double), cudaMemcpyHostToDevice, ctx->st));
      for (int q = q0; q < q1; q++) {
        const double* src = ctx->stage + (size_t)(q - q0) * n;
        const double sub = which ? 0.0 : chi[q];
        if (ctx->is32) {
          if (scatter) k_scatter_plane<float><<<grid, bx, 0, ctx->st>>>(ctx->Cf, ctx->cls, ctx->links, src, q, sub, which ? B_view<float>(ctx) : pop_view<float>(ctx));
          if (which) k_phi_accumulate<float><<<grid, bx, 0, ctx->st>>>(ctx->Cf, ctx->cls, src, q == 0, acc, q == 8 ? (float*)ctx->phi[ctx->pcur] : nullptr);
        } else {
          if (scatter) k_scatter_plane<double><<<grid, bx, 0, ctx->st>>>(ctx->Cd, ctx->cls, ctx->links, src, q, sub, which ? B_view<double>(ctx) : pop_view<double>(ctx));
          if (which) k_phi_accumulate<double><<<grid, bx, 0, ctx->st>>>(ctx->Cd, ctx->cls, src, q == 0, acc, q == 8 ? (double*)ctx->phi[ctx->pcur] : nullptr);
        }
        ctx->launches[3] += which ? 2 : 1;
      }
      CK(cudaGetLastError());
      CK(cudaStreamSynchronize(ctx->st));   // the staging planes are reused by the next chunk
    }
  }
  if (B) {
    ctx->B_valid = Bp ? 1 : 0;
    if (ctx->is32) launch_ghost<float>(ctx); else launch_ghost<double>(ctx);   // ghost values follow the new phi (Eq. 9)
  }
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(ctx->st));
  return LBM_OK;
}

int lbm_sample_populations(lbm_ctx* ctx, int64_t n_idx, const int64_t* idx, double* N, double* B) {
  if (!ctx || n_idx < 0 || (n_idx > 0 && !idx)) return fail(ctx, LBM_EINVAL, "bad argument");
  if (B && !ctx->B_valid)
    return fail(ctx, LBM_EINVAL, "B is not stored under this schedule: call lbm_keep_B(ctx, 1) before lbm_step");
  for (int64_t t = 0; t < n_idx; t++)
    if (idx[t] < 0 || (size_t)idx[t] >= ctx->n) return fail(ctx, LBM_EINVAL, "sample index out of range");
  // chunks sized by the index buffer and by the staging area (9 doubles per sample)
  const int64_t chunk = (int64_t)std::min<size_t>(ctx->samp_cap, std::max<size_t>(1, kStagePlanes * ctx->n / 9));
  for (int64_t t0 = 0; t0 < n_idx; t0 += chunk) {
    const int64_t m = std::min<int64_t>(chunk, n_idx - t0);
    CK(cudaMemcpyAsync(ctx->samp_idx, idx + t0, (size_t)m * sizeof(long long), cudaMemcpyHostToDevice, ctx->st));
    const unsigned gb = (unsigned)((m + 127) / 128);
    for (int which = 0; which < 2; which++) {
      double* host = which ? B : N;
      if (!host) continue;
      if (ctx->is32)
        k_gather_samples<float><<<gb, 128, 0, ctx->st>>>(ctx->Cf, ctx->cls, ctx->links, which ? B_view<float>(ctx) : pop_view<float>(ctx),
                                                         which ? 0 : 1, (long long)m, ctx->samp_idx, ctx->stage);
      else
        k_gather_samples<double><<<gb, 128, 0, ctx->st>>>(ctx->Cd, ctx->cls, ctx->links, which ? B_view<double>(ctx) : pop_view<double>(ctx),
                                                          which ? 0 : 1, (long long)m, ctx->samp_idx, ctx->stage);
      ctx->launches[3]++;
      CK(cudaGetLastError());
      // device [q][m] -> host [q][n_idx] at column t0
      CK(cudaMemcpy2DAsync(host + t0, (size_t)n_idx * sizeof(double), ctx->stage, (size_t)m * sizeof(double),
                           (size_t)m * sizeof(double), 9, cudaMemcpyDeviceToHost, ctx->st));
      CK(cudaStreamSynchronize(ctx->st));
    }
  }
  return LBM_OK;
}

int lbm_get_classification(lbm_ctx* ctx, uint8_t* cls, int32_t* n_ghost, int32_t* ghost_idx,
                           double* ghost_nx, double* ghost_ny, double* ghost_depth,
                           int32_t* ghost_corner, double* ghost_wgt) {
  if (!ctx) return fail(ctx, LBM_EINVAL, "null context");
  const size_t g = (size_t)ctx->ng;
  if (n_ghost) *n_ghost = ctx->ng;
  if (cls) CK(cudaMemcpyAsync(cls, ctx->cls, ctx->n, cudaMemcpyDeviceToHost, ctx->st));
  if (g > 0) {
    if (ghost_idx) CK(cudaMemcpyAsync(ghost_idx, ctx->gidx, g * sizeof(int), cudaMemcpyDeviceToHost, ctx->st));
    if (ghost_nx) CK(cudaMemcpyAsync(ghost_nx, ctx->gnx, g * sizeof(double), cudaMemcpyDeviceToHost, ctx->st));
    if (ghost_ny) CK(cudaMemcpyAsync(ghost_ny, ctx->gny, g * sizeof(double), cudaMemcpyDeviceToHost, ctx->st));
    if (ghost_depth) CK(cudaMemcpyAsync(ghost_depth, ctx->gdepth, g * sizeof(double), cudaMemcpyDeviceToHost, ctx->st));
    if (ghost_corner) CK(cudaMemcpyAsync(ghost_corner, ctx->corner, 4 * g * sizeof(int), cudaMemcpyDeviceToHost, ctx->st));
    if (ghost_wgt) CK(cudaMemcpyAsync(ghost_wgt, ctx->wgt_d, 4 * g * sizeof(double), cudaMemcpyDeviceToHost, ctx->st));
  }
  CK(cudaStreamSynchronize(ctx->st));
  return LBM_OK;
}

int lbm_diag(lbm_ctx* ctx, double out[8]) {
  if (!ctx || !out) return fail(ctx, LBM_EINVAL, "null argument");
  int bx;
  const dim3 grid = row_grid(ctx->P.nx, ctx->P.ny, &bx);
  const long long m = (long long)grid.x * grid.y;
  if ((size_t)m * sizeof(DiagVec) > (kStagePlanes * ctx->n + 64) * sizeof(double)) return fail(ctx, LBM_EINVAL, "grid too small for diag staging");
  DiagVec* part = reinterpret_cast<DiagVec*>(ctx->stage);
  if (ctx->is32)
    k_diag_partial<float><<<grid, bx, 0, ctx->st>>>(ctx->Cf, ctx->cls, ctx->links, pop_view<float>(ctx),
                                                    (const float*)ctx->phi[ctx->pcur], part);
  else
    k_diag_partial<double><<<grid, bx, 0, ctx->st>>>(ctx->Cd, ctx->cls, ctx->links, pop_view<double>(ctx),
                                                     (const double*)ctx->phi[ctx->pcur], part);
  k_diag_final<<<1, 1024, 0, ctx->st>>>(part, m, ctx->diag_out);
  ctx->launches[3] += 2;
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(out, ctx->diag_out, 8 * sizeof(double), cudaMemcpyDeviceToHost, ctx->st));
  CK(cudaStreamSynchronize(ctx->st));
  return LBM_OK;
}

int lbm_diag_static(lbm_ctx* ctx, double* d_out) {
  if (!ctx || !d_out) return fail(ctx, LBM_EINVAL, "null argument");
  if (!ctx->diag_static) {
    char buf[300];
    snprintf(buf, sizeof buf, "lbm_diag_static: cudaGetSymbolAddress of the static scratch failed at lbm_create: %s",
             cudaGetErrorString((cudaError_t)ctx->diag_static_err));
    return fail(ctx, LBM_ECUDA, buf);
  }
  int bx;
  const dim3 grid = row_grid(ctx->P.nx, ctx->P.ny, &bx);
  const long long m = (long long)grid.x * grid.y;
  if (m > kDiagStaticMax) {
    char buf[300];
    snprintf(buf, sizeof buf, "lbm_diag_static: this grid needs %lld block partials, the static scratch holds %lld "
             "(ceil(nx / 256) * ny must not exceed it); use lbm_diag", m, kDiagStaticMax);
    return fail(ctx, LBM_EINVAL, buf);
  }
  // every one of the m slots is written by its block before k_diag_final reads slots 0 .. m-1: whatever an earlier
  // call left in the array is never read, nothing has to be cleared
  DiagVec* part = ctx->diag_static;
  if (ctx->is32)
    k_diag_partial<float><<<grid, bx, 0, ctx->st>>>(ctx->Cf, ctx->cls, ctx->links, pop_view<float>(ctx),
                                                    (const float*)ctx->phi[ctx->pcur], part);
  else
    k_diag_partial<double><<<grid, bx, 0, ctx->st>>>(ctx->Cd, ctx->cls, ctx->links, pop_view<double>(ctx),
                                                     (const double*)ctx->phi[ctx->pcur], part);
  k_diag_final<<<1, 1024, 0, ctx->st>>>(part, m, d_out);
  ctx->launches[3] += 2;
  CK(cudaGetLastError());
  return LBM_OK;
}

int lbm_layout_copy_timed(lbm_ctx* ctx, int32_t iters, double* ms_per_pass) {
  if (!ctx || iters < 1 || !ms_per_pass) return fail(ctx, LBM_EINVAL, "bad argument");
  if (ctx->packed) return fail(ctx, LBM_EINVAL, "the dense SoA layout this helper measures is not kept under PACK / SPARSE; create the context with LBM_SCHEDULE_PAIR");
  if (ctx->inplace) return fail(ctx, LBM_EINVAL, "an INPLACE context has no second buffer to copy into; create the context with LBM_SCHEDULE_PAIR");
  const size_t rs = ctx->is32 ? 4 : 8, nps = 32 / rs;
  if (ctx->n % nps != 0 || ctx->Cd.ps % nps != 0) return fail(ctx, LBM_EINVAL, "nx*ny is not a whole number of 32-byte sectors");
  const size_t nsec = ctx->n / nps, psec = ctx->Cd.ps / nps;
  const float4* src = (const float4*)ctx->N[ctx->cur];
  float4* dst = (float4*)ctx->N[ctx->cur ^ 1];          // scratch: the next step overwrites it
  const float4* psrc = (const float4*)ctx->phi[ctx->pcur];
  float4* pdst = (float4*)ctx->stage;                    // scratch (phi[pcur ^ 1] holds the previous ghost values)
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0));
  CK(cudaEventCreate(&e1));
  const int blocks = 148 * 32;
  for (int it = 0; it < iters + 2; it++) {
    if (it == 2) cudaEventRecord(e0, ctx->st);
    if (ctx->is32) k_copy_sectors<8><<<blocks, 256, 0, ctx->st>>>(ctx->cl16, src, dst, psrc, pdst, nsec, psec);
    else k_copy_sectors<4><<<blocks, 256, 0, ctx->st>>>(ctx->cl16, src, dst, psrc, pdst, nsec, psec);
    ctx->launches[3]++;
  }
  cudaEventRecord(e1, ctx->st);
  CK(cudaEventSynchronize(e1));
  float ms = 0.f;
  CK(cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  CK(cudaGetLastError());
  *ms_per_pass = (double)ms / iters;
  return LBM_OK;
}

int lbm_launch_counts(lbm_ctx* ctx, int64_t counts[4], int32_t reset) {
  if (!ctx) return fail(ctx, LBM_EINVAL, "null context");
  if (counts) for (int k = 0; k < 4; k++) counts[k] = ctx->launches[k];
  if (reset) for (int k = 0; k < 4; k++) ctx->launches[k] = 0;
  return LBM_OK;
}

int lbm_node_update_batch(const lbm_params* prm, int64_t count, const double* N, const double* phi_nb,
                          double* Nstar, double* Bstar, double* fields) {
  lbm_ctx* ctx = nullptr;
  const char* why;
  if (validate(prm, &why) != LBM_OK) return fail(nullptr, LBM_EINVAL, why);
  if (count < 0 || !N || !phi_nb) return fail(nullptr, LBM_EINVAL, "bad argument");
  if (count == 0) return LBM_OK;
  const size_t c9 = (size_t)count * 9 * sizeof(double), c8 = (size_t)count * 8 * sizeof(double);
  double* d = nullptr;
  CK(cudaMalloc(&d, 4 * c9 + c8));
  double *dN = d, *dP = d + 9 * count, *dNs = d + 18 * count, *dBs = d + 27 * count, *dF = d + 36 * count;
  cudaError_t e = cudaMemcpy(dN, N, c9, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(dP, phi_nb, c9, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    const unsigned gb = (unsigned)((count + 127) / 128);
    if (prm->precision == 32)
      k_node_batch<float><<<gb, 128>>>(make_consts<float>(*prm), (long long)count, dN, dP, dNs, dBs, dF);
    else
      k_node_batch<double><<<gb, 128>>>(make_consts<double>(*prm), (long long)count, dN, dP, dNs, dBs, dF);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess && Nstar) e = cudaMemcpy(Nstar, dNs, c9, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess && Bstar) e = cudaMemcpy(Bstar, dBs, c9, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess && fields) e = cudaMemcpy(fields, dF, c8, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  cudaFree(d);
  if (e != cudaSuccess) return cuda_fail(nullptr, e, "lbm_node_update_batch");
  return LBM_OK;
}

}  // extern "C"

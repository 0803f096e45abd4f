// lbm_kernels.cuh — CUDA kernels of liblbm_b200 (sm_100a).  See DESIGN.md "Kernels".
//
// State layout in HBM (structure of arrays, x fastest, idx = j*nx + i):
//   pop[q*ps + idx] (ps = padded plane stride, Consts::ps) post-COLLISION deviations n_q* = N_q* - chi_q of the last step, stored at the
//                   node that produced them; propagation (A16-A17) is the pull on the next read:
//                   N_q(x, t+1) = N_q*(x - c_q, t), or N_opp(q)*(x, t) if x - c_q is solid
//                   (half-way bounce-back, R12).  Double-buffered.
//   phi[2][idx]     order parameter incl. ghost values, double-buffered so that the ghost update
//                   is a Jacobi sweep (R13) and tiles may read halos while others write.
//   cls[idx]        node class (1 byte); links[idx] bounce-back link bits, read only on
//                   fluid-boundary nodes (bit q-1 set <=> node x - c_q is solid).
#pragma once
#include <stdint.h>
#include "lbm_math.cuh"

namespace lbm {

// opposite direction of Eq. A5's ordering: 1<->3, 2<->4, 5<->7, 6<->8
__host__ __device__ constexpr int opp(int q) {
  return q == 0 ? 0 : (q < 5 ? ((q + 1) % 4) + 1 : ((q - 3) % 4) + 5);
}

// Periodic neighbourhood of node (i, j): linear indices of x - c_q (pull sources) and x + c_q.
struct Nbr {
  int src[9];  // idx of x - c_q
  int dst[9];  // idx of x + c_q
};

__device__ __forceinline__ Nbr make_nbr(int i, int j, int nx, int ny) {
  const int im = (i == 0) ? nx - 1 : i - 1, ip = (i == nx - 1) ? 0 : i + 1;
  const int jm = (j == 0) ? ny - 1 : j - 1, jp = (j == ny - 1) ? 0 : j + 1;
  const int rm = jm * nx, r0 = j * nx, rp = jp * nx;
  Nbr b;
  b.src[0] = r0 + i;  b.dst[0] = r0 + i;
  b.src[1] = r0 + im; b.dst[1] = r0 + ip;
  b.src[2] = rm + i;  b.dst[2] = rp + i;
  b.src[3] = r0 + ip; b.dst[3] = r0 + im;
  b.src[4] = rp + i;  b.dst[4] = rm + i;
  b.src[5] = rm + im; b.dst[5] = rp + ip;
  b.src[6] = rm + ip; b.dst[6] = rp + im;
  b.src[7] = rp + ip; b.dst[7] = rm + im;
  b.src[8] = rp + im; b.dst[8] = rm + ip;
  return b;
}

// ------------------------------------------------------------------------------------------
// (1) classification (one-time).  PAPER.md:21: fluid (solid) boundary node = has >= 1 solid
// (fluid) neighbour in the D2Q9 stencil; periodic wrap.  Integer logic only => bit-exact.
// cls == nullptr: count ghosts only (lbm_plan).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_classify(const uint8_t* __restrict__ mask, int nx, int ny,
                                                  uint8_t* __restrict__ cls,
                                                  uint8_t* __restrict__ links,
                                                  int* __restrict__ block_count,
                                                  unsigned long long* __restrict__ total) {
  const long long n = (long long)nx * ny;
  const long long k = (long long)blockIdx.x * 256 + threadIdx.x;
  int is_ghost = 0;
  if (k < n) {
    const int i = (int)(k % nx), j = (int)(k / nx);
    const Nbr b = make_nbr(i, j, nx, ny);
    const int solid = mask[k] != 0;
    unsigned lk = 0;
    int other = 0;
#pragma unroll
    for (int q = 1; q < 9; q++) {
      const int s = mask[b.src[q]] != 0;
      lk |= (unsigned)s << (q - 1);
      other |= (s != solid);
    }
    const uint8_t c = solid ? (other ? 2 : 3) : (other ? 1 : 0);
    is_ghost = (c == 2);
    if (cls) {
      cls[k] = c;
      links[k] = solid ? 0 : (uint8_t)lk;
    }
  }
  const int cnt = __syncthreads_count(is_ghost);
  if (threadIdx.x == 0) {
    if (block_count) block_count[blockIdx.x] = cnt;
    if (total && cnt) atomicAdd(total, (unsigned long long)cnt);
  }
}

// exclusive scan of the per-block ghost counts (single block; one-time)
__global__ void __launch_bounds__(1024) k_scan_blocks(const int* __restrict__ cnt, int nb,
                                                      int* __restrict__ off, int* __restrict__ total) {
  __shared__ int wsum[32];
  __shared__ int carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int base = 0; base < nb; base += 1024) {
    const int t = base + threadIdx.x;
    const int v = t < nb ? cnt[t] : 0;
    int x = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int y = __shfl_up_sync(0xffffffffu, x, d);
      if (lane >= d) x += y;
    }
    if (lane == 31) wsum[w] = x;
    __syncthreads();
    if (w == 0) {
      int s = wsum[lane];
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, s, d);
        if (lane >= d) s += y;
      }
      wsum[lane] = s;  // inclusive over warps
    }
    __syncthreads();
    const int wo = w ? wsum[w - 1] : 0;
    if (t < nb) off[t] = carry + wo + x - v;
    __syncthreads();
    if (threadIdx.x == 1023) carry += wo + x;
    __syncthreads();
  }
  if (threadIdx.x == 0) *total = carry;
}

// class byte and link byte of every node as one 16-bit word (WARP schedule)
__global__ void __launch_bounds__(256) k_pack_cl16(const uint8_t* __restrict__ cls,
                                                   const uint8_t* __restrict__ links, long long n,
                                                   uint16_t* __restrict__ cl16) {
  const long long k = (long long)blockIdx.x * 256 + threadIdx.x;
  if (k < n) cl16[k] = (uint16_t)(cls[k] | ((cls[k] == 1 ? links[k] : 0u) << 8));
}

// index-sorted compaction of ghost nodes
__global__ void __launch_bounds__(256) k_compact_ghosts(const uint8_t* __restrict__ cls, long long n,
                                                        const int* __restrict__ block_off,
                                                        int* __restrict__ gidx) {
  __shared__ int wcnt[8];
  const long long k = (long long)blockIdx.x * 256 + threadIdx.x;
  const int flag = (k < n) && (cls[k] == 2);
  const unsigned bal = __ballot_sync(0xffffffffu, flag);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) wcnt[w] = __popc(bal);
  __syncthreads();
  int wo = 0;
  for (int v = 0; v < w; v++) wo += wcnt[v];
  if (flag) gidx[block_off[blockIdx.x] + wo + __popc(bal & ((1u << lane) - 1u))] = (int)k;
}

// Per-ghost geometry (one-time): analytic unit normal of the owning disk / wall row (:100, :60),
// depth, x_F = x_G + n_s (:66) and its bilinear stencil.  All in fp64 WITHOUT fma contraction so
// that the list can be compared bit for bit.
struct Disk { double cx, cy, r; };

// one smoothing pass of the solid indicator for the mask-only normals (NEXT row f2): centre weight
// 60 and the sixth-order isotropic weights 32, 12, 1 (x120) at |c|^2 = 1, 2, 4; integers, periodic.
// from_cls: the input is the class array (solid <=> class >= 2) instead of an int field.
__global__ void __launch_bounds__(256) k_mask_smooth(const uint8_t* __restrict__ cls, const int* __restrict__ in,
                                                     int* __restrict__ out, int nx, int ny) {
  const long long k = (long long)blockIdx.x * 256 + threadIdx.x;
  if (k >= (long long)nx * ny) return;
  const int i = (int)(k % nx), j = (int)(k / nx);
  const int ox[12] = {1, 0, -1, 0, 1, -1, -1, 1, 2, 0, -2, 0};
  const int oy[12] = {0, 1, 0, -1, 1, 1, -1, -1, 0, 2, 0, -2};
  const int wg[12] = {32, 32, 32, 32, 12, 12, 12, 12, 1, 1, 1, 1};
  auto val = [&](int ii, int jj) -> int {
    const long long q = (long long)jj * nx + ii;
    return cls ? (cls[q] >= 2 ? 1 : 0) : in[q];
  };
  int acc = 60 * val(i, j);
#pragma unroll
  for (int t = 0; t < 12; t++) {
    int ii = i + ox[t], jj = j + oy[t];
    ii = ii < 0 ? ii + nx : (ii >= nx ? ii - nx : ii);
    jj = jj < 0 ? jj + ny : (jj >= ny ? jj - ny : jj);
    acc += wg[t] * val(ii, jj);
  }
  out[k] = acc;
}

__device__ __forceinline__ double minimg_d(double d, double L) {
  d = fmod(d, L);
  if (d >= 0.5 * L) d = __dsub_rn(d, L);
  if (d < -0.5 * L) d = __dadd_rn(d, L);
  return d;
}
__device__ __forceinline__ int wrapi_d(int a, int n) {
  a %= n;
  return a < 0 ? a + n : a;
}

template <typename R>
__global__ void __launch_bounds__(128) k_ghost_geometry(int ng, const int* __restrict__ gidx, int nx,
                                                        int ny, int wall_rows,
                                                        const Disk* __restrict__ disks, int n_disks,
                                                        const int* __restrict__ cell_start,
                                                        const int* __restrict__ cell_disks, int ncx, int cell_size,
                                                        const int* __restrict__ smooth2,
                                                        const uint8_t* __restrict__ cls,
                                                        double* __restrict__ gnx, double* __restrict__ gny,
                                                        double* __restrict__ gdepth,
                                                        int* __restrict__ corner, double* __restrict__ wgt_d,
                                                        R* __restrict__ wgt, uint8_t* __restrict__ csolid,
                                                        double2* __restrict__ gfrac, int* __restrict__ err) {
  const int g = blockIdx.x * 128 + threadIdx.x;
  if (g >= ng) return;
  const int k = gidx[g];
  const int i = k % nx, j = k / nx;
  double nxs = 0.0, nys = 0.0, depth = 0.0;
  int found = 0;
  if (wall_rows && (j == 0 || j == ny - 1)) {
    nys = (j == 0) ? 1.0 : -1.0;
    depth = 0.5;  // half-way wall (R17)
    found = 1;
  } else {
    // candidates: the disks whose bounding box overlaps this node's cell, in increasing disk index
    // (so that "least depth, first wins ties" (R17) is the same as a scan over all disks)
    double best = 0.0;
    const int cell = (j / cell_size) * ncx + (i / cell_size);
    for (int t = cell_start[cell]; t < cell_start[cell + 1]; t++) {
      const Disk dk = disks[cell_disks[t]];
      const double dx = minimg_d(__dsub_rn((double)i, dk.cx), (double)nx);
      const double dy = minimg_d(__dsub_rn((double)j, dk.cy), (double)ny);
      const double r2 = __dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy));
      if (r2 <= __dmul_rn(dk.r, dk.r)) {
        const double dist = __dsqrt_rn(r2);
        const double dep = __dsub_rn(dk.r, dist);
        if (!found || dep < best) {
          best = dep;
          found = 1;
          depth = dep;
          if (dist > 0.0) { nxs = __ddiv_rn(dx, dist); nys = __ddiv_rn(dy, dist); }
          else { nxs = 0.0; nys = 0.0; }
        }
      }
    }
  }
  if (!found && n_disks == 0 && smooth2 != nullptr) {
    // NEXT row f2: no analytic shape was given.  Normal from the mask alone: minus the
    // sixth-order isotropic gradient (12 points, weights x120 = 32, 12, 1: exact integer sums) of the
    // solid indicator smoothed twice (k_mask_smooth); (0,0) where it vanishes.
    const int ox[12] = {1, 0, -1, 0, 1, -1, -1, 1, 2, 0, -2, 0};
    const int oy[12] = {0, 1, 0, -1, 1, 1, -1, -1, 0, 2, 0, -2};
    const int wg[12] = {32, 32, 32, 32, 12, 12, 12, 12, 1, 1, 1, 1};
    long long gxs = 0, gys = 0;
#pragma unroll
    for (int t = 0; t < 12; t++) {
      const int ii = wrapi_d(i + ox[t], nx), jj = wrapi_d(j + oy[t], ny);
      const long long v = smooth2[jj * nx + ii];
      gxs += (long long)(wg[t] * ox[t]) * v;
      gys += (long long)(wg[t] * oy[t]) * v;
    }
    const double ax = -(double)gxs, ay = -(double)gys;
    const double m = __dsqrt_rn(__dadd_rn(__dmul_rn(ax, ax), __dmul_rn(ay, ay)));
    if (m > 0.0) { nxs = __ddiv_rn(ax, m); nys = __ddiv_rn(ay, m); }
    depth = 0.0;
    found = 1;
  }
  if (!found) atomicExch(err, 1);
  gnx[g] = nxs; gny[g] = nys; gdepth[g] = depth;
  const double xF = __dadd_rn((double)i, nxs), yF = __dadd_rn((double)j, nys);
  const double fi = floor(xF), fj = floor(yF);
  const double fx = __dsub_rn(xF, fi), fy = __dsub_rn(yF, fj);
  const int i0 = wrapi_d((int)fi, nx), j0 = wrapi_d((int)fj, ny);
  const int i1 = wrapi_d(i0 + 1, nx), j1 = wrapi_d(j0 + 1, ny);
  const int c0 = j0 * nx + i0, c1 = j0 * nx + i1, c2 = j1 * nx + i0, c3 = j1 * nx + i1;
  const double w0 = __dmul_rn(__dsub_rn(1.0, fx), __dsub_rn(1.0, fy));
  const double w1 = __dmul_rn(fx, __dsub_rn(1.0, fy));
  const double w2 = __dmul_rn(__dsub_rn(1.0, fx), fy);
  const double w3 = __dmul_rn(fx, fy);
  if (gfrac) gfrac[g] = make_double2(fx, fy);
  corner[4 * g + 0] = c0; corner[4 * g + 1] = c1; corner[4 * g + 2] = c2; corner[4 * g + 3] = c3;
  wgt_d[4 * g + 0] = w0; wgt_d[4 * g + 1] = w1; wgt_d[4 * g + 2] = w2; wgt_d[4 * g + 3] = w3;
  wgt[4 * g + 0] = (R)w0; wgt[4 * g + 1] = (R)w1; wgt[4 * g + 2] = (R)w2; wgt[4 * g + 3] = (R)w3;
  csolid[g] = (uint8_t)((cls[c0] >= 2) | ((cls[c1] >= 2) << 1) | ((cls[c2] >= 2) << 2) | ((cls[c3] >= 2) << 3));
}

// Processing order of the ghost update: tile-major (32 x 32 node tiles, index order inside a tile),
// so that the ghosts of one CTA gather phi from the same few sectors (L1 hits instead of DRAM
// re-fetches; the index-sorted list, the API's order, strides over the whole row between
// neighbours).  The update is a Jacobi sweep (R13): the order does not change any value.
__global__ void __launch_bounds__(256) k_ghost_tile_keys(int ng, const int* __restrict__ gidx, int nx,
                                                         unsigned* __restrict__ keys, int* __restrict__ vals) {
  const int g = blockIdx.x * 256 + threadIdx.x;
  if (g >= ng) return;
  const int k = gidx[g];
  const int i = k % nx, j = k / nx;
  keys[g] = (unsigned)(j >> 5) * (unsigned)((nx + 31) >> 5) + (unsigned)(i >> 5);
  vals[g] = g;
}
// The list entry the per-step kernel reads: {node index, code} + (f_x, f_y).  code bits 0-1 / 2-3: i0 - i + 1 and
// j0 - j + 1 of the interpolation cell's base corner (x_F = x_G + n_s lies within one node of x_G, :66), bits 4-7:
// corner is a solid node.  The four corner indices and weights follow from it; storing them took 53 B (fp64) per
// ghost node, this takes 24 B (16 B in fp32).
template <typename R> struct GhostFrac;
template <> struct GhostFrac<double> { using T = double2; };
template <> struct GhostFrac<float> { using T = float2; };
template <typename R>
__global__ void __launch_bounds__(256) k_ghost_permute(int ng, const int* __restrict__ perm,
                                                       const int* __restrict__ gidx, const int4* __restrict__ corner,
                                                       const double2* __restrict__ gfrac, const uint8_t* __restrict__ csolid,
                                                       int nx, int ny, uint2* __restrict__ gent_p,
                                                       typename GhostFrac<R>::T* __restrict__ gfr_p) {
  const int t = blockIdx.x * 256 + threadIdx.x;
  if (t >= ng) return;
  const int g = perm[t];
  const int k = gidx[g], c0 = corner[g].x;
  int di = c0 % nx - k % nx, dj = c0 / nx - k / nx;   // base corner relative to the node, periodic
  if (di > 1) di -= nx;
  if (di < -1) di += nx;
  if (dj > 1) dj -= ny;
  if (dj < -1) dj += ny;
  gent_p[t] = make_uint2((unsigned)k, (unsigned)(di + 1) | ((unsigned)(dj + 1) << 2) | ((unsigned)csolid[g] << 4));
  const double2 f = gfrac[g];
  typename GhostFrac<R>::T o;
  o.x = (R)f.x; o.y = (R)f.y;
  gfr_p[t] = o;
}

// ------------------------------------------------------------------------------------------
// (2) ghost-node order-parameter update, Eq. 9 (:78-80): phi_F by bilinear interpolation at
// x_F = x_G + n_s (:66); Jacobi (R13): fluid corners carry this time's phi (phi_cur), solid
// corners the previous ghost values (phi_prev; bulk solid nodes are constant in both buffers).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void bilinear_weights(double fx, double fy, double (&w)[4]) {   // as the oracle: no contraction
  const double gx = __dsub_rn(1.0, fx), gy = __dsub_rn(1.0, fy);
  w[0] = __dmul_rn(gx, gy); w[1] = __dmul_rn(fx, gy); w[2] = __dmul_rn(gx, fy); w[3] = __dmul_rn(fx, fy);
}
__device__ __forceinline__ void bilinear_weights(float fx, float fy, float (&w)[4]) {
  const float gx = 1.0f - fx, gy = 1.0f - fy;
  w[0] = gx * gy; w[1] = fx * gy; w[2] = gx * fy; w[3] = fx * fy;
}
template <typename R>
__global__ void __launch_bounds__(128) k_ghost_update(const Consts<R> C, int ng,
                                                      const uint2* __restrict__ gent,
                                                      const typename GhostFrac<R>::T* __restrict__ gfr,
                                                      const R* __restrict__ phi_prev,
                                                      R* __restrict__ phi_cur) {
  const int g = blockIdx.x * 128 + threadIdx.x;
  if (g >= ng) return;
  const uint2 e = gent[g];
  const typename GhostFrac<R>::T f = gfr[g];
  const int nx = C.nx, ny = C.ny;
  const int k = (int)e.x, i = k % nx, j = k / nx;
  int i0 = i + (int)(e.y & 3u) - 1, j0 = j + (int)((e.y >> 2) & 3u) - 1;
  i0 = i0 < 0 ? i0 + nx : (i0 >= nx ? i0 - nx : i0);
  j0 = j0 < 0 ? j0 + ny : (j0 >= ny ? j0 - ny : j0);
  const int i1 = i0 + 1 == nx ? 0 : i0 + 1, j1 = j0 + 1 == ny ? 0 : j0 + 1;
  const int c0 = j0 * nx + i0, c1 = j0 * nx + i1, c2 = j1 * nx + i0, c3 = j1 * nx + i1;
  const unsigned sb = e.y >> 4;
  R w[4];
  bilinear_weights(f.x, f.y, w);
  const R p0 = (sb & 1u) ? phi_prev[c0] : phi_cur[c0];
  const R p1 = (sb & 2u) ? phi_prev[c1] : phi_cur[c1];
  const R p2 = (sb & 4u) ? phi_prev[c2] : phi_cur[c2];
  const R p3 = (sb & 8u) ? phi_prev[c3] : phi_cur[c3];
  const R phiF = ((w[0] * p0 + w[1] * p1) + w[2] * p2) + w[3] * p3;
  phi_cur[k] = ghost_rule<R>(C, phiF);
}

// ------------------------------------------------------------------------------------------
// pulled (post-stream) population q of node k: propagation A16-A17 + half-way bounce-back (R12)
// ------------------------------------------------------------------------------------------
// Where a set of nine population planes lives: dense (pop[q * ps + idx]) or group-compacted (PACK / SPARSE, see
// k_pair_mask below).  The fused kernels address their layout directly; everything off the hot path (lbm_init,
// lbm_get, lbm_diag, lbm_get/set_populations) goes through this view, so that a compacted context needs no dense
// copy of its state.
template <typename R>
struct PopView {
  R* base;
  size_t ps;            // dense: element stride between planes
  const uint2* ptab;    // nullptr: dense
  int nx, nw, G, group_major;
  size_t cps;
  __device__ __forceinline__ bool has(int idx) const {   // storage exists for this node (its group holds a fluid node)
    if (!ptab) return true;
    const int j = idx / nx, p = (idx - j * nx) / G;
    return (ptab[(size_t)j * nw + (p >> 5)].x >> (p & 31)) & 1u;
  }
  __device__ __forceinline__ size_t off(int q, int idx) const {
    if (!ptab) return (size_t)q * ps + (size_t)idx;
    const int j = idx / nx, i = idx - j * nx, p = i / G;
    const uint2 tb = ptab[(size_t)j * nw + (p >> 5)];
    const size_t ci = (size_t)tb.y + (size_t)__popc(tb.x & ((1u << (p & 31)) - 1u));
    return group_major ? (ci * 9 + (size_t)q) * G + (size_t)(i - p * G) : ((size_t)q * cps + ci) * G + (size_t)(i - p * G);
  }
  __device__ __forceinline__ R& at(int q, int idx) const { return base[off(q, idx)]; }
};
template <typename R>
inline PopView<R> dense_view(R* base, size_t ps, int nx) { return PopView<R>{base, ps, nullptr, nx, 0, 1, 0, 0}; }

template <typename R>
__device__ __forceinline__ void pull9(const PopView<R>& P, int k, const Nbr& b, unsigned lk, R (&v)[9]) {
  v[0] = P.at(0, k);
#pragma unroll
  for (int q = 1; q < 9; q++) v[q] = ((lk >> (q - 1)) & 1u) ? P.at(opp(q), k) : P.at(q, b.src[q]);
}

template <typename R>
__device__ __forceinline__ void pull9(const R* __restrict__ pop, size_t n, int k, const Nbr& b,
                                      unsigned lk, R (&v)[9]) {
  v[0] = pop[k];
  if (lk == 0) {
#pragma unroll
    for (int q = 1; q < 9; q++) v[q] = pop[q * n + b.src[q]];
  } else {
#pragma unroll
    for (int q = 1; q < 9; q++)
      v[q] = ((lk >> (q - 1)) & 1u) ? pop[opp(q) * n + k] : pop[q * n + b.src[q]];
  }
}

template <typename R>
__device__ __forceinline__ void load_phi9(const R* __restrict__ phi, const Nbr& b, R (&ph)[9]) {
#pragma unroll
  for (int q = 0; q < 9; q++) ph[q] = phi[b.dst[q]];
}

// link bits of a node as the readers of the state see them (see Consts::all_links)
template <typename R>
__device__ __forceinline__ unsigned link_bits(const Consts<R>& C, unsigned c, const uint8_t* __restrict__ links, int k) {
  if (C.all_links) return 0xffu;
  return (c == 1) ? links[k] : 0u;
}

// ------------------------------------------------------------------------------------------
// BASELINE schedule, kernel (3): fused pull-stream + collide, one thread per node.
// Reads 9 pulled N, the 3x3 phi neighbourhood, 1 class byte; writes 9 N* and 9 B*.
// ------------------------------------------------------------------------------------------
template <typename R>
__global__ void __launch_bounds__(256) k_collide_baseline(const Consts<R> C,
                                                          const uint8_t* __restrict__ cls,
                                                          const uint8_t* __restrict__ links,
                                                          const R* __restrict__ Nsrc, R* __restrict__ Ndst,
                                                          R* __restrict__ Bdst,
                                                          const R* __restrict__ phi) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= C.nx) return;
  const size_t n = C.ps;   // plane stride
  const int k = j * C.nx + i;
  const uint8_t c = cls[k];
  if (c >= 2) return;
  const Nbr b = make_nbr(i, j, C.nx, C.ny);
  const unsigned lk = (c == 1) ? links[k] : 0u;
  R nn[9], ph[9], ns[9], bs[9];
  load_phi9<R>(phi, b, ph);
  pull9<R>(Nsrc, n, k, b, lk, nn);
  node_update<R, true>(C, nn, ph, ns, bs, nullptr);
#pragma unroll
  for (int q = 0; q < 9; q++) {
    Ndst[q * n + k] = ns[q];
    Bdst[q * n + k] = bs[q];
  }
}

// BASELINE schedule: phi(x, t+1) = sum_i B_i(x, t+1) (A13, :311) from the pulled B*.
template <typename R>
__global__ void __launch_bounds__(256) k_phi_sum(const Consts<R> C, const uint8_t* __restrict__ cls,
                                                 const uint8_t* __restrict__ links,
                                                 const R* __restrict__ Bsrc, R* __restrict__ phi) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= C.nx) return;
  const size_t n = C.ps;   // plane stride
  const int k = j * C.nx + i;
  const uint8_t c = cls[k];
  if (c >= 2) return;
  const Nbr b = make_nbr(i, j, C.nx, C.ny);
  const unsigned lk = link_bits(C, c, links, k);
  R v[9];
  pull9<R>(Bsrc, n, k, b, lk, v);
  R s = v[0];
#pragma unroll
  for (int q = 1; q < 9; q++) s += v[q];
  phi[k] = s;
}

// ------------------------------------------------------------------------------------------
// INPLACE schedule (f4: single-buffer streaming, the AA pattern): the canonical state N_i, B_i in ONE buffer each.
// Every thread writes only the slots it read, so no other thread's input is ever overwritten and the launch order
// does not matter.  The stored value is, as everywhere, the post-collision population; where it is parked alternates:
//   even time ("standard"): N_q*(y) in slot q of y; the reader at x pulls slot q of x - c_q (own slot opp(q) on a link);
//   odd time  ("local"):    N_q*(y) in slot opp(q) of y + c_q (in slot q of y itself if y + c_q is solid): the reader
//                           at x finds all nine in its own opposite slots.
// k_collide_aa_nbr takes standard to local, k_collide_aa_local takes local to standard.  The collision never reads
// B_i, so the B planes simply follow the same parking rule (k_phi_sum reads them afterwards).
// ------------------------------------------------------------------------------------------
template <typename R>
__global__ void __launch_bounds__(256) k_collide_aa_nbr(const Consts<R> C, const uint8_t* __restrict__ cls,
                                                        const uint8_t* __restrict__ links, R* __restrict__ N,
                                                        R* __restrict__ B, const R* __restrict__ phi) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= C.nx) return;
  const size_t n = C.ps;
  const int k = j * C.nx + i;
  const uint8_t c = cls[k];
  if (c >= 2) return;
  const Nbr b = make_nbr(i, j, C.nx, C.ny);
  const unsigned lk = (c == 1) ? links[k] : 0u;
  R nn[9], ph[9], ns[9], bs[9];
  load_phi9<R>(phi, b, ph);
  pull9<R>(N, n, k, b, lk, nn);
  node_update<R, true>(C, nn, ph, ns, bs, nullptr);
  N[k] = ns[0];
  B[k] = bs[0];
#pragma unroll
  for (int q = 1; q < 9; q++) {
    // towards x + c_q = x - c_opp(q): the slot nn[opp(q)] was read from; a solid node there sends it back (R12)
    const bool back = (lk >> (opp(q) - 1)) & 1u;
    const size_t dst = back ? (size_t)q * n + k : (size_t)opp(q) * n + b.src[opp(q)];
    N[dst] = ns[q];
    B[dst] = bs[q];
  }
}

template <typename R>
__global__ void __launch_bounds__(256) k_collide_aa_local(const Consts<R> C, const uint8_t* __restrict__ cls,
                                                          R* __restrict__ N, R* __restrict__ B,
                                                          const R* __restrict__ phi) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= C.nx) return;
  const size_t n = C.ps;
  const int k = j * C.nx + i;
  if (cls[k] >= 2) return;
  const Nbr b = make_nbr(i, j, C.nx, C.ny);
  R nn[9], ph[9], ns[9], bs[9];
  load_phi9<R>(phi, b, ph);
  nn[0] = N[k];
#pragma unroll
  for (int q = 1; q < 9; q++) nn[q] = N[(size_t)opp(q) * n + k];
  node_update<R, true>(C, nn, ph, ns, bs, nullptr);
#pragma unroll
  for (int q = 0; q < 9; q++) {
    N[(size_t)q * n + k] = ns[q];
    B[(size_t)q * n + k] = bs[q];
  }
}

// ------------------------------------------------------------------------------------------
// init (R14): N_i(x, 0) = N_i^eq(p = 0, u0(x)) (Eq. A4), B_i = phi0 N_i; stored "un-streamed" so
// that the pull of the first step returns exactly these values: slot (q, y) holds N_q(y + c_q, 0)
// if y + c_q is fluid, else N_opp(q)(y, 0) (the value the bounce-back link will hand back).
// ------------------------------------------------------------------------------------------
template <typename R>
__device__ __forceinline__ R neq_dev_p0(int q, R ux, R uy) {
  // deviation of Eq. A4 at p = 0
  const int cx[9] = {0, 1, 0, -1, 0, 1, -1, -1, 1}, cy[9] = {0, 0, 1, 0, -1, 1, 1, -1, -1};
  const R u2 = ux * ux + uy * uy;
  if (q == 0) return R(-2.0 / 3.0) * u2;
  const R w = q < 5 ? R(1.0 / 9.0) : R(1.0 / 36.0);
  const R cu = cx[q] * ux + cy[q] * uy;
  return w * (R(3.0) * cu + R(4.5) * cu * cu - R(1.5) * u2);
}

template <typename R>
__global__ void __launch_bounds__(256) k_init(const Consts<R> C, const uint8_t* __restrict__ cls,
                                              const uint8_t* __restrict__ links,
                                              const double* __restrict__ phi0,
                                              const double* __restrict__ u0, const PopView<R> Npop,
                                              R* __restrict__ Bpop, R* __restrict__ phiA,
                                              R* __restrict__ phiB) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= C.nx) return;
  const size_t n = C.ps;   // plane stride
  const int k = j * C.nx + i;
  const uint8_t c = cls[k];
  if (c >= 2) {
    phiA[k] = C.phi_solid;
    phiB[k] = C.phi_solid;
    const bool stored = Npop.has(k);   // a solid node travels with its group only if the group holds a fluid node
#pragma unroll
    for (int q = 0; q < 9; q++) {
      if (stored) Npop.at(q, k) = R(0);
      if (Bpop) Bpop[q * n + k] = R(0);
    }
    return;
  }
  const Nbr b = make_nbr(i, j, C.nx, C.ny);
  const unsigned lk = (c == 1) ? links[k] : 0u;
  const R chi[9] = {C.chi0, C.chi1, C.chi1, C.chi1, C.chi1, C.chi5, C.chi5, C.chi5, C.chi5};
  R s = R(0);
#pragma unroll
  for (int q = 0; q < 9; q++) {
    // is y + c_q solid?  y + c_q = y - c_opp(q): link bit of opp(q)
    const int oq = opp(q);
    const bool blocked = q > 0 && ((lk >> (oq - 1)) & 1u);
    const int src = blocked ? k : b.dst[q];
    const int qq = blocked ? oq : q;
    const R ux = u0 ? (R)u0[src] : R(0), uy = u0 ? (R)u0[(size_t)C.nx * C.ny + src] : R(0);
    const R dev = neq_dev_p0<R>(qq, ux, uy);
    Npop.at(q, k) = dev;
    if (Bpop) Bpop[q * n + k] = (R)phi0[src] * (chi[qq] + dev);
    // phi(x, 0) = sum_i B_i(x, 0) = sum_i phi0(x) N_i^eq(u0(x)) in the oracle's order (A13)
    const R uxk = u0 ? (R)u0[k] : R(0), uyk = u0 ? (R)u0[(size_t)C.nx * C.ny + k] : R(0);
    s += (R)phi0[k] * (chi[q] + neq_dev_p0<R>(q, uxk, uyk));
  }
  phiA[k] = s;
  phiB[k] = s;
}

// ------------------------------------------------------------------------------------------
// lbm_get: macroscopic fields at the current time into double staging planes
// ------------------------------------------------------------------------------------------
template <typename R>
__global__ void __launch_bounds__(256) k_moments(const Consts<R> C, const uint8_t* __restrict__ cls,
                                                 const uint8_t* __restrict__ links,
                                                 const PopView<R> Nsrc, const R* __restrict__ phi,
                                                 double* __restrict__ o_rho, double* __restrict__ o_phi,
                                                 double* __restrict__ o_ux, double* __restrict__ o_uy,
                                                 double* __restrict__ o_p) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= C.nx) return;
  const size_t n = C.ps;   // plane stride
  const int k = j * C.nx + i;
  const uint8_t c = cls[k];
  if (o_phi) o_phi[k] = (double)phi[k];
  if (c >= 2) {
    if (o_rho) o_rho[k] = 0.0;
    if (o_ux) o_ux[k] = 0.0;
    if (o_uy) o_uy[k] = 0.0;
    if (o_p) o_p[k] = 0.0;
    return;
  }
  const Nbr b = make_nbr(i, j, C.nx, C.ny);
  const unsigned lk = link_bits(C, c, links, k);
  R nn[9], ph[9], ns[9], bs[9];
  NodeOut<R> o;
  load_phi9<R>(phi, b, ph);
  pull9<R>(Nsrc, k, b, lk, nn);
  node_update<R, false>(C, nn, ph, ns, bs, &o);
  if (o_rho) o_rho[k] = (double)o.rho;
  if (o_ux) o_ux[k] = (double)o.ux;
  if (o_uy) o_uy[k] = (double)o.uy;
  if (o_p) o_p[k] = (double)o.p;
}

// post-stream population plane q (full N_q = chi_q + deviation, or B_q) into a double plane
template <typename R>
__global__ void __launch_bounds__(256) k_gather_plane(const Consts<R> C, const uint8_t* __restrict__ cls,
                                                      const uint8_t* __restrict__ links,
                                                      const PopView<R> pop, int q, double add,
                                                      double* __restrict__ out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= C.nx) return;
  const size_t n = C.ps;   // plane stride
  const int k = j * C.nx + i;
  const uint8_t c = cls[k];
  if (c >= 2) { out[k] = 0.0; return; }
  const Nbr b = make_nbr(i, j, C.nx, C.ny);
  const unsigned lk = link_bits(C, c, links, k);
  R v;
  if (q == 0) v = pop.at(0, k);
  else v = ((lk >> (q - 1)) & 1u) ? pop.at(opp(q), k) : pop.at(q, b.src[q]);
  out[k] = (double)v + add;
}

// lbm_set_populations: the inverse of k_gather_plane.  in[k] = post-stream N_q(x_k, t) (or B_q); the state keeps
// the value at the node the pull will take it from: slot (q, x - c_q), or the node's own slot opp(q) behind a
// bounce-back link.  Every slot a fluid node will pull from has exactly one writer.
template <typename R>
__global__ void __launch_bounds__(256) k_scatter_plane(const Consts<R> C, const uint8_t* __restrict__ cls,
                                                       const uint8_t* __restrict__ links,
                                                       const double* __restrict__ in, int q, double sub,
                                                       const PopView<R> pop) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= C.nx) return;
  const size_t n = C.ps;   // plane stride
  const int k = j * C.nx + i;
  const uint8_t c = cls[k];
  if (c >= 2) return;
  const Nbr b = make_nbr(i, j, C.nx, C.ny);
  const unsigned lk = (c == 1) ? links[k] : 0u;
  const R v = (R)(in[k] - sub);
  if (q == 0) pop.at(0, k) = v;
  else if ((lk >> (q - 1)) & 1u) pop.at(opp(q), k) = v;
  else pop.at(q, b.src[q]) = v;
}
// phi = sum_q B_q on fluid nodes (A13, :311), accumulated plane by plane in the oracle's order q = 0 .. 8
template <typename R>
__global__ void __launch_bounds__(256) k_phi_accumulate(const Consts<R> C, const uint8_t* __restrict__ cls,
                                                        const double* __restrict__ in, int first,
                                                        double* __restrict__ acc, R* __restrict__ phi_final) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= C.nx) return;
  const int k = j * C.nx + i;
  if (cls[k] >= 2) return;
  const double s = (first ? 0.0 : acc[k]) + in[k];
  acc[k] = s;
  if (phi_final) phi_final[k] = (R)s;
}

// same at selected nodes: out[q*m + t]
template <typename R>
__global__ void __launch_bounds__(128) k_gather_samples(const Consts<R> C, const uint8_t* __restrict__ cls,
                                                        const uint8_t* __restrict__ links,
                                                        const PopView<R> pop, int add_chi,
                                                        long long m, const long long* __restrict__ idx,
                                                        double* __restrict__ out) {
  const long long t = (long long)blockIdx.x * 128 + threadIdx.x;
  if (t >= m) return;
  const size_t n = C.ps;   // plane stride
  const int k = (int)idx[t];
  const uint8_t c = cls[k];
  const Nbr b = make_nbr(k % C.nx, k / C.nx, C.nx, C.ny);
  const unsigned lk = link_bits(C, c, links, k);
  const double chi[9] = {(double)C.chi0, (double)C.chi1, (double)C.chi1, (double)C.chi1, (double)C.chi1,
                         (double)C.chi5, (double)C.chi5, (double)C.chi5, (double)C.chi5};
  for (int q = 0; q < 9; q++) {
    double v = 0.0;
    if (c < 2) {
      R x;
      if (q == 0) x = pop.at(0, k);
      else x = ((lk >> (q - 1)) & 1u) ? pop.at(opp(q), k) : pop.at(q, b.src[q]);
      v = (double)x + (add_chi ? chi[q] : 0.0);
    }
    out[q * m + t] = v;
  }
}

// ------------------------------------------------------------------------------------------
// (a8) diagnostics: warp-shuffle + fixed-tree block reduction into per-block partials, then a
// single-block fixed-order pass.  Deterministic for a given grid.
// partial layout: [6][nblocks]: sum phi, sum (1-phi), KE, max|u|^2, min phi, max phi; + count, nan
// ------------------------------------------------------------------------------------------
struct DiagVec { double s_phi, s_omp, ke, umax2, pmin, pmax, cnt, bad; };

__device__ __forceinline__ DiagVec diag_combine(const DiagVec& a, const DiagVec& b) {
  DiagVec r;
  r.s_phi = a.s_phi + b.s_phi; r.s_omp = a.s_omp + b.s_omp; r.ke = a.ke + b.ke;
  r.umax2 = fmax(a.umax2, b.umax2); r.pmin = fmin(a.pmin, b.pmin); r.pmax = fmax(a.pmax, b.pmax);
  r.cnt = a.cnt + b.cnt; r.bad = fmax(a.bad, b.bad);
  return r;
}
__device__ __forceinline__ DiagVec diag_shfl_down(const DiagVec& a, int d) {
  DiagVec r;
  r.s_phi = __shfl_down_sync(0xffffffffu, a.s_phi, d); r.s_omp = __shfl_down_sync(0xffffffffu, a.s_omp, d);
  r.ke = __shfl_down_sync(0xffffffffu, a.ke, d); r.umax2 = __shfl_down_sync(0xffffffffu, a.umax2, d);
  r.pmin = __shfl_down_sync(0xffffffffu, a.pmin, d); r.pmax = __shfl_down_sync(0xffffffffu, a.pmax, d);
  r.cnt = __shfl_down_sync(0xffffffffu, a.cnt, d); r.bad = __shfl_down_sync(0xffffffffu, a.bad, d);
  return r;
}
__device__ __forceinline__ DiagVec diag_identity() {
  DiagVec r;
  r.s_phi = 0; r.s_omp = 0; r.ke = 0; r.umax2 = 0; r.cnt = 0; r.bad = 0;
  r.pmin = __longlong_as_double(0x7ff0000000000000LL); r.pmax = -r.pmin;
  return r;
}
__device__ __forceinline__ DiagVec diag_block_reduce(DiagVec v, DiagVec* sh) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v = diag_combine(v, diag_shfl_down(v, d));
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  if (lane == 0) sh[w] = v;
  __syncthreads();
  if (w == 0) {
    v = lane < nw ? sh[lane] : diag_identity();
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v = diag_combine(v, diag_shfl_down(v, d));
  }
  return v;  // valid in thread 0
}

template <typename R>
__global__ void __launch_bounds__(256) k_diag_partial(const Consts<R> C, const uint8_t* __restrict__ cls,
                                                      const uint8_t* __restrict__ links,
                                                      const PopView<R> Nsrc, const R* __restrict__ phi,
                                                      DiagVec* __restrict__ partial) {
  __shared__ DiagVec sh[32];
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  DiagVec v = diag_identity();
  if (i < C.nx) {
    const size_t n = C.ps;   // plane stride
    const int k = j * C.nx + i;
    const uint8_t c = cls[k];
    if (c < 2) {
      const Nbr b = make_nbr(i, j, C.nx, C.ny);
      const unsigned lk = link_bits(C, c, links, k);
      R nn[9], ph[9], ns[9], bs[9];
      NodeOut<R> o;
      load_phi9<R>(phi, b, ph);
      pull9<R>(Nsrc, k, b, lk, nn);
      node_update<R, false>(C, nn, ph, ns, bs, &o);
      const double f = (double)ph[0], ux = (double)o.ux, uy = (double)o.uy;
      const double u2 = ux * ux + uy * uy;
      v.s_phi = f; v.s_omp = 1.0 - f; v.ke = 0.5 * (double)o.rho * u2; v.umax2 = u2;
      v.pmin = f; v.pmax = f; v.cnt = 1.0;
      v.bad = (f != f || u2 != u2) ? 1.0 : 0.0;
      if (v.bad != 0.0) { v.umax2 = 0.0; v.pmin = diag_identity().pmin; v.pmax = -v.pmin; }
    }
  }
  v = diag_block_reduce(v, sh);
  if (threadIdx.x == 0) partial[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = v;
}

__global__ void __launch_bounds__(1024) k_diag_final(const DiagVec* __restrict__ partial, long long m,
                                                     double* __restrict__ out) {
  __shared__ DiagVec sh[32];
  DiagVec v = diag_identity();
  for (long long t = threadIdx.x; t < m; t += 1024) v = diag_combine(v, partial[t]);
  v = diag_block_reduce(v, sh);
  if (threadIdx.x == 0) {
    out[0] = v.s_phi; out[1] = v.s_omp; out[2] = v.ke; out[3] = sqrt(v.umax2);
    out[4] = v.pmin; out[5] = v.pmax; out[6] = v.cnt; out[7] = v.bad;
  }
}

// ------------------------------------------------------------------------------------------
// Measurement helper (lbm_layout_copy_timed): the ceiling of the SoA-with-holes layout.  One thread
// per 32-byte sector of a population plane; a sector that holds a fluid node is copied whole, for
// all 9 planes and phi.  No halos, no arithmetic: what a pure streaming pass over the state costs.
// NPS = nodes per sector (8 in fp32, 4 in fp64).
// ------------------------------------------------------------------------------------------
template <int NPS>
__global__ void __launch_bounds__(256) k_copy_sectors(const uint16_t* __restrict__ cl16, const float4* __restrict__ src,
                                                      float4* __restrict__ dst, const float4* __restrict__ phi_src,
                                                      float4* __restrict__ phi_dst, size_t nsec, size_t plane_sec) {
  for (size_t k = (size_t)blockIdx.x * 256 + threadIdx.x; k < nsec; k += (size_t)gridDim.x * 256) {
    bool any = false;
    const unsigned* w = reinterpret_cast<const unsigned*>(cl16) + k * (NPS / 2);
#pragma unroll
    for (int t = 0; t < NPS / 2; t++) any |= ((w[t] & 0xffu) < 2u) || (((w[t] >> 16) & 0xffu) < 2u);
    if (any) {
#pragma unroll
      for (int q = 0; q < 9; q++) {
        const float4 a = src[(q * plane_sec + k) * 2], b = src[(q * plane_sec + k) * 2 + 1];
        dst[(q * plane_sec + k) * 2] = a;
        dst[(q * plane_sec + k) * 2 + 1] = b;
      }
      phi_dst[2 * k] = phi_src[2 * k];
      phi_dst[2 * k + 1] = phi_src[2 * k + 1];
    }
  }
}

// ------------------------------------------------------------------------------------------
// PACK schedule: group-compacted population planes.  A plane stores only the aligned groups of G
// x-adjacent nodes (G = nodes per lane of the kernel: 2, or 4 for the fp32 quad variant) that hold a
// fluid node, row after row, without holes.  ptab[r * nw + w] = {bit b set <=> group 32 w + b of row r
// holds a fluid node, compact index of the first group of that word}; the compact index of group p of
// row r is ptab[..].y + popc(ptab[..].x & ((1 << (p & 31)) - 1)).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_pair_mask(const uint8_t* __restrict__ cls, int nx, int ny, int nw, int G,
                                                   unsigned* __restrict__ pmask, int* __restrict__ pcount) {
  const long long t = (long long)blockIdx.x * 256 + threadIdx.x;
  if (t >= (long long)ny * nw) return;
  const int r = (int)(t / nw), w = (int)(t % nw);
  unsigned m = 0;
  for (int b = 0; b < 32; b++) {
    const int x = G * (32 * w + b);
    if (x < nx) {
      const size_t k = (size_t)r * nx + x;
      bool any = false;
      for (int c = 0; c < G; c++) any |= cls[k + c] < 2;
      if (any) m |= 1u << b;
    }
  }
  pmask[t] = m;
  pcount[t] = __popc(m);
}
__global__ void __launch_bounds__(256) k_pair_tab(const unsigned* __restrict__ pmask, const int* __restrict__ pbase,
                                                  long long nwords, uint2* __restrict__ ptab) {
  const long long t = (long long)blockIdx.x * 256 + threadIdx.x;
  if (t < nwords) ptab[t] = make_uint2(pmask[t], (unsigned)pbase[t]);
}
// dense (pop[q * ps + k]) <-> compact copies of the 9 planes; TO_COMPACT packs, else unpacks (the solid nodes of a
// group travel with it; other dense entries are untouched).  Compact element (q, group ci, node c): plane-major
// popc[(q * cps + ci) * G + c] (PACK), or group-major popc[(ci * 9 + q) * G + c] (SPARSE: the nine vectors of a
// group are contiguous, so a row of a strip is one contiguous run).
template <typename R, bool TO_COMPACT>
__global__ void __launch_bounds__(256) k_pair_repack(const uint2* __restrict__ ptab, int nx, int ny, int nw, int G,
                                                     size_t ps, size_t cps, R* __restrict__ dense,
                                                     R* __restrict__ compact, int group_major) {
  const long long t = (long long)blockIdx.x * 256 + threadIdx.x;   // one thread per group
  const int npr = nx / G;
  if (t >= (long long)ny * npr) return;
  const int r = (int)(t / npr), p = (int)(t % npr);
  const uint2 tb = ptab[(size_t)r * nw + (p >> 5)];
  if (!((tb.x >> (p & 31)) & 1u)) return;
  const size_t ci = (size_t)tb.y + (size_t)__popc(tb.x & ((1u << (p & 31)) - 1u));
  const size_t k = (size_t)r * nx + (size_t)G * p;
  for (int q = 0; q < 9; q++)
    for (int c = 0; c < G; c++) {
      const size_t e = group_major ? (ci * 9 + q) * G + c : (q * cps + ci) * G + c;
      if (TO_COMPACT) compact[e] = dense[q * ps + k + c];
      else dense[q * ps + k + c] = compact[e];
    }
}

// test hook: independent nodes
template <typename R>
__global__ void __launch_bounds__(128) k_node_batch(const Consts<R> C, long long count,
                                                    const double* __restrict__ Nin,
                                                    const double* __restrict__ phin,
                                                    double* __restrict__ Ns, double* __restrict__ Bs,
                                                    double* __restrict__ fields) {
  const long long t = (long long)blockIdx.x * 128 + threadIdx.x;
  if (t >= count) return;
  const R chi[9] = {C.chi0, C.chi1, C.chi1, C.chi1, C.chi1, C.chi5, C.chi5, C.chi5, C.chi5};
  const double chid[9] = {(double)C.chi0, (double)C.chi1, (double)C.chi1, (double)C.chi1, (double)C.chi1,
                          (double)C.chi5, (double)C.chi5, (double)C.chi5, (double)C.chi5};
  R nn[9], ph[9], ns[9], bs[9];
  NodeOut<R> o;
  for (int q = 0; q < 9; q++) {
    nn[q] = (R)(Nin[9 * t + q] - chid[q]);   // deviation taken in double, then rounded
    ph[q] = (R)phin[9 * t + q];
  }
  (void)chi;
  node_update<R, true>(C, nn, ph, ns, bs, &o);
  for (int q = 0; q < 9; q++) {
    if (Ns) Ns[9 * t + q] = (double)ns[q] + chid[q];
    if (Bs) Bs[9 * t + q] = (double)bs[q];
  }
  if (fields) {
    double* f = fields + 8 * t;
    f[0] = o.rho; f[1] = o.tau; f[2] = o.ux; f[3] = o.uy; f[4] = o.p; f[5] = o.Fx; f[6] = o.Fy; f[7] = o.gnorm;
  }
}

}  // namespace lbm

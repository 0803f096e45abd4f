// lbm_warp.cuh — WARP schedule: the fused pull-stream + collide + segregation + phi(t+1) kernel,
// barrier-free, with an asynchronous-copy pipeline per warp.  Same arithmetic per node as
// lbm_fused.cuh (node_update), same HBM state (9 N planes, phi, class), different decomposition:
//
//   * one warp owns 30 output columns (+1 halo column per side, collided redundantly) and marches
//     down TY rows (+1 halo row per end).  Warps never wait on one another (no __syncthreads).
//   * phi(x, t+1) = sum_q B_q*(x - c_q, t) (A13 after A16-A17, :311-322) is assembled in registers:
//     the three B* that move in x come from the neighbouring lanes by warp shuffle, the row moves
//     are carried from one iteration of the march to the next.  Bounce-back links (R12) hand the
//     node its own opposite B* back; solid lanes contribute zeros.
//   * loads run D rows ahead of the collision through cp.async (LDGSTS) into a private shared-memory
//     ring of the warp: every lane copies the nine pulled N of its node (per-element predication:
//     solid nodes are never fetched; a bounce-back link redirects the copy to the node's own
//     opposite population), its phi and the 4-byte word holding its class/link word.  One commit
//     group per march row; cp.async.wait_group D-1 at the top of an iteration guarantees the row
//     being collided has landed.  Register-ring prefetching was tried first (profiles/
//     r1_v2, r1_v3): the six per-warp scoreboards alias loads of different rows, so a deep register
//     pipeline stalls at the first re-use of a scoreboard; commit groups do not have that limit.
//   * all indices are 32-bit element offsets (9 n < 2^32 is checked by lbm_create); the row parts are
//     warp-uniform, the column parts (x, x-1, x+1 with periodic wrap) per-lane constants.
#pragma once
#include "lbm_kernels.cuh"

namespace lbm {

template <int BYTES>
__device__ __forceinline__ void cp_async(unsigned saddr, const void* gptr) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(saddr), "l"(gptr), "n"(BYTES) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// shared-memory ring of one warp
template <typename R, int D>
struct WarpRing {
  static constexpr int NS = D + 1;      // N stages: march rows i .. i+D
  static constexpr int PS = D + 3;      // phi stages: rows i-1 .. i+D+1
  static constexpr int CS = D + 1;      // class stages: rows i+D .. i+2D
  static constexpr int PW = 36;         // phi row: entry 0 = column x0-2, 1..32 = lanes, 33 = x0+31
  R N[NS][9][32];
  R P[PS][PW];
  unsigned Cw[CS][32];
};

template <typename R, int D, int WARPS, int MINB, bool WRITE_B>
__global__ void __launch_bounds__(32 * WARPS, MINB)
    k_fused_warp(const Consts<R> C, const uint16_t* __restrict__ cl16, const R* __restrict__ Nsrc,
                 R* __restrict__ Ndst, R* __restrict__ Bdst, const R* __restrict__ phi_in,
                 R* __restrict__ phi_out, int TY) {
  using Ring = WarpRing<R, D>;
  constexpr unsigned FULL = 0xffffffffu;
  constexpr int SZ = (int)sizeof(R);
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Ring& S = reinterpret_cast<Ring*>(smem_raw)[threadIdx.x >> 5];
  const unsigned sbase = (unsigned)__cvta_generic_to_shared(&S);
  const unsigned sN0 = sbase + (unsigned)offsetof(Ring, N), sP0 = sbase + (unsigned)offsetof(Ring, P),
                 sC0 = sbase + (unsigned)offsetof(Ring, Cw);

  const int nx = C.nx, ny = C.ny;
  const unsigned n = (unsigned)C.ps;   // plane stride
  const int lane = threadIdx.x & 31;
  const int x0 = (blockIdx.x * WARPS + (threadIdx.x >> 5)) * 30;
  if (x0 >= nx) return;                                  // whole warp; the kernel has no block barrier
  const int xend = min(x0 + 30, nx);                     // one past the last output column
  const int lx = x0 - 1 + lane;                          // logical column, may be -1 or nx
  const bool col_active = lx <= xend;
  const bool col_out = lane >= 1 && lx < xend;
  // every lane keeps its place in the periodic column sequence (inactive lanes too: their phi
  // entries are the right halo lane's neighbours); nx may be smaller than the strip
  auto wrapx = [nx](int v) { v %= nx; return v < 0 ? v + nx : v; };
  const int x = wrapx(lx);
  const unsigned eC = (unsigned)x, eW = (unsigned)wrapx(x - 1), eE = (unsigned)wrapx(x + 1);
  // lanes 0 and 31 also fetch the phi column outside the strip that their stencil needs
  const bool edge = lane == 0 || lane == 31;
  const unsigned eX = lane == 0 ? eW : eE;
  const unsigned pX = lane == 0 ? 0u : 33u;
  const unsigned solid_mask = col_active ? 0u : 3u;      // OR-ed into the class byte: inactive lanes are solid
  const int j0 = blockIdx.y * TY;
  const int rows = min(TY, ny - j0);
  const int last = rows + 1;                             // last march row (march row m = grid row j0-1+m)

  // element offset of march row m (periodic in y)
  auto rowoff = [=](int m) -> unsigned {
    int r = j0 - 1 + m;
    r = r < 0 ? r + ny : (r >= ny ? r - ny : r);
    return (unsigned)r * (unsigned)nx;
  };
  // ---- issue helpers (all asynchronous) ----
  auto issue_phi = [&](int m, int slot) {   // phi of march row m into phi stage `slot`
    const unsigned u = rowoff(m);
    const unsigned d = sP0 + (unsigned)(slot * Ring::PW) * SZ;
    cp_async<SZ>(d + (unsigned)(lane + 1) * SZ, phi_in + (u + eC));
    if (edge) cp_async<SZ>(d + pX * SZ, phi_in + (u + eX));
  };
  auto issue_cls = [&](int m, int slot) {   // the aligned 4 bytes that hold the class word of (x, m)
    const unsigned k = rowoff(m) + eC;
    cp_async<4>(sC0 + (unsigned)(slot * 32 + lane) * 4u, cl16 + (k & ~1u));
  };
  auto class_word = [&](unsigned raw, int m) -> unsigned {
    const unsigned k = rowoff(m) + eC;
    return ((raw >> ((k & 1u) * 16u)) & 0xffffu) | solid_mask;
  };
  auto issue_N = [&](int m, int slot, unsigned w) {   // nine pulled N of march row m (class word w)
    const bool fl = (w & 0xffu) < 2u;
    const unsigned lk = fl ? (w >> 8) : 0u;
    const bool any_link = __any_sync(FULL, lk != 0u);
    if (!fl) return;
    const unsigned uS = rowoff(m - 1), uC = rowoff(m), uN = rowoff(m + 1);
    const unsigned kC = uC + eC;
    const unsigned d = sN0 + (unsigned)(slot * 9 * 32 + lane) * SZ;
    const unsigned src[9] = {kC, (1u * n + uC) + eW, (2u * n + uS) + eC, (3u * n + uC) + eE, (4u * n + uN) + eC,
                             (5u * n + uS) + eW, (6u * n + uS) + eE, (7u * n + uN) + eE, (8u * n + uN) + eW};
    cp_async<SZ>(d, Nsrc + kC);
    if (!any_link) {   // warp-uniform
#pragma unroll
      for (int q = 1; q < 9; q++) cp_async<SZ>(d + (unsigned)(q * 32) * SZ, Nsrc + src[q]);
    } else {
#pragma unroll
      for (int q = 1; q < 9; q++) {
        const bool b = (lk >> (q - 1)) & 1u;
        cp_async<SZ>(d + (unsigned)(q * 32) * SZ, Nsrc + (b ? (unsigned)opp(q) * n + kC : src[q]));
      }
    }
  };

  // ---- prologue ----
  // group A: phi rows -1 .. D, class words of rows 0 .. 2D-1 (rows 0..D-1 go straight to `hist`)
  unsigned long long hist = 0ull;   // class words of march rows i .. i+D-1, 16 bits each
  unsigned w_pro[D];
#pragma unroll
  for (int m = 0; m < D; m++) w_pro[m] = m <= last ? (unsigned)cl16[rowoff(m) + eC] : 3u;
  for (int m = -1; m <= D; m++)
    if (m <= last + 1) issue_phi(m, (m + Ring::PS) % Ring::PS);
  for (int m = D; m < 2 * D; m++)
    if (m <= last) issue_cls(m, m % Ring::CS);
  cp_async_commit();
#pragma unroll
  for (int m = 0; m < D; m++) {
    w_pro[m] |= solid_mask;
    hist |= (unsigned long long)(w_pro[m] & 0xffffu) << (16 * m);
  }
  // groups -D .. -1: pulled N of rows 0 .. D-1
#pragma unroll
  for (int m = 0; m < D; m++) {
    issue_N(m, m % Ring::NS, m <= last ? w_pro[m] : 3u);
    cp_async_commit();
  }

  unsigned kout = (unsigned)(j0 - 1) * (unsigned)nx + eC;   // own node of march row i (used for 1 <= i <= rows)
  R acc_prev = R(0), up_prev = R(0);
  bool fl_prev = false;
  // phi slot of row m is (m + PS) % PS, N slot m % NS, class slot m % CS; tracked incrementally
  int slotN_i = 0, slotN_iD = D % Ring::NS;
  int slotP_im1 = (Ring::PS - 1) % Ring::PS, slotP_new = (D + 1) % Ring::PS;
  int slotC_iD = D % Ring::CS, slotC_new = (2 * D) % Ring::CS;
  auto inc = [](int s, int mod) { return s + 1 == mod ? 0 : s + 1; };

  for (int i = 0; i <= last; i++) {
    cp_async_wait<D - 1>();   // groups up to i-D have landed: N of row i, phi of row i+1, class of row i+D
    __syncwarp();             // phi entries are read across lanes
    // ---- issue: N of march row i+D, phi of row i+D+1, class word of row i+2D ----
    {
      const int m = i + D;
      unsigned w = 3u;
      if (m <= last) w = class_word(S.Cw[slotC_iD][lane], m);
      hist |= (unsigned long long)w << (16 * D);
      if (m <= last) issue_N(m, slotN_iD, w);
      if (m + 1 <= last + 1) issue_phi(m + 1, slotP_new);
      if (m + D <= last) issue_cls(m + D, slotC_new);
      cp_async_commit();
    }

    // ---- collide march row i ----
    const unsigned w_cur = (unsigned)hist & 0xffffu;
    hist >>= 16;
    const bool fl = (w_cur & 0xffu) < 2u;
    const unsigned lk = fl ? (w_cur >> 8) : 0u;
    R bs[9];
#pragma unroll
    for (int q = 0; q < 9; q++) bs[q] = R(0);
    R bb = R(0);
    if (fl) {
      const int pa = slotP_im1, pb = inc(pa, Ring::PS), pc = inc(pb, Ring::PS);
      const R* pS = S.P[pa] + lane;   // entries lane, lane+1, lane+2 = columns x-1, x, x+1
      const R* pC = S.P[pb] + lane;
      const R* pN = S.P[pc] + lane;
      const R ph[9] = {pC[1], pC[2], pN[1], pC[0], pS[1], pN[2], pN[0], pS[0], pS[2]};
      R nn[9], ns[9];
#pragma unroll
      for (int q = 0; q < 9; q++) nn[q] = S.N[slotN_i][q][lane];
      node_update<R, true>(C, nn, ph, ns, bs, nullptr);
      if (col_out && i >= 1 && i <= rows) {
#pragma unroll
        for (int q = 0; q < 9; q++) Ndst[(unsigned)q * n + kout] = ns[q];
        if (WRITE_B) {
#pragma unroll
          for (int q = 0; q < 9; q++) Bdst[(unsigned)q * n + kout] = bs[q];
        }
      }
      if (lk) {   // half-way bounce-back: link q hands the node its own B_opp(q)* back
#pragma unroll
        for (int q = 1; q < 9; q++) bb += ((lk >> (q - 1)) & 1u) ? bs[opp(q)] : R(0);
      }
    }
    // contributions of row i to phi(t+1) of rows i-1 (down), i (mid), i+1 (up)
    const R mid = bs[0] + __shfl_up_sync(FULL, bs[1], 1) + __shfl_down_sync(FULL, bs[3], 1);
    const R upw = bs[2] + __shfl_up_sync(FULL, bs[5], 1) + __shfl_down_sync(FULL, bs[6], 1);
    const R down = bs[4] + __shfl_down_sync(FULL, bs[7], 1) + __shfl_up_sync(FULL, bs[8], 1);
    if (i >= 2 && col_out && fl_prev) phi_out[kout - (unsigned)nx] = acc_prev + down;
    acc_prev = (up_prev + mid) + bb;
    up_prev = upw;
    fl_prev = fl;

    kout += (unsigned)nx;
    slotN_i = inc(slotN_i, Ring::NS); slotN_iD = inc(slotN_iD, Ring::NS);
    slotP_im1 = inc(slotP_im1, Ring::PS); slotP_new = inc(slotP_new, Ring::PS);
    slotC_iD = inc(slotC_iD, Ring::CS); slotC_new = inc(slotC_new, Ring::CS);
  }
  cp_async_wait<0>();
}

template <typename R>
struct WarpCfg {   // pipeline depth and CTA shape per precision (smem: fp32 6.0 KB, fp64 8.9 KB per warp)
  static constexpr int D = sizeof(R) == 8 ? 2 : 3;
  static constexpr int WARPS = 4;
  static constexpr int MINB = sizeof(R) == 8 ? 5 : 6;
};

template <typename R>
int launch_fused_warp(const Consts<R>& C, const uint16_t* cl16, const R* Nsrc, R* Ndst, R* Bdst,
                      const R* phi_in, R* phi_out, cudaStream_t st) {
  using Cfg = WarpCfg<R>;
  constexpr int D = Cfg::D, WARPS = Cfg::WARPS, MINB = Cfg::MINB;
  const int nwx = (C.nx + 29) / 30;
  const int gx = (nwx + WARPS - 1) / WARPS;
  // rows per warp march: long marches amortise the two halo rows; small grids need enough CTAs
  int TY = 64;
  while (TY > 8 && (long long)gx * ((C.ny + TY - 1) / TY) < 148 * 8) TY >>= 1;
  const dim3 grid((unsigned)gx, (unsigned)((C.ny + TY - 1) / TY), 1);
  const size_t smem = sizeof(WarpRing<R, D>) * WARPS;
  static bool attr_set[2] = {false, false};
  auto kern = Bdst ? k_fused_warp<R, D, WARPS, MINB, true> : k_fused_warp<R, D, WARPS, MINB, false>;
  if (!attr_set[Bdst ? 1 : 0]) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return (int)e;
    attr_set[Bdst ? 1 : 0] = true;
  }
  kern<<<grid, 32 * WARPS, smem, st>>>(C, cl16, Nsrc, Ndst, Bdst, phi_in, phi_out, TY);
  return 0;
}

}  // namespace lbm

// lbm_warp.cuh — WARP schedule: the fused pull-stream + collide + segregation + phi(t+1) kernel with
// no shared memory and no block barrier.  Same arithmetic per node as lbm_fused.cuh (node_update),
// same HBM state (9 N planes, phi, class), different decomposition:
//
//   * one warp owns 30 output columns (+1 halo column per side, collided redundantly) and marches
//     down TY rows (+1 halo row per end).  Warps never wait on one another.
//   * phi(x, t+1) = sum_q B_q*(x - c_q, t) (A13 after A16-A17, :311-322) is assembled in registers:
//     the three B* that move in x come from the neighbouring lanes by warp shuffle, the row moves
//     are carried from one iteration of the march to the next.  Bounce-back links (R12) hand the
//     node its own opposite B* back; solid lanes contribute zeros.
//   * the march is software-pipelined: class word and phi row two rows ahead, the nine pulled N of the
//     next row, are in flight while the current row is collided, so one warp keeps ~2 rows of loads
//     outstanding without help from occupancy.
//   * class byte and bounce-back link byte travel as one 16-bit word (cl16).
#pragma once
#include "lbm_kernels.cuh"

namespace lbm {

template <typename R>
__device__ __forceinline__ void load_pulled(R (&nn)[9], const R* __restrict__ Nsrc, size_t n, unsigned lk,
                                            bool any_link, int k, int kW, int kE, int kS, int kN, int kSW,
                                            int kSE, int kNW, int kNE) {
  nn[0] = Nsrc[k];
  if (!any_link) {   // warp-uniform: no lane of this warp has a bounce-back link on this row
    nn[1] = Nsrc[1 * n + kW];  nn[2] = Nsrc[2 * n + kS];
    nn[3] = Nsrc[3 * n + kE];  nn[4] = Nsrc[4 * n + kN];
    nn[5] = Nsrc[5 * n + kSW]; nn[6] = Nsrc[6 * n + kSE];
    nn[7] = Nsrc[7 * n + kNE]; nn[8] = Nsrc[8 * n + kNW];
  } else {
    const int src[9] = {k, kW, kS, kE, kN, kSW, kSE, kNE, kNW};
#pragma unroll
    for (int q = 1; q < 9; q++) {
      const bool b = (lk >> (q - 1)) & 1u;
      const size_t off = b ? (size_t)opp(q) * n + (size_t)k : (size_t)q * n + (size_t)src[q];
      nn[q] = Nsrc[off];
    }
  }
}

template <typename R, int WARPS, int MINB, bool WRITE_B>
__global__ void __launch_bounds__(32 * WARPS, MINB)
    k_fused_warp(const Consts<R> C, const uint16_t* __restrict__ cl16, const R* __restrict__ Nsrc,
                 R* __restrict__ Ndst, R* __restrict__ Bdst, const R* __restrict__ phi_in,
                 R* __restrict__ phi_out, int TY) {
  constexpr unsigned FULL = 0xffffffffu;
  const int nx = C.nx, ny = C.ny;
  const size_t n = (size_t)nx * ny;
  const int lane = threadIdx.x & 31;
  const int x0 = (blockIdx.x * WARPS + (threadIdx.x >> 5)) * 30;
  if (x0 >= nx) return;                                  // whole warp; the kernel has no block barrier
  const int xend = min(x0 + 30, nx);                     // one past the last output column
  const int lx = x0 - 1 + lane;                          // logical column, may be -1 or nx
  const bool col_active = lx <= xend;
  const bool col_out = lane >= 1 && lx < xend;
  int x = lx;
  if (x < 0) x += nx;
  if (x >= nx) x -= nx;
  if (!col_active) x = 0;
  const int xm = (x == 0) ? nx - 1 : x - 1, xp = (x == nx - 1) ? 0 : x + 1;
  const int j0 = blockIdx.y * TY;
  const int rows = min(TY, ny - j0);

  auto wrap_row = [ny](int r) { return r < 0 ? r + ny : (r >= ny ? r - ny : r); };
  auto load_cl = [&](int rbase) -> unsigned { return col_active ? (unsigned)cl16[rbase + x] : 3u; };

  // ---- prologue: rows j0-2 .. j0 of phi, class words of rows j0-1 and j0, pulled N of row j0-1 ----
  int bS = wrap_row(j0 - 2) * nx, bC = wrap_row(j0 - 1) * nx, bN = wrap_row(j0) * nx;
  R pS[3], pC[3], pN[3], pNN[3];
  pS[0] = phi_in[bS + xm]; pS[1] = phi_in[bS + x]; pS[2] = phi_in[bS + xp];
  pC[0] = phi_in[bC + xm]; pC[1] = phi_in[bC + x]; pC[2] = phi_in[bC + xp];
  pN[0] = phi_in[bN + xm]; pN[1] = phi_in[bN + x]; pN[2] = phi_in[bN + xp];
  unsigned w_cur = load_cl(bC), w_next = load_cl(bN), w_nn = 3u;
  R ncur[9], nnext[9];
#pragma unroll
  for (int q = 0; q < 9; q++) ncur[q] = nnext[q] = R(0);
  {
    const bool fl = (w_cur & 0xffu) < 2u;
    const unsigned lk = fl ? (w_cur >> 8) : 0u;
    const bool any_link = __any_sync(FULL, lk != 0u);
    if (fl) load_pulled<R>(ncur, Nsrc, n, lk, any_link, bC + x, bC + xm, bC + xp, bS + x, bN + x, bS + xm,
                           bS + xp, bN + xm, bN + xp);
  }

  R acc_prev = R(0), up_prev = R(0);
  bool fl_prev = false;
  for (int rr = -1; rr <= rows; rr++) {
    // rows: bC = row rr (collided now), bN = row rr+1 (its N are fetched now), bNN = row rr+2
    const int bNN = wrap_row(j0 + rr + 2) * nx;
    const bool more = rr < rows;
    if (more) {
      w_nn = load_cl(bNN);
      pNN[0] = phi_in[bNN + xm]; pNN[1] = phi_in[bNN + x]; pNN[2] = phi_in[bNN + xp];
      const bool fln = (w_next & 0xffu) < 2u;
      const unsigned lkn = fln ? (w_next >> 8) : 0u;
      const bool any_link = __any_sync(FULL, lkn != 0u);
      if (fln) load_pulled<R>(nnext, Nsrc, n, lkn, any_link, bN + x, bN + xm, bN + xp, bC + x, bNN + x,
                              bC + xm, bC + xp, bNN + xm, bNN + xp);
    }

    const bool fl = (w_cur & 0xffu) < 2u;
    const unsigned lk = fl ? (w_cur >> 8) : 0u;
    const int k = bC + x;
    R bs[9];
#pragma unroll
    for (int q = 0; q < 9; q++) bs[q] = R(0);
    R bb = R(0);
    if (fl) {
      const R ph[9] = {pC[1], pC[2], pN[1], pC[0], pS[1], pN[2], pN[0], pS[0], pS[2]};
      R ns[9];
      node_update<R, true>(C, ncur, ph, ns, bs, nullptr);
      if (col_out && rr >= 0 && rr < rows) {
#pragma unroll
        for (int q = 0; q < 9; q++) Ndst[q * n + k] = ns[q];
        if (WRITE_B) {
#pragma unroll
          for (int q = 0; q < 9; q++) Bdst[q * n + k] = bs[q];
        }
      }
      if (lk) {   // half-way bounce-back: link q hands the node its own B_opp(q)* back
#pragma unroll
        for (int q = 1; q < 9; q++) bb += ((lk >> (q - 1)) & 1u) ? bs[opp(q)] : R(0);
      }
    }
    // contributions of row rr to phi(t+1) of rows rr-1 (down), rr (mid), rr+1 (up)
    const R mid = bs[0] + __shfl_up_sync(FULL, bs[1], 1) + __shfl_down_sync(FULL, bs[3], 1);
    const R up = bs[2] + __shfl_up_sync(FULL, bs[5], 1) + __shfl_down_sync(FULL, bs[6], 1);
    const R down = bs[4] + __shfl_down_sync(FULL, bs[7], 1) + __shfl_up_sync(FULL, bs[8], 1);
    if (rr >= 1 && col_out && fl_prev) phi_out[(size_t)(j0 + rr - 1) * nx + x] = acc_prev + down;
    acc_prev = (up_prev + mid) + bb;
    up_prev = up;
    fl_prev = fl;

    // rotate the pipeline registers
    w_cur = w_next; w_next = w_nn;
#pragma unroll
    for (int q = 0; q < 9; q++) ncur[q] = nnext[q];
#pragma unroll
    for (int i = 0; i < 3; i++) { pS[i] = pC[i]; pC[i] = pN[i]; pN[i] = pNN[i]; }
    bS = bC; bC = bN; bN = bNN;
  }
}

template <typename R>
void launch_fused_warp(const Consts<R>& C, const uint16_t* cl16, const R* Nsrc, R* Ndst, R* Bdst,
                       const R* phi_in, R* phi_out, cudaStream_t st) {
  constexpr int WARPS = 4;
  constexpr int MINB = sizeof(R) == 8 ? 4 : 5;
  const int nwx = (C.nx + 29) / 30;
  const int gx = (nwx + WARPS - 1) / WARPS;
  // rows per warp march: long marches amortise the two halo rows; small grids need enough CTAs
  int TY = 64;
  while (TY > 8 && (long long)gx * ((C.ny + TY - 1) / TY) < 148 * 8) TY >>= 1;
  const dim3 grid((unsigned)gx, (unsigned)((C.ny + TY - 1) / TY), 1);
  if (Bdst)
    k_fused_warp<R, WARPS, MINB, true><<<grid, 32 * WARPS, 0, st>>>(C, cl16, Nsrc, Ndst, Bdst, phi_in, phi_out, TY);
  else
    k_fused_warp<R, WARPS, MINB, false><<<grid, 32 * WARPS, 0, st>>>(C, cl16, Nsrc, Ndst, Bdst, phi_in, phi_out, TY);
}

}  // namespace lbm

// lbm_fused.cuh — FUSED schedule: one kernel per time step does pull-stream + collide + segregation
// AND produces phi(t+1) = sum_i B_i(x, t+1) (A13, :311) from the post-collision B_i* of the node's
// neighbours, which never leave the SM: B is not part of the HBM state at all.
//
// Why: the collision reads B only through phi = sum_i B_i, and B_i* is a local function of
// (phi, N*, p, n_phi) (Eq. A12, :307).  So the only thing the next step needs from B* is its
// streamed sum.  Per fluid-node update the kernel moves 9 N reads + 9 N writes + phi read/write
// + 1 class byte (20 values + 1 B) instead of the canonical 36 values.
//
// How: a CTA of TX threads owns TX-2 output columns and marches over TY rows (+1 halo row at each
// end).  Row by row every thread collides its node (halo columns/rows redundantly: their N* is
// not written) and parks the 9 B_i* in a 4-slot ring of rows in shared memory; once row r+1 is
// parked, phi(t+1) of row r is the pull-sum over the ring (bounce-back links read the node's own
// opposite B*).  One __syncthreads per row (4 slots make the second one unnecessary).
#pragma once
#include "lbm_kernels.cuh"

namespace lbm {

template <typename R, int TX, bool WRITE_B>
__global__ void __launch_bounds__(TX) k_fused_step(const Consts<R> C, const uint8_t* __restrict__ cls,
                                                   const uint8_t* __restrict__ links,
                                                   const R* __restrict__ Nsrc, R* __restrict__ Ndst,
                                                   R* __restrict__ Bdst, const R* __restrict__ phi_in,
                                                   R* __restrict__ phi_out, int TY) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  R(*sB)[9][TX] = reinterpret_cast<R(*)[9][TX]>(smem_raw);   // [4][9][TX]

  const int nx = C.nx, ny = C.ny;
  const size_t n = C.ps;   // plane stride
  const int tx = threadIdx.x;
  const int x0 = blockIdx.x * (TX - 2);
  const int j0 = blockIdx.y * TY;
  const int rows = min(TY, ny - j0);
  const int lx = x0 - 1 + tx;                                  // logical column, may be -1 or nx
  const bool col_active = lx <= min(x0 + TX - 2, nx);          // output columns + one halo each side
  const bool col_out = tx >= 1 && tx <= TX - 2 && lx < nx;
  int x = lx;
  if (x < 0) x += nx;
  if (x >= nx) x -= nx;
  if (!col_active) x = 0;
  const int xm = (x == 0) ? nx - 1 : x - 1, xp = (x == nx - 1) ? 0 : x + 1;

  unsigned c_prev = 3, lk_prev = 0;
  for (int rr = -1; rr <= rows; rr++) {
    int r = j0 + rr;
    if (r < 0) r += ny;
    if (r >= ny) r -= ny;
    const int slot = (rr + 1) & 3;
    unsigned c = 3, lk = 0;
    if (col_active) {
      const int r0 = r * nx;
      const int k = r0 + x;
      c = cls[k];
      if (c < 2) {
        lk = (c == 1) ? links[k] : 0u;
        const int rm = ((r == 0) ? ny - 1 : r - 1) * nx, rp = ((r == ny - 1) ? 0 : r + 1) * nx;
        R nn[9], ph[9], ns[9], bs[9];
        ph[0] = phi_in[k];
        ph[1] = phi_in[r0 + xp]; ph[3] = phi_in[r0 + xm];
        ph[2] = phi_in[rp + x];  ph[4] = phi_in[rm + x];
        ph[5] = phi_in[rp + xp]; ph[6] = phi_in[rp + xm];
        ph[7] = phi_in[rm + xm]; ph[8] = phi_in[rm + xp];
        nn[0] = Nsrc[k];
        if (lk == 0) {
          nn[1] = Nsrc[1 * n + r0 + xm]; nn[2] = Nsrc[2 * n + rm + x];
          nn[3] = Nsrc[3 * n + r0 + xp]; nn[4] = Nsrc[4 * n + rp + x];
          nn[5] = Nsrc[5 * n + rm + xm]; nn[6] = Nsrc[6 * n + rm + xp];
          nn[7] = Nsrc[7 * n + rp + xp]; nn[8] = Nsrc[8 * n + rp + xm];
        } else {
          const int src[9] = {k, r0 + xm, rm + x, r0 + xp, rp + x, rm + xm, rm + xp, rp + xp, rp + xm};
#pragma unroll
          for (int q = 1; q < 9; q++)
            nn[q] = ((lk >> (q - 1)) & 1u) ? Nsrc[opp(q) * n + k] : Nsrc[q * n + src[q]];
        }
        node_update<R, true>(C, nn, ph, ns, bs, nullptr);
        if (col_out && rr >= 0 && rr < rows) {
#pragma unroll
          for (int q = 0; q < 9; q++) Ndst[q * n + k] = ns[q];
          if (WRITE_B) {
#pragma unroll
            for (int q = 0; q < 9; q++) Bdst[q * n + k] = bs[q];
          }
        }
#pragma unroll
        for (int q = 0; q < 9; q++) sB[slot][q][tx] = bs[q];
      }
    }
    __syncthreads();
    if (rr >= 1 && col_out && c_prev < 2) {
      // phi(t+1) of row rr-1: pull-sum of B* (A13 after A16-A17), oracle's summation order
      const int cxq[9] = {0, 1, 0, -1, 0, 1, -1, -1, 1}, cyq[9] = {0, 0, 1, 0, -1, 1, 1, -1, -1};
      const int s0 = rr & 3;   // slot of row rr-1
      R s = sB[s0][0][tx];
#pragma unroll
      for (int q = 1; q < 9; q++) {
        const R v = ((lk_prev >> (q - 1)) & 1u) ? sB[s0][opp(q)][tx]
                                                : sB[(rr - cyq[q]) & 3][q][tx - cxq[q]];
        s += v;
      }
      int rprev = j0 + rr - 1;   // rr-1 in [0, rows): never wraps
      phi_out[(size_t)rprev * nx + x] = s;
    }
    c_prev = c;
    lk_prev = lk;
  }
}

template <typename R>
void launch_fused_step(const Consts<R>& C, const uint8_t* cls, const uint8_t* links, const R* Nsrc,
                       R* Ndst, R* Bdst, const R* phi_in, R* phi_out, cudaStream_t st) {
  constexpr int TX = 128;
  const int gx = (C.nx + TX - 3) / (TX - 2);
  // rows per CTA: long marches amortise the two halo rows; short ones give small grids enough CTAs
  int TY = 64;
  while (TY > 8 && (long long)gx * ((C.ny + TY - 1) / TY) < 148 * 8) TY >>= 1;
  const dim3 grid((unsigned)gx, (unsigned)((C.ny + TY - 1) / TY), 1);
  const size_t smem = 4 * 9 * TX * sizeof(R);
  if (Bdst)
    k_fused_step<R, TX, true><<<grid, TX, smem, st>>>(C, cls, links, Nsrc, Ndst, Bdst, phi_in, phi_out, TY);
  else
    k_fused_step<R, TX, false><<<grid, TX, smem, st>>>(C, cls, links, Nsrc, Ndst, Bdst, phi_in, phi_out, TY);
}

}  // namespace lbm

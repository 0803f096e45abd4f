// lbm_sparse.cuh — SPARSE schedule: the fused pull-stream + collide + segregation + phi(t+1) kernel with
// lanes mapped to FLUID GROUPS instead of columns.
//
// State: group-compacted planes as under PACK (lbm_kernels.cuh: k_pair_mask, ptab) — only the aligned groups of NL
// x-adjacent nodes that hold a fluid node are stored, row after row — but group-major: the nine 16-byte vectors of
// a group are contiguous, so a row of a strip is ONE contiguous run.  What changes is who works on what:
//
//   * one persistent CTA per SM owns "marches": a strip of at most SP_S groups, a run of rows (lbm_create cuts the
//     work into marches of equal weight: one wave, no tail).
//   * SP_K loader warps (rows split by parity) bring every row on chip with three 1-D bulk copies (cp.async.bulk
//     -> UBLKCP, complete_tx on the row slot's mbarrier): the row's run of the compact planes, its group metadata,
//     its dense phi row.  Rows live in a shared-memory ring sized in entries, not rows.
//   * the SP_W consumer warps take "passes" from an atomic counter: 32 consecutive ENTRIES of the row-major
//     sequence of the strip's active groups (a pass may span several rows; 30 outputs + one helper lane per
//     side).  Every lane therefore holds a group with a fluid node: no issue slot is spent on solid lanes.
//   * propagation (A16-A17) is a gather from the ring: same-row neighbours are the adjacent entries, the
//     groups above / below are found by popcount on the row's group mask.  Half-way bounce-back (R12)
//     selects the node's own opposite population, as in the PAIR kernel.
//   * phi(x, t+1) = sum_q B_q*(x - c_q, t) (A13): every output lane writes the three partial sums its row sends to
//     the rows above / at / below (x-moves by warp shuffle between x-adjacent lanes, direct stores into the columns
//     of a neighbour group without a lane) into per-entry slots of the TARGET row, each address written by exactly
//     one lane; SP_K finaliser warps add the three once all consumers are past the row and store phi(t+1).  No
//     atomics on data: results are run-to-run identical.
//   * synchronisation: one mbarrier per row slot (loader -> consumers, TMA transaction bytes), one monotone "no
//     claim on the rows below R" counter per consumer warp (consumers -> finalisers) and one monotone "retired"
//     counter per row class (finaliser -> loader).  No __syncthreads inside a march; every wait is bounded (a
//     schedule bug traps after ~4 s instead of hanging the device).
//   Measured (profiles/r2_sparse.txt): correct, but slower than PACK — the gather costs the instructions the fuller
//   lanes save, and the ring leaves under two rows of look-ahead in 227 KB.  PACK stays the AUTO schedule.
#pragma once
#include "lbm_pair.cuh"

namespace lbm {

#ifndef LBM_SP_WARPS
#define LBM_SP_WARPS 12
#endif
#ifndef LBM_SP_CAP
#define LBM_SP_CAP 928
#endif
constexpr int SP_S = 126;                 // body groups of a strip; S + 2 halo groups = 128 mask bits
constexpr int SP_W = LBM_SP_WARPS;        // consumer warps
constexpr int SP_NR = 16;                 // row slots (phi rows, row info, full barriers)
constexpr int SP_CAP = LBM_SP_CAP;        // entries of the population ring
constexpr int SP_TYMAX = 512;             // rows of a march
constexpr int SP_MINPOS = 8;              // a row takes at least this many positions of the pass sequence, so
                                          // that a pass of 32 positions spans at most 5 rows
constexpr int SP_K = 2;                   // loader warps and finaliser warps; helper k serves rows R = k (mod K)
constexpr int SP_CAPK = SP_CAP / SP_K;    // every loader fills its own part of the ring
constexpr int SP_THREADS = 32 * (SP_W + 2 * SP_K);
static_assert(SP_NR % SP_K == 0 && SP_CAP % (2 * SP_K) == 0, "helper classes");

// per (strip, row) descriptor, built once by k_sp_desc
struct __align__(16) SpDesc {
  uint32_t ci0;       // compact index of the strip's first body group in this row (insertion point if absent)
  uint32_t ciL, ciR;  // compact indices of the halo groups left / right of the body (valid if hl / hr)
  uint16_t a;         // active body groups
  uint8_t hl, hr;     // halo group active
  uint32_t bits[4];   // bit c + 1 set <=> group c of the strip holds a fluid node, c = -1 .. S
  uint2 metaL, metaR; // metadata of the halo groups
  uint8_t pre[4];     // popcount of the words below
  uint32_t pad[3];
};
static_assert(sizeof(SpDesc) == 64, "descriptor layout");

// per compact group: x = column of the group | fluid bits << 16 | left neighbour group active << 20 |
// right neighbour group active << 21; y = bounce-back link byte of each node
struct SpMarch { int strip, j0, rows, pad; };

struct SpRow {        // shared-memory copy of what the consumers need of a row
  uint32_t off;       // ring index of entry 0
  uint32_t ci0;       // compact index of the first body entry
  uint32_t n;         // entries: hl + a + hr
  uint32_t hlr;       // bit 0: left halo entry present, bit 1: right halo entry present
  uint32_t bits[4];
  uint32_t pre;       // four prefix bytes
  uint32_t jrow;      // grid row
  uint2 metaL, metaR;
};

template <typename V>
struct SpSmem {
  V N[SP_CAP][9];       // group-major, like the compact planes in HBM: a row is one contiguous run
  uint2 meta[SP_CAP];
  V phi[SP_NR][SP_S + 4];
  V A[3][SP_CAP];       // per entry: what the rows above / at / below contribute to its phi(t+1)
  SpRow row[SP_NR];
  uint32_t T[SP_TYMAX + 4];
  unsigned long long full[SP_NR];
  int rstart[SP_NR];
  int done[32];
  int ret_row[SP_K];    // class k: rows R = k (mod K) below ret_row[k] are retired
  int next_pass;        // pass counter of the march
  int pad[3 - SP_K % 4];
};

// ---- mbarrier / bulk-copy / ordered shared-memory access ----
__device__ __forceinline__ void mbar_init(unsigned a, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(a), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_inval(unsigned a) {
  asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(a) : "memory");
}
__device__ __forceinline__ void mbar_arrive_tx(unsigned a, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(a), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_test(unsigned a, unsigned parity) {
  unsigned ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(a), "r"(parity)
      : "memory");
  return ok != 0;
}
// a wait that cannot hang the device: a schedule bug traps instead (reported as a CUDA error by lbm_step)
__device__ __forceinline__ void mbar_wait(unsigned a, unsigned parity) {
  if (mbar_test(a, parity)) return;
  const long long t0 = clock64();
  while (!mbar_test(a, parity))
    if (clock64() - t0 > 8000000000LL) __trap();
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned mbar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(mbar)
               : "memory");
}
__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.cta.shared.s32 %0, [%1];" : "=r"(v) : "r"((unsigned)__cvta_generic_to_shared(p)) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
  asm volatile("st.release.cta.shared.s32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(p)), "r"(v) : "memory");
}
__device__ __forceinline__ void wait_counter(const int* p, int target) {
  if (ld_acquire(p) >= target) return;
  const long long t0 = clock64();
  while (ld_acquire(p) < target) {
    __nanosleep(64);
    if (clock64() - t0 > 8000000000LL) __trap();
  }
}

// a lane's vector with one scalar shifted in from the left / right neighbour node
template <typename V>
__device__ __forceinline__ V shift_in_left(V own, typename LaneOf<V>::R s) {
  using L = LaneOf<V>;
  typename L::R x[L::NL], y[L::NL];
  L::unpack(own, x);
  y[0] = s;
#pragma unroll
  for (int c = 1; c < L::NL; c++) y[c] = x[c - 1];
  return L::pack(y);
}
template <typename V>
__device__ __forceinline__ V shift_in_right(V own, typename LaneOf<V>::R s) {
  using L = LaneOf<V>;
  typename L::R x[L::NL], y[L::NL];
  L::unpack(own, x);
#pragma unroll
  for (int c = 0; c < L::NL - 1; c++) y[c] = x[c + 1];
  y[L::NL - 1] = s;
  return L::pack(y);
}
template <typename V>
__device__ __forceinline__ typename LaneOf<V>::R first_of(V v) {
  typename LaneOf<V>::R x[LaneOf<V>::NL];
  LaneOf<V>::unpack(v, x);
  return x[0];
}
template <typename V>
__device__ __forceinline__ typename LaneOf<V>::R last_of(V v) {
  typename LaneOf<V>::R x[LaneOf<V>::NL];
  LaneOf<V>::unpack(v, x);
  return x[LaneOf<V>::NL - 1];
}

// entry index, within its row, of group c (c = -1 .. S): the number of active groups with a smaller column
__device__ __forceinline__ int sp_rank(const SpRow& r, int c, unsigned* bit) {
  const unsigned b = (unsigned)(c + 1);
  const unsigned w = r.bits[b >> 5];
  *bit = (w >> (b & 31u)) & 1u;
  return (int)((r.pre >> (8u * (b >> 5))) & 0xffu) + __popc(w & ((1u << (b & 31u)) - 1u));
}

template <typename V, bool WRITE_B>
__global__ void __launch_bounds__(SP_THREADS, 1)
    k_fused_sparse(const Consts<typename LaneOf<V>::R> C, const typename LaneOf<V>::R* __restrict__ Nsrc,
                   typename LaneOf<V>::R* __restrict__ Ndst, typename LaneOf<V>::R* __restrict__ Bdst,
                   const typename LaneOf<V>::R* __restrict__ phi_in, typename LaneOf<V>::R* __restrict__ phi_out,
                   const SpDesc* __restrict__ desc, const uint16_t* __restrict__ cnt, const uint2* __restrict__ gmeta,
                   const SpMarch* __restrict__ marches, const int* __restrict__ cta_first, int sw) {
  using L = LaneOf<V>;
  using R = typename L::R;
  constexpr int NL = L::NL;
  constexpr unsigned FULL = 0xffffffffu;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SpSmem<V>& S = *reinterpret_cast<SpSmem<V>*>(smem_raw);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nx = C.nx, ny = C.ny;
  const int ng = nx / NL;                                      // groups per row
  const unsigned psBd = (unsigned)C.ps * (unsigned)sizeof(R);  // dense plane stride in bytes (B planes)
  const V zero = splat<V>(R(0));

  // stale ring entries are read (and discarded, or multiplied by a zero mask): they must be finite
  for (int k = tid; k < 9 * SP_CAP; k += SP_THREADS) (&S.N[0][0])[k] = zero;
  for (int k = tid; k < SP_NR * (SP_S + 4); k += SP_THREADS) (&S.phi[0][0])[k] = zero;
  for (int k = tid; k < SP_CAP; k += SP_THREADS) S.meta[k] = make_uint2(0u, 0u);

  for (int mi = cta_first[blockIdx.x]; mi < cta_first[blockIdx.x + 1]; mi++) {
    const SpMarch mar = marches[mi];
    const int c0 = mar.strip * sw;                             // first body group of the strip (sw <= SP_S groups wide)
    const int seff = min(sw, ng - c0);                         // body groups of this strip
    const int TY = mar.rows;
    const int nR = TY + 4;                                     // ring rows R = 0 .. TY+3 <-> grid rows j0-2 ..
    const SpDesc* sdesc = desc + (size_t)mar.strip * ny;
    const uint16_t* scnt = cnt + (size_t)mar.strip * ny;
    auto grid_row = [&](int Rr) -> int {
      int j = mar.j0 - 2 + Rr;
      j %= ny;
      return j < 0 ? j + ny : j;
    };
    __syncthreads();   // previous march finished; zero fill visible
    // ---- pass sequence: T[k] = positions of processed rows R = 1 .. k (k = 0 .. TY+2) ----
    if (warp == 0) {
      unsigned run = 0;
      for (int base = 0; base < TY + 2; base += 32) {
        const int k = base + lane;
        unsigned v = 0;
        if (k < TY + 2) v = max((unsigned)scnt[grid_row(k + 1)], (unsigned)SP_MINPOS);
        unsigned s = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          const unsigned t = __shfl_up_sync(FULL, s, d);
          if (lane >= d) s += t;
        }
        if (k < TY + 2) S.T[k + 1] = run + s;
        run += __shfl_sync(FULL, s, 31);
      }
      if (lane == 0) S.T[0] = 0;
    }
    if (tid == 32) {
      for (int k = 0; k < SP_NR; k++) mbar_init((unsigned)__cvta_generic_to_shared(&S.full[k]), 1);
      for (int k = 0; k < SP_K; k++) S.ret_row[k] = k;
      S.next_pass = 0;
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid < 32) S.done[tid] = 0;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    const int P = (int)S.T[TY + 2];
    const int NP = (P + 29) / 30;

    if (warp >= SP_W && warp < SP_W + SP_K) {
      // ===================== loader warp k: rows R = k (mod K) -> its part of the ring (TMA) =====================
      const int kc = warp - SP_W;
      const int rbase = kc * SP_CAPK;
      int head = 0, Rret = kc;
      int j = grid_row(kc);
      int jn = j + SP_K >= ny ? j + SP_K - ny : j + SP_K;
      SpDesc dn = sdesc[j];
      for (int Rload = kc; Rload < nR; Rload += SP_K) {
        const SpDesc d = dn;
        const int jcur = j;
        j = jn;
        jn = j + SP_K >= ny ? j + SP_K - ny : j + SP_K;
        if (Rload + SP_K < nR) dn = sdesc[j];
        const int n = (int)d.hl + (int)d.a + (int)d.hr;
        const int need = (n + 8) & ~1;
        // wait for a row slot and for ring space (the rows of a class are retired in order by its finaliser)
        int start = -1;
        long long t0 = 0;
        for (;;) {
          if (Rload - Rret < SP_NR) {
            if (Rret == Rload) { start = 0; }
            else {
              const int tail = S.rstart[Rret & (SP_NR - 1)];
              if (head >= tail) {
                if (head + need <= SP_CAPK) start = head;
                else if (need < tail) start = 0;
              } else if (head + need < tail) start = head;
            }
          }
          if (start >= 0) break;
          const int r = ld_acquire(&S.ret_row[kc]);
          if (r == Rret) {
            __nanosleep(32);
            if (t0 == 0) t0 = clock64();
            else if (clock64() - t0 > 8000000000LL) __trap();
          }
          Rret = r;
        }
        const int slot = Rload & (SP_NR - 1);
        const bool contL = d.hl && d.ciL + 1u == d.ci0;
        const bool contR = d.hr && d.ciR == d.ci0 + d.a;
        const unsigned runCi = d.ci0 - (contL ? 1u : 0u);
        const int runLen = (int)d.a + (contL ? 1 : 0) + (contR ? 1 : 0);
        int off0 = rbase + start + 2;
        int runRing = off0 + ((d.hl && !contL) ? 1 : 0);
        if ((runRing ^ (int)runCi) & 1) { off0++; runRing++; }
        head = start + need;
        // nobody has written the row's phi(t+1) contributions yet: the sums from above and below start at zero
        for (int e = lane; e < n; e += 32) { S.A[0][off0 + e] = zero; S.A[2][off0 + e] = zero; }
        __syncwarp();
        if (lane == 0) {
          SpRow& rw = S.row[slot];
          rw.off = (uint32_t)off0; rw.ci0 = d.ci0; rw.n = (uint32_t)n; rw.hlr = (uint32_t)d.hl | ((uint32_t)d.hr << 1);
          rw.bits[0] = d.bits[0]; rw.bits[1] = d.bits[1]; rw.bits[2] = d.bits[2]; rw.bits[3] = d.bits[3];
          rw.pre = (uint32_t)d.pre[0] | ((uint32_t)d.pre[1] << 8) | ((uint32_t)d.pre[2] << 16) | ((uint32_t)d.pre[3] << 24);
          rw.jrow = (uint32_t)jcur; rw.metaL = d.metaL; rw.metaR = d.metaR;
          S.rstart[slot] = start;
          // one elected lane issues every bulk copy of the row (uniform datapath, no per-lane serialisation)
          const unsigned mb = (unsigned)__cvta_generic_to_shared(&S.full[slot]);
          const bool wl = d.hl && !contL, wr = d.hr && !contR;
          const unsigned mStart = d.ci0 & ~1u, mEnd = (d.ci0 + d.a + 1u) & ~1u;
          const unsigned metaBytes = d.a ? (mEnd - mStart) * 8u : 0u;
          const unsigned phiBytes = (unsigned)(seff + 4) * 16u;
          const unsigned bytes = 9u * 16u * ((unsigned)runLen + (wl ? 1u : 0u) + (wr ? 1u : 0u)) + metaBytes + phiBytes;
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          mbar_arrive_tx(mb, bytes);
          const char* src = reinterpret_cast<const char*>(Nsrc);   // group ci: 9 vectors of 16 bytes at ci * 144
          if (runLen > 0)
            bulk_g2s((unsigned)__cvta_generic_to_shared(&S.N[runRing][0]), src + (size_t)runCi * 144u, (unsigned)runLen * 144u, mb);
          if (wl) bulk_g2s((unsigned)__cvta_generic_to_shared(&S.N[off0][0]), src + (size_t)d.ciL * 144u, 144u, mb);
          if (wr) bulk_g2s((unsigned)__cvta_generic_to_shared(&S.N[off0 + n - 1][0]), src + (size_t)d.ciR * 144u, 144u, mb);
          if (metaBytes)
            bulk_g2s((unsigned)__cvta_generic_to_shared(&S.meta[off0 + (int)d.hl - (int)(d.ci0 & 1u)]), gmeta + mStart, metaBytes, mb);
          // phi: logical groups c0-2 .. c0+seff+1 of the periodic row, cut where they wrap
          int g = c0 - 2, left = seff + 4, dsti = 0;
          const R* prow = phi_in + (size_t)jcur * (size_t)nx;
          while (left > 0) {
            int gw = g % ng;
            if (gw < 0) gw += ng;
            const int len = min(left, ng - gw);
            bulk_g2s((unsigned)__cvta_generic_to_shared(&S.phi[slot][dsti]), prow + (size_t)gw * NL, (unsigned)len * 16u, mb);
            g += len; left -= len; dsti += len;
          }
        }
        __syncwarp();
      }
    } else if (warp >= SP_W + SP_K) {
      // ==== finaliser warp k: retires the rows R = k (mod K) in order, stores phi(t+1), recycles the sum buffers ====
      const int kc = warp - SP_W - SP_K;
      for (int Rret = kc; Rret < nR; Rret += SP_K) {
        const int want = min(Rret + 1, TY + 2);
        long long t0 = 0;
        for (;;) {   // every consumer past row Rret + 1
          int mind = lane < SP_W ? ld_acquire(&S.done[lane]) : 0x7fffffff;
#pragma unroll
          for (int dd = 16; dd >= 1; dd >>= 1) mind = min(mind, __shfl_xor_sync(FULL, mind, dd));
          if (mind >= want) break;
          __nanosleep(32);
          if (t0 == 0) t0 = clock64();
          else if (clock64() - t0 > 8000000000LL) __trap();
        }
        if (Rret >= 2 && Rret <= TY + 1) {   // phi(t+1) of the row: the three partial sums of its entries, on fluid nodes
          const SpRow& rw = S.row[Rret & (SP_NR - 1)];
          const int hlF = (int)(rw.hlr & 1u);
          const int nb = (int)rw.n - hlF - (int)(rw.hlr >> 1);   // body entries
          R* prow = phi_out + (size_t)rw.jrow * (size_t)nx + (size_t)c0 * NL;
          const int x0 = (int)rw.off + hlF;
          for (int e = lane; e < nb; e += 32) {
            const uint2 mt = S.meta[x0 + e];
            const int c = (int)(mt.x & 0xffffu) - c0;
            const V v = (S.A[0][x0 + e] + S.A[1][x0 + e]) + S.A[2][x0 + e];
            const unsigned fl = (mt.x >> 16) & 0xfu;
            R* dst = prow + c * NL;
            if (fl == (1u << NL) - 1u) store_vec<V>(dst, v);
            else {
              R x[NL];
              L::unpack(v, x);
#pragma unroll
              for (int k = 0; k < NL; k++)
                if ((fl >> k) & 1u) dst[k] = x[k];
            }
          }
        }
        __syncwarp();
        if (lane == 0) st_release(&S.ret_row[kc], Rret + SP_K);
      }
    } else {
      // ===================================== consumer warps =====================================
      int waitedR = -1;   // full[] observed for ring rows <= waitedR
      auto row_scan = [&](int from, int s) -> int {   // processed row R >= from holding position s: T[R-1] <= s < T[R]
        int r = from;
        while ((int)S.T[r] <= s) r++;
        return r;
      };
      // passes are handed out in order to whichever warp is free: the passes in flight stay consecutive, so the
      // rows they span (which the ring must hold) stay few even when warps fall behind one another
      int Rprev = 1;
      for (;;) {
        int p = 0;
        if (lane == 0) p = atomicAdd(&S.next_pass, 1);
        p = __shfl_sync(FULL, p, 0);
        if (p >= NP) break;
        const int s0 = 30 * p - 1;
        const int R0 = row_scan(Rprev, max(s0, 0));
        Rprev = R0;
        if (lane == 0) st_release(&S.done[warp], R0 - 1);   // no claim on the rows before this pass any more
        const int s = s0 + lane;
        int Rl = R0;
#pragma unroll
        for (int k = 0; k < 5; k++)
          if (R0 + k <= TY + 1 && s >= (int)S.T[R0 + k]) Rl = R0 + k + 1;
        const bool pos_ok = s >= 0 && s < P;
        const int e = s - (int)S.T[Rl - 1];
        const int Rmax = __shfl_sync(FULL, Rl, 31);
        // rows R0-1 .. Rmax+1 must have landed
        while (waitedR < Rmax + 1) {
          waitedR++;
          mbar_wait((unsigned)__cvta_generic_to_shared(&S.full[waitedR & (SP_NR - 1)]), (unsigned)(waitedR / SP_NR) & 1u);
        }
        const SpRow& rw = S.row[Rl & (SP_NR - 1)];
        const bool active = pos_ok && e < (int)rw.n;
        const bool outl = active && lane >= 1 && lane <= 30;
        uint2 mt = make_uint2(0u, 0u);
        int c = 0;
        bool body = false;
        if (active) {
          if (e == 0 && (rw.hlr & 1u)) { mt = rw.metaL; c = -1; }
          else if (e == (int)rw.n - 1 && (rw.hlr & 2u)) { mt = rw.metaR; c = seff; }
          else { mt = S.meta[rw.off + e]; c = (int)(mt.x & 0xffffu) - c0; body = true; }
        }
        bool fl[NL];
        unsigned lk[NL];
        bool any_fl = false, all_fl = true;
        unsigned lk_any = 0u;
#pragma unroll
        for (int k = 0; k < NL; k++) {
          fl[k] = active && ((mt.x >> (16 + k)) & 1u);
          lk[k] = fl[k] ? ((mt.y >> (8 * k)) & 0xffu) : 0u;
          any_fl |= fl[k]; all_fl &= fl[k]; lk_any |= lk[k];
        }
        const bool adjL = active && ((mt.x >> 20) & 1u) && e > 0;
        const bool adjR = active && ((mt.x >> 21) & 1u) && e + 1 < (int)rw.n;

        V bs[9];
        V bb = zero;
        int eu = 0, ed = 0, eo = 0;          // ring entries of group c in the rows above / below, and of the lane's own group
        unsigned bU = 0, bD = 0;             // group c holds a fluid node in the row above / below
        unsigned nbU = 0, nbD = 0;           // bit 0 / 1: group c-1 / c+1 holds a fluid node in the row above (nbU) / below (nbD)
        if (active) {
          const SpRow& ru = S.row[(Rl - 1) & (SP_NR - 1)];
          const SpRow& rd = S.row[(Rl + 1) & (SP_NR - 1)];
          eu = (int)ru.off + sp_rank(ru, c, &bU);
          ed = (int)rd.off + sp_rank(rd, c, &bD);
          eo = (int)rw.off + e;
          if (c >= 1) {
            nbU |= (ru.bits[c >> 5] >> (c & 31)) & 1u;
            nbD |= (rd.bits[c >> 5] >> (c & 31)) & 1u;
          }
          if (c + 1 < seff) {
            nbU |= ((ru.bits[(c + 2) >> 5] >> ((c + 2) & 31)) & 1u) << 1;
            nbD |= ((rd.bits[(c + 2) >> 5] >> ((c + 2) & 31)) & 1u) << 1;
          }
          // own-position populations of the node's row, and the neighbours' (propagation A16-A17)
          const V o0 = S.N[eo][0], o1 = S.N[eo][1], o2 = S.N[eo][2], o3 = S.N[eo][3], o4 = S.N[eo][4],
                  o5 = S.N[eo][5], o6 = S.N[eo][6], o7 = S.N[eo][7], o8 = S.N[eo][8];
          V nn[9];
          nn[0] = o0;
          nn[1] = shift_in_left<V>(o1, reinterpret_cast<const R*>(&S.N[eo - 1][1])[NL - 1]);
          nn[3] = shift_in_right<V>(o3, reinterpret_cast<const R*>(&S.N[eo + 1][3])[0]);
          nn[2] = S.N[eu][2];
          nn[5] = shift_in_left<V>(S.N[eu][5], reinterpret_cast<const R*>(&S.N[eu - 1][5])[NL - 1]);
          nn[6] = shift_in_right<V>(S.N[eu][6], reinterpret_cast<const R*>(&S.N[eu + (int)bU][6])[0]);
          nn[4] = S.N[ed][4];
          nn[7] = shift_in_right<V>(S.N[ed][7], reinterpret_cast<const R*>(&S.N[ed + (int)bD][7])[0]);
          nn[8] = shift_in_left<V>(S.N[ed][8], reinterpret_cast<const R*>(&S.N[ed - 1][8])[NL - 1]);
          if (lk_any) {   // half-way bounce-back (R12): the node's own opposite population
            const V own[9] = {o0, o1, o2, o3, o4, o5, o6, o7, o8};
#pragma unroll
            for (int q = 1; q < 9; q++) {
              R a[NL], o[NL];
              L::unpack(nn[q], a);
              L::unpack(own[opp(q)], o);
#pragma unroll
              for (int k = 0; k < NL; k++)
                if ((lk[k] >> (q - 1)) & 1u) a[k] = o[k];
              nn[q] = L::pack(a);
            }
          }
          // phi stencil (R8): nodes c*NL - 1 .. c*NL + NL of the three rows; row buffers start at group -2
          const R* pu = reinterpret_cast<const R*>(&S.phi[(Rl - 1) & (SP_NR - 1)][c + 2]);
          const R* pc = reinterpret_cast<const R*>(&S.phi[Rl & (SP_NR - 1)][c + 2]);
          const R* pd = reinterpret_cast<const R*>(&S.phi[(Rl + 1) & (SP_NR - 1)][c + 2]);
          const V pS = *reinterpret_cast<const V*>(pu), pC = *reinterpret_cast<const V*>(pc), pN = *reinterpret_cast<const V*>(pd);
          const V ph[9] = {pC, shift_in_right<V>(pC, pc[NL]), pN, shift_in_left<V>(pC, pc[-1]), pS,
                           shift_in_right<V>(pN, pd[NL]), shift_in_left<V>(pN, pd[-1]),
                           shift_in_left<V>(pS, pu[-1]), shift_in_right<V>(pS, pu[NL])};
          V ns[9];
          collide_lane<V>(C, nn, ph, fl, all_fl, ns, bs);
          if (outl && body && Rl >= 2 && Rl <= TY + 1) {
            const unsigned ci = rw.ci0 + (unsigned)(e - (int)(rw.hlr & 1u));
            char* dst = reinterpret_cast<char*>(Ndst) + (size_t)ci * 144u;
#pragma unroll
            for (int q = 0; q < 9; q++) store_vec<V>(dst + 16 * q, ns[q]);
            if (WRITE_B) {
              char* dstB = reinterpret_cast<char*>(Bdst + ((size_t)rw.jrow * (size_t)nx + (size_t)(c0 + c) * NL));
#pragma unroll
              for (int q = 0; q < 9; q++) *reinterpret_cast<V*>(dstB + (size_t)psBd * (unsigned)q) = bs[q];
            }
          }
          if (lk_any) {   // link q hands the node its own B_opp(q)* back
            R b[NL];
#pragma unroll
            for (int k = 0; k < NL; k++) b[k] = R(0);
#pragma unroll
            for (int q = 1; q < 9; q++) {
              R o[NL];
              L::unpack(bs[opp(q)], o);
#pragma unroll
              for (int k = 0; k < NL; k++)
                if ((lk[k] >> (q - 1)) & 1u) b[k] += o[k];
            }
            bb = L::pack(b);
          }
        } else {
#pragma unroll
          for (int q = 0; q < 9; q++) bs[q] = zero;
        }
        // contributions of this group's row to phi(t+1) of the rows above (U), at (M) and below (D): the B*
        // that move in x cross to the x-adjacent lane by shuffle; a neighbour group without a fluid node has
        // no lane, so the node next to it gets the spill by a direct store
        const R z = R(0);
        const R l1 = __shfl_up_sync(FULL, last_of<V>(bs[1]), 1), l5 = __shfl_up_sync(FULL, last_of<V>(bs[5]), 1),
                l8 = __shfl_up_sync(FULL, last_of<V>(bs[8]), 1);
        const R r3 = __shfl_down_sync(FULL, first_of<V>(bs[3]), 1), r6 = __shfl_down_sync(FULL, first_of<V>(bs[6]), 1),
                r7 = __shfl_down_sync(FULL, first_of<V>(bs[7]), 1);
        if (outl) {
          if (body) {
            const V mid = (bs[0] + shift_in_left<V>(bs[1], adjL ? l1 : z)) + shift_in_right<V>(bs[3], adjR ? r3 : z);
            const V upw = (bs[2] + shift_in_left<V>(bs[5], adjL ? l5 : z)) + shift_in_right<V>(bs[6], adjR ? r6 : z);
            const V dwn = (bs[4] + shift_in_right<V>(bs[7], adjR ? r7 : z)) + shift_in_left<V>(bs[8], adjL ? l8 : z);
            S.A[1][eo] = mid + bb;
            if (bD) S.A[0][ed] = upw;     // the group above me in the next row: what arrives from below it
            if (bU) S.A[2][eu] = dwn;
          }
          // a body group next to mine without a fluid node in this row has no lane: its columns in the rows
          // above / below still receive the B* that leave my edge node diagonally
          if (c + 1 < seff && !(((rw.bits[(c + 2) >> 5]) >> ((c + 2) & 31)) & 1u)) {
            if (nbD & 2u) reinterpret_cast<R*>(&S.A[0][ed + (int)bD])[0] = last_of<V>(bs[5]);
            if (nbU & 2u) reinterpret_cast<R*>(&S.A[2][eu + (int)bU])[0] = last_of<V>(bs[8]);
          }
          if (c >= 1 && !(((rw.bits[c >> 5]) >> (c & 31)) & 1u)) {
            if (nbD & 1u) reinterpret_cast<R*>(&S.A[0][ed - 1])[NL - 1] = first_of<V>(bs[6]);
            if (nbU & 1u) reinterpret_cast<R*>(&S.A[2][eu - 1])[NL - 1] = first_of<V>(bs[7]);
          }
        }
        // done with every row before the first row of my next pass
        __syncwarp();
      }
      __syncwarp();
      if (lane == 0) st_release(&S.done[warp], TY + 2);
    }
    __syncthreads();
    if (tid == 32)
      for (int k = 0; k < SP_NR; k++) mbar_inval((unsigned)__cvta_generic_to_shared(&S.full[k]));
  }
}

// ---- one-time builders (lbm_create) ----
// per compact group: column, fluid bits, x-neighbour groups active, link bytes
__global__ void __launch_bounds__(256) k_sp_meta(const uint8_t* __restrict__ cls, const uint8_t* __restrict__ links,
                                                 const uint2* __restrict__ ptab, int nx, int ny, int nw, int G,
                                                 uint2* __restrict__ gmeta) {
  const long long t = (long long)blockIdx.x * 256 + threadIdx.x;
  const int ng = nx / G;
  if (t >= (long long)ny * ng) return;
  const int r = (int)(t / ng), p = (int)(t % ng);
  const uint2* prow = ptab + (size_t)r * nw;
  auto act = [&](int g) -> unsigned { return (prow[g >> 5].x >> (g & 31)) & 1u; };
  if (!act(p)) return;
  const uint2 tb = prow[p >> 5];
  const size_t ci = (size_t)tb.y + (size_t)__popc(tb.x & ((1u << (p & 31)) - 1u));
  const size_t k = (size_t)r * nx + (size_t)G * p;
  unsigned fl = 0, lk = 0;
  for (int c = 0; c < G; c++)
    if (cls[k + c] < 2) { fl |= 1u << c; lk |= (unsigned)links[k + c] << (8 * c); }
  const unsigned aL = act(p == 0 ? ng - 1 : p - 1), aR = act(p == ng - 1 ? 0 : p + 1);
  gmeta[ci] = make_uint2((unsigned)p | (fl << 16) | (aL << 20) | (aR << 21), lk);
}

__global__ void __launch_bounds__(128) k_sp_desc(const uint2* __restrict__ ptab, const uint2* __restrict__ gmeta, int nx,
                                                 int ny, int nw, int G, int nstrips, int sw, SpDesc* __restrict__ desc,
                                                 uint16_t* __restrict__ cnt) {
  const long long t = (long long)blockIdx.x * 128 + threadIdx.x;
  if (t >= (long long)nstrips * ny) return;
  const int strip = (int)(t / ny), r = (int)(t % ny);
  const int ng = nx / G;
  const int c0 = strip * sw, seff = min(sw, ng - c0);
  const uint2* prow = ptab + (size_t)r * nw;
  auto wrapg = [&](int g) -> int { g %= ng; return g < 0 ? g + ng : g; };
  auto act = [&](int g) -> unsigned { return (prow[g >> 5].x >> (g & 31)) & 1u; };
  auto cidx = [&](int g) -> unsigned {
    const uint2 tb = prow[g >> 5];
    return tb.y + (unsigned)__popc(tb.x & ((1u << (g & 31)) - 1u));
  };
  SpDesc d;
  memset(&d, 0, sizeof d);
  for (int c = -1; c <= seff; c++)
    if (act(wrapg(c0 + c))) d.bits[(c + 1) >> 5] |= 1u << ((c + 1) & 31);
  unsigned run = 0;
  for (int w = 0; w < 4; w++) { d.pre[w] = (uint8_t)run; run += (unsigned)__popc(d.bits[w]); }
  d.hl = (uint8_t)(d.bits[0] & 1u);
  d.hr = (uint8_t)((d.bits[(seff + 1) >> 5] >> ((seff + 1) & 31)) & 1u);
  d.a = (uint16_t)(run - d.hl - d.hr);
  d.ci0 = cidx(c0);
  d.ciL = cidx(wrapg(c0 - 1));
  d.ciR = cidx(wrapg(c0 + seff));
  if (d.hl) d.metaL = gmeta[d.ciL];
  if (d.hr) d.metaR = gmeta[d.ciR];
  desc[t] = d;
  cnt[t] = (uint16_t)run;
}

}  // namespace lbm

// lbm_pair.cuh — PAIR schedule: the fused pull-stream + collide + segregation + phi(t+1) kernel in
// which every lane owns NL x-adjacent nodes (an aligned group: 2 in fp64, 4 in fp32, 2 in fp32 when
// nx is not a multiple of 4), every value moves as an aligned 8- or 16-byte vector, and fp32
// arithmetic is packed (FFMA2/FADD2/FMUL2).  Same arithmetic per node as the other schedules
// (node_update_t), same HBM state.
//
//   * a warp owns a strip of 32 NL columns: 30 NL output columns and one halo LANE per side (only
//     the halo column next to the outputs is needed; groups must stay aligned), and marches down TY
//     rows (+1 halo row per end).  No shared data between warps, no block barrier.
//   * every population is fetched from HBM exactly once per strip, UNSHIFTED, at its own node, by
//     cp.async (LDGSTS) into a private shared-memory ring DP+1 rows ahead of the collision; groups
//     with no fluid node are not fetched.  Propagation (A16-A17, :318-322) is done on chip: the row
//     part by reading the ring slot of the neighbouring row, the column part by one warp shuffle
//     per shifted plane.  Half-way bounce-back (R12) selects the node's own opposite population,
//     which is already on chip.
//   * phi(x, t+1) = sum_q B_q*(x - c_q, t) (A13) is assembled in registers: the B* that move in x
//     shift through the lane's registers and one shuffle, the row moves are carried from one march
//     row to the next; links add the node's own B_opp(q)*.
//   * stores are aligned vectors at the node's own position; a 32-byte sector that holds any fluid
//     node is written whole (zeros on its solid nodes): partial sectors made HBM read-modify-write.
#pragma once
#include <mutex>
#include <utility>
#include <vector>

#include "lbm_kernels.cuh"

namespace lbm {

__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Opt-in to more than 48 KB of dynamic shared memory.  The attribute belongs to (kernel, device), so it is
// remembered per pair; safe to call from several host threads.
inline bool ensure_smem_attr(const void* kern, size_t smem) {
  static std::mutex mu;
  static std::vector<std::pair<const void*, int>> done;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return false;
  std::lock_guard<std::mutex> lk(mu);
  for (const auto& d : done)
    if (d.first == kern && d.second == dev) return true;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return false;
  done.emplace_back(kern, dev);
  return true;
}

// pipeline depth and CTA shape per precision (overridable at build time for tuning sweeps)
#ifndef LBM_PAIR_DP32
#define LBM_PAIR_DP32 1
#endif
#ifndef LBM_PAIR_DP64
#define LBM_PAIR_DP64 1
#endif
// One warp per CTA: the warps share nothing, and a CTA's slot (registers, ring) is only handed on when its last warp
// has finished its march, so with 3-warp CTAs the warps that met more solid rows left their slots idle (11.2 of 12
// warps resident on average at 8192^2; mid-size grids lost more: profiles/r2_small_grids.md).  MINB = warps per SM.
#ifndef LBM_PAIR_MINB32
#define LBM_PAIR_MINB32 15
#endif
#ifndef LBM_PAIR_MINB64
#define LBM_PAIR_MINB64 12
#endif
#ifndef LBM_PAIR_MINBQ
#define LBM_PAIR_MINBQ 12
#endif
#ifndef LBM_PAIR_WARPS
#define LBM_PAIR_WARPS 1
#endif
#ifndef LBM_PAIR_FULLSECTOR
#define LBM_PAIR_FULLSECTOR 1
#endif
#ifndef LBM_PAIR_SECTOR
#define LBM_PAIR_SECTOR 32   // bytes of the write granule that is completed with zeros
#endif
#ifndef LBM_PAIR_CG16
#define LBM_PAIR_CG16 1   // 16-byte cp.async bypasses L1 (.cg): LDGSTS.ca parks its lines in L1, whose size
                          // (what the shared-memory carve-out leaves) then caps the bytes in flight
#endif
#ifndef LBM_PAIR_TY
#define LBM_PAIR_TY 64
#endif
#ifndef LBM_PACK_QUAD
#define LBM_PACK_QUAD 1   // PACK schedule in fp32: 4 nodes per lane and per compacted group (16-byte copies)
#endif
#ifndef LBM_PAIR_QUAD
#define LBM_PAIR_QUAD 1   // PAIR schedule in fp32: 4 nodes per lane when nx % 4 == 0 (16-byte copies can bypass L1)
#endif

// ---- lane value types: NL nodes of one lane ----
struct __align__(16) D2 {   // two fp64 nodes: two interleaved dependency chains
  double x, y;
};
struct __align__(16) Q4 {   // four fp32 nodes: two packed f32x2 streams
  F2 a, b;
};

__device__ __forceinline__ D2 operator+(D2 a, D2 b) { return D2{a.x + b.x, a.y + b.y}; }
__device__ __forceinline__ D2 operator-(D2 a, D2 b) { return D2{a.x - b.x, a.y - b.y}; }
__device__ __forceinline__ D2 operator*(D2 a, D2 b) { return D2{a.x * b.x, a.y * b.y}; }
__device__ __forceinline__ D2 operator-(D2 a) { return D2{-a.x, -a.y}; }
__device__ __forceinline__ D2 operator+(D2 a, double b) { return D2{a.x + b, a.y + b}; }
__device__ __forceinline__ D2 operator+(double a, D2 b) { return D2{a + b.x, a + b.y}; }
__device__ __forceinline__ D2 operator-(D2 a, double b) { return D2{a.x - b, a.y - b}; }
__device__ __forceinline__ D2 operator-(double a, D2 b) { return D2{a - b.x, a - b.y}; }
__device__ __forceinline__ D2 operator*(D2 a, double b) { return D2{a.x * b, a.y * b}; }
__device__ __forceinline__ D2 operator*(double a, D2 b) { return D2{a * b.x, a * b.y}; }
__device__ __forceinline__ D2 rcp_(D2 a) { return D2{1.0 / a.x, 1.0 / a.y}; }
__device__ __forceinline__ D2 rsqrt0_(D2 a) { return D2{rsqrt0_(a.x), rsqrt0_(a.y)}; }

__device__ __forceinline__ Q4 operator+(Q4 a, Q4 b) { return Q4{a.a + b.a, a.b + b.b}; }
__device__ __forceinline__ Q4 operator-(Q4 a, Q4 b) { return Q4{a.a - b.a, a.b - b.b}; }
__device__ __forceinline__ Q4 operator*(Q4 a, Q4 b) { return Q4{a.a * b.a, a.b * b.b}; }
__device__ __forceinline__ Q4 operator-(Q4 a) { return Q4{-a.a, -a.b}; }
__device__ __forceinline__ Q4 operator+(Q4 a, float b) { return Q4{a.a + b, a.b + b}; }
__device__ __forceinline__ Q4 operator+(float a, Q4 b) { return Q4{a + b.a, a + b.b}; }
__device__ __forceinline__ Q4 operator-(Q4 a, float b) { return Q4{a.a - b, a.b - b}; }
__device__ __forceinline__ Q4 operator-(float a, Q4 b) { return Q4{a - b.a, a - b.b}; }
__device__ __forceinline__ Q4 operator*(Q4 a, float b) { return Q4{a.a * b, a.b * b}; }
__device__ __forceinline__ Q4 operator*(float a, Q4 b) { return Q4{a * b.a, a * b.b}; }
__device__ __forceinline__ Q4 rcp_(Q4 a) { return Q4{rcp_(a.a), rcp_(a.b)}; }
__device__ __forceinline__ Q4 rsqrt0_(Q4 a) { return Q4{rsqrt0_(a.a), rsqrt0_(a.b)}; }

// traits: scalar type, nodes per lane, (un)packing into per-node scalars
template <typename V> struct LaneOf;
template <> struct LaneOf<F2> {
  using R = float;
  static constexpr int NL = 2;
  static __device__ __forceinline__ void unpack(F2 v, float (&x)[2]) { x[0] = v.v.x; x[1] = v.v.y; }
  static __device__ __forceinline__ F2 pack(const float (&x)[2]) { return f2(x[0], x[1]); }
};
template <> struct LaneOf<D2> {
  using R = double;
  static constexpr int NL = 2;
  static __device__ __forceinline__ void unpack(D2 v, double (&x)[2]) { x[0] = v.x; x[1] = v.y; }
  static __device__ __forceinline__ D2 pack(const double (&x)[2]) { return D2{x[0], x[1]}; }
};
template <> struct LaneOf<Q4> {
  using R = float;
  static constexpr int NL = 4;
  static __device__ __forceinline__ void unpack(Q4 v, float (&x)[4]) {
    x[0] = v.a.v.x; x[1] = v.a.v.y; x[2] = v.b.v.x; x[3] = v.b.v.y;
  }
  static __device__ __forceinline__ Q4 pack(const float (&x)[4]) { return Q4{f2(x[0], x[1]), f2(x[2], x[3])}; }
};

// propagation in x by one node: the value arriving from the left neighbour (c_x = +1) / from the
// right neighbour (c_x = -1); one element crosses the lane boundary by shuffle
template <typename V>
__device__ __forceinline__ V from_left(V a) {
  using L = LaneOf<V>;
  typename L::R x[L::NL], y[L::NL];
  L::unpack(a, x);
  y[0] = __shfl_up_sync(0xffffffffu, x[L::NL - 1], 1);
#pragma unroll
  for (int c = 1; c < L::NL; c++) y[c] = x[c - 1];
  return L::pack(y);
}
template <typename V>
__device__ __forceinline__ V from_right(V a) {
  using L = LaneOf<V>;
  typename L::R x[L::NL], y[L::NL];
  L::unpack(a, x);
#pragma unroll
  for (int c = 0; c < L::NL - 1; c++) y[c] = x[c + 1];
  y[L::NL - 1] = __shfl_down_sync(0xffffffffu, x[0], 1);
  return L::pack(y);
}
template <typename V>
__device__ __forceinline__ V splat(typename LaneOf<V>::R s) {
  using L = LaneOf<V>;
  typename L::R x[L::NL];
#pragma unroll
  for (int c = 0; c < L::NL; c++) x[c] = s;
  return L::pack(x);
}

#ifndef LBM_PAIR_STORE_CS
#define LBM_PAIR_STORE_CS 0
#endif
// vector store of a lane's NL values; optionally with the streaming (evict-first) cache hint
template <typename V>
__device__ __forceinline__ void store_vec(void* p, V v) {
#if LBM_PAIR_STORE_CS
  if constexpr (sizeof(V) == 8) {
    const float2 t = *reinterpret_cast<const float2*>(&v);
    __stcs(reinterpret_cast<float2*>(p), t);
  } else {
    const float4 t = *reinterpret_cast<const float4*>(&v);
    __stcs(reinterpret_cast<float4*>(p), t);
  }
#else
  *reinterpret_cast<V*>(p) = v;
#endif
}

template <int BYTES>
__device__ __forceinline__ void cp_async_vec(unsigned saddr, const void* gptr) {
  // 4- and 8-byte copies exist only as .ca; 16-byte copies bypass L1 (.cg): each sector then crosses the
  // L2 -> SM link once per 16-byte lane, but L1 capacity no longer limits how many rows are in flight
#if LBM_PAIR_CG16
  if constexpr (BYTES == 16) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(saddr), "l"(gptr) : "memory");
    return;
  }
#endif
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(saddr), "l"(gptr), "n"(BYTES) : "memory");
}

// shared-memory ring of one warp: row stages hold the own-position populations and phi of the strip;
// class stages the packed class words (NL 16-bit words per lane)
// PACK schedule only: {group mask word, compact index of its first group} per class row.  Kept out of
// the ring of the other schedules: 3 CTAs x 64 KB is the most that fits the 196 KB shared-memory carve-out,
// one KB more selects the 228 KB carve-out, halves L1 and costs 30 % (LDGSTS allocates its lines in L1).
template <int CS, bool PACKED> struct RingTab { uint2 Tb[CS][32]; };
template <int CS> struct RingTab<CS, false> {};
template <typename V, int DP, bool PACKED>
struct PairRing : RingTab<2 * DP + 2, PACKED> {
  static constexpr int NL = LaneOf<V>::NL;
  static constexpr int NS = DP + 2;        // population rows i-1 (until refilled) .. i+1+DP
  static constexpr int PS = DP + 3;        // phi rows i-1 .. i+1+DP
  static constexpr int CS = 2 * DP + 2;    // class rows i .. i+1+2DP
  V N[NS][9][32];
  V P[PS][32];
  unsigned short Cw[CS][32][NL];
};

// collide the NL nodes of a lane (fl[c]: node c is fluid).  All nodes always go through the
// arithmetic together: packed FFMA2 in fp32, interleaved dependency chains in fp64.  A node that is
// not fluid gets B* = 0 through the mask and stores N* = 0, so that its slots stay finite.
template <typename V>
__device__ __forceinline__ void collide_lane(const Consts<typename LaneOf<V>::R>& C, const V (&n)[9],
                                             const V (&ph)[9], const bool (&fl)[LaneOf<V>::NL], bool all_fluid,
                                             V (&ns)[9], V (&bs)[9]) {
  using L = LaneOf<V>;
  using R = typename L::R;
  R m[L::NL];
#pragma unroll
  for (int c = 0; c < L::NL; c++) m[c] = fl[c] ? R(1) : R(0);
  node_update_t<V, R, true, true>(C, n, ph, ns, bs, nullptr, L::pack(m));
  if (!all_fluid) {
#pragma unroll
    for (int q = 0; q < 9; q++) {
      R x[L::NL];
      L::unpack(ns[q], x);
#pragma unroll
      for (int c = 0; c < L::NL; c++) x[c] = fl[c] ? x[c] : R(0);
      ns[q] = L::pack(x);
    }
  }
}

// PACKED: the population planes are pair-compacted (PACK schedule, see k_pair_mask): Nsrc / Ndst hold only
// the pairs with a fluid node, plane stride cpsB bytes, addressed through ptab (nw words per row).
template <typename V, int DP, int WARPS, int MINB, bool WRITE_B, bool PACKED>
__global__ void __launch_bounds__(32 * WARPS, MINB)
    k_fused_pair(const Consts<typename LaneOf<V>::R> C, const uint16_t* __restrict__ cl16,
                 const typename LaneOf<V>::R* __restrict__ Nsrc, typename LaneOf<V>::R* __restrict__ Ndst,
                 typename LaneOf<V>::R* __restrict__ Bdst, const typename LaneOf<V>::R* __restrict__ phi_in,
                 typename LaneOf<V>::R* __restrict__ phi_out, int TY, const uint2* __restrict__ ptab, int nw,
                 unsigned cpsB) {
  using L = LaneOf<V>;
  using R = typename L::R;
  using Ring = PairRing<V, DP, PACKED>;
  constexpr int NL = L::NL;
  constexpr int OUTC = 30 * NL;            // output columns of a strip
  constexpr unsigned FULL = 0xffffffffu;
  constexpr int VB = NL * (int)sizeof(R);  // bytes of a lane vector
  constexpr int NS = Ring::NS, PS = Ring::PS, CS = Ring::CS;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Ring& S = reinterpret_cast<Ring*>(smem_raw)[threadIdx.x >> 5];
  const int lane = threadIdx.x & 31;
  const unsigned sN0 = (unsigned)__cvta_generic_to_shared(&S.N[0][0][PACKED ? 0 : lane]);
  const unsigned sP0 = (unsigned)__cvta_generic_to_shared(&S.P[0][lane]);
  const unsigned sC0 = (unsigned)__cvta_generic_to_shared(&S.Cw[0][lane][0]);
  unsigned sT0 = 0;
  if constexpr (PACKED) sT0 = (unsigned)__cvta_generic_to_shared(&S.Tb[0][lane]);
  constexpr unsigned N_STAGE = 9 * 32 * VB, N_PLANE = 32 * VB, P_STAGE = 32 * VB, C_STAGE = 32 * NL * 2;

  const int nx = C.nx, ny = C.ny;   // nx is a multiple of NL (checked by the launcher)
  const unsigned psB = PACKED ? cpsB : (unsigned)C.ps * (unsigned)sizeof(R);   // plane stride in bytes (< 2^32: lbm_create)
  const unsigned psBd = (unsigned)C.ps * (unsigned)sizeof(R);                  // dense stride (B planes of lbm_keep_B)
  const int g = blockIdx.x * WARPS + (threadIdx.x >> 5);
  if (OUTC * g >= nx) return;                            // whole warp; the kernel has no block barrier
  const int xend = min(OUTC * g + OUTC, nx);             // one past the last output column (multiple of NL)
  const int lxa = OUTC * g - NL + NL * lane;             // logical column of the lane's first node
  const bool col_out = lane >= 1 && lane <= 30 && lxa < xend;
  int xa = lxa % nx;                                     // every lane is a valid periodic group
  if (xa < 0) xa += nx;
  const int pword = (xa / NL) >> 5;                      // PACK: word and bit of the lane's group in ptab
  const unsigned pbit = (unsigned)(xa / NL) & 31u, plt = (1u << pbit) - 1u;
  // lanes whose groups share a 32-byte sector of a population plane (rows keep the sector phase only
  // if the row pitch is a multiple of 32 bytes); a sector that holds any fluid node is stored whole
  // (zeros on its solid nodes), so that HBM never has to read-modify-write a partial sector
  const int sector = (lxa + 32 * NL) * (int)sizeof(R) / LBM_PAIR_SECTOR;
  const unsigned gmask = (LBM_PAIR_FULLSECTOR && (nx * (int)sizeof(R)) % LBM_PAIR_SECTOR == 0) ? __match_any_sync(FULL, sector) : (1u << lane);
  const int j0 = blockIdx.y * TY;
  const int rows = min(TY, ny - j0);
  const int last = rows + 1;                             // march row m = grid row j0-1+m; collided: 0..last

  auto wrap_row = [=](int m) -> int {                    // grid row of march row m, periodic in y
    int r = j0 - 1 + m;
    return r < 0 ? r + ny : (r >= ny ? r - ny : r);
  };
  auto inc = [](int v, int mod) { return v + 1 == mod ? 0 : v + 1; };
  // ---- asynchronous fetches (slots and row offsets are passed in: no modulo in the march) ----
  auto issue_cls = [&](int r, int sc) {   // the NL class words of the lane in grid row r (one aligned word)
    cp_async_vec<NL * 2>(sC0 + (unsigned)sc * C_STAGE, cl16 + ((unsigned)r * (unsigned)nx + (unsigned)xa));
    if constexpr (PACKED) cp_async_vec<8>(sT0 + (unsigned)sc * 256u, ptab + ((size_t)r * nw + pword));
  };
  // own-position populations and phi of one march row; lower/upper: the row feeds c_y <= 0 / c_y >= 0
  auto issue_row = [&](unsigned u, int sn, int sp, int sc, bool lower, bool upper) {
    unsigned cmin = 3u;   // least class of the lane's nodes: 0,1 fluid; 2 ghost; 3 bulk solid
#pragma unroll
    for (int c = 0; c < NL; c++) {
      const unsigned cc = S.Cw[sc][lane][c] & 0xffu;
      cmin = min(cmin, cc);
    }
    const unsigned k = u + (unsigned)xa;
    if (cmin != 3u) cp_async_vec<VB>(sP0 + (unsigned)sp * P_STAGE, phi_in + k);
    if (cmin < 2u) {
      unsigned ke = k;                                             // element offset of the group in a plane
      unsigned d = sN0 + (unsigned)sn * N_STAGE;
      if constexpr (PACKED) {
        const uint2 tb = S.Tb[sc][lane];
        const unsigned ci = tb.y + (unsigned)__popc(tb.x & plt);
        ke = ci * (unsigned)NL;
        d += (unsigned)lane * VB;   // entry = lane (an entry aligned to the compact index was tried: no gain)
      }
      const char* src = reinterpret_cast<const char*>(Nsrc + ke);   // plane q is src + q * psB
      if (lower && upper) {
        cp_async_vec<VB>(d + 0 * N_PLANE, src);
        cp_async_vec<VB>(d + 1 * N_PLANE, src + (size_t)psB * 1u);
        cp_async_vec<VB>(d + 3 * N_PLANE, src + (size_t)psB * 3u);
      }
      if (upper) {
        cp_async_vec<VB>(d + 2 * N_PLANE, src + (size_t)psB * 2u);
        cp_async_vec<VB>(d + 5 * N_PLANE, src + (size_t)psB * 5u);
        cp_async_vec<VB>(d + 6 * N_PLANE, src + (size_t)psB * 6u);
      }
      if (lower) {
        cp_async_vec<VB>(d + 4 * N_PLANE, src + (size_t)psB * 4u);
        cp_async_vec<VB>(d + 7 * N_PLANE, src + (size_t)psB * 7u);
        cp_async_vec<VB>(d + 8 * N_PLANE, src + (size_t)psB * 8u);
      }
    }
  };

  // ---- prologue: ring slot of march row m is (m + 1) mod ring size ----
  const V zero = splat<V>(R(0));
  {   // stale ring entries are read (and discarded) for solid nodes: they must be finite
#pragma unroll
    for (int s = 0; s < NS; s++)
#pragma unroll
      for (int q = 0; q < 9; q++) S.N[s][q][lane] = zero;
#pragma unroll
    for (int s = 0; s < PS; s++) S.P[s][lane] = zero;
  }
  for (int m = -1; m <= 2 * DP; m++)
    if (m <= last + 1) issue_cls(wrap_row(m), (m + 1) % CS);
  cp_async_commit();
  cp_async_wait<0>();
  for (int m = -1; m <= DP; m++) {
    if (m <= last + 1)
      issue_row((unsigned)wrap_row(m) * (unsigned)nx, (m + 1) % NS, (m + 1) % PS, (m + 1) % CS, m >= 0, m <= last);
    cp_async_commit();
  }

  // march state: ring slots of rows i-1, i, i+1 (populations, phi), of the rows being fetched, and
  // the grid rows of the two fetch fronts
  int sN_a = 0, sN_b = 1 % NS, sN_c = 2 % NS;
  int sP_a = 0, sP_b = 1, sP_c = 2, sP_f = (DP + 2) % PS;
  int sC_i = 1 % CS, sC_f = (DP + 2) % CS, sC_n = (2 * DP + 2) % CS;
  int rf = wrap_row(DP + 1), rc = wrap_row(2 * DP + 1);
  unsigned kout = (unsigned)(j0 - 1) * (unsigned)nx + (unsigned)xa;   // own group of march row i (1 <= i <= rows)
  V acc_prev = zero, up_prev = zero;
  bool fl_prev[NL];
#pragma unroll
  for (int c = 0; c < NL; c++) fl_prev[c] = false;

  for (int i = 0; i <= last; i++) {
    cp_async_wait<DP - 1>();   // row i+1 and the class words of row i+1+DP have landed
    // operands that live in the slot about to be refilled: planes 2,5,6 of row i-1
    const int lm = lane, lc = lane, ln = lane;   // ring entries of the lane's group in rows i-1, i, i+1
    const V Bp0 = S.N[sN_a][2][lm], Bp1 = S.N[sN_a][5][lm], Bp2 = S.N[sN_a][6][lm];
    const V pS = S.P[sP_a][lane];
    // ---- issue: populations and phi of row i+1+DP, class words of row i+1+2DP ----
    if (i + 1 + DP <= last + 1) issue_row((unsigned)rf * (unsigned)nx, sN_a, sP_f, sC_f, true, i + 1 + DP <= last);
    if (i + 1 + 2 * DP <= last + 1) issue_cls(rc, sC_n);
    cp_async_commit();

    // ---- on-chip operands of march row i ----
    const V A0 = S.N[sN_b][0][lc], A1 = S.N[sN_b][1][lc], A3 = S.N[sN_b][3][lc];
    const V Cn0 = S.N[sN_c][4][ln], Cn1 = S.N[sN_c][7][ln], Cn2 = S.N[sN_c][8][ln];
    const V pC = S.P[sP_b][lane], pN = S.P[sP_c][lane];

    bool fl[NL];
    unsigned lk[NL];
    bool any_fl = false, all_fl = true;
    unsigned lk_any = 0u;
#pragma unroll
    for (int c = 0; c < NL; c++) {
      const unsigned w = S.Cw[sC_i][lane][c];
      fl[c] = (w & 0xffu) < 2u;
      lk[c] = fl[c] ? (w >> 8) : 0u;
      any_fl |= fl[c]; all_fl &= fl[c]; lk_any |= lk[c];
    }
    const bool any_link = __any_sync(FULL, lk_any != 0u);

    // pulled populations: propagation A16-A17 on chip
    V nn[9];
    nn[0] = A0;  nn[1] = from_left(A1);   nn[3] = from_right(A3);
    nn[2] = Bp0; nn[5] = from_left(Bp1);  nn[6] = from_right(Bp2);
    nn[4] = Cn0; nn[7] = from_right(Cn1); nn[8] = from_left(Cn2);
    if (any_link) {   // warp-uniform; half-way bounce-back (R12): own opposite population, same row
      const V own[9] = {A0, A1, S.N[sN_b][2][lc], A3, S.N[sN_b][4][lc], S.N[sN_b][5][lc],
                        S.N[sN_b][6][lc], S.N[sN_b][7][lc], S.N[sN_b][8][lc]};   // plane q at (x, i)
#pragma unroll
      for (int q = 1; q < 9; q++) {
        R a[NL], o[NL];
        L::unpack(nn[q], a);
        L::unpack(own[opp(q)], o);
#pragma unroll
        for (int c = 0; c < NL; c++)
          if ((lk[c] >> (q - 1)) & 1u) a[c] = o[c];
        nn[q] = L::pack(a);
      }
    }
    const unsigned fmask = __ballot_sync(FULL, col_out && any_fl);
    // dense planes: my sector holds a fluid node; compact planes have no holes: my pair holds one
    const bool st = col_out && i >= 1 && i <= rows && (PACKED ? any_fl : (fmask & gmask) != 0u);
    // phi stencil (R8): west / east neighbours of the three rows (shuffles: all lanes take part)
    const V pCw = from_left(pC), pCe = from_right(pC), pNw = from_left(pN), pNe = from_right(pN);
    const V pSw = from_left(pS), pSe = from_right(pS);

    V bs[9];
    V bb = zero;
    if (any_fl || st) {   // st without a fluid node: a solid group completing a sector with zeros
      const V ph[9] = {pC, pCe, pN, pCw, pS, pNe, pNw, pSw, pSe};
      V ns[9];
      collide_lane<V>(C, nn, ph, fl, all_fl, ns, bs);
      if (st) {
        unsigned ko = kout;
        if constexpr (PACKED) {
          const uint2 tb = S.Tb[sC_i][lane];
          ko = (tb.y + (unsigned)__popc(tb.x & plt)) * (unsigned)NL;
        }
        char* dst = reinterpret_cast<char*>(Ndst + ko);
#pragma unroll
        for (int q = 0; q < 9; q++) store_vec<V>(dst + (size_t)psB * (unsigned)q, ns[q]);
        if (WRITE_B) {
          char* dstB = reinterpret_cast<char*>(Bdst + kout);
#pragma unroll
          for (int q = 0; q < 9; q++) *reinterpret_cast<V*>(dstB + (size_t)psBd * (unsigned)q) = bs[q];
        }
      }
      if (lk_any) {   // link q hands the node its own B_opp(q)* back
        R b[NL];
#pragma unroll
        for (int c = 0; c < NL; c++) b[c] = R(0);
#pragma unroll
        for (int q = 1; q < 9; q++) {
          R o[NL];
          L::unpack(bs[opp(q)], o);
#pragma unroll
          for (int c = 0; c < NL; c++)
            if ((lk[c] >> (q - 1)) & 1u) b[c] += o[c];
        }
        bb = L::pack(b);
      }
    } else {
#pragma unroll
      for (int q = 0; q < 9; q++) bs[q] = zero;
    }
    // contributions of row i to phi(t+1) of rows i-1 (down), i (mid), i+1 (up)
    const V mid = bs[0] + from_left(bs[1]) + from_right(bs[3]);
    const V upw = bs[2] + from_left(bs[5]) + from_right(bs[6]);
    const V down = bs[4] + from_right(bs[7]) + from_left(bs[8]);
    if (i >= 2 && col_out) {
      const V pn = acc_prev + down;
      R* dst = phi_out + (kout - (unsigned)nx);
      bool allp = true;
#pragma unroll
      for (int c = 0; c < NL; c++) allp &= fl_prev[c];
      if (allp) store_vec<V>(dst, pn);
      else {
        R x[NL];
        L::unpack(pn, x);
#pragma unroll
        for (int c = 0; c < NL; c++)
          if (fl_prev[c]) dst[c] = x[c];
      }
    }
    acc_prev = (up_prev + mid) + bb;
    up_prev = upw;
#pragma unroll
    for (int c = 0; c < NL; c++) fl_prev[c] = fl[c];

    kout += (unsigned)nx;
    sN_a = sN_b; sN_b = sN_c; sN_c = inc(sN_c, NS);
    sP_a = sP_b; sP_b = sP_c; sP_c = inc(sP_c, PS); sP_f = inc(sP_f, PS);
    sC_i = inc(sC_i, CS); sC_f = inc(sC_f, CS); sC_n = inc(sC_n, CS);
    rf = inc(rf, ny); rc = inc(rc, ny);
  }
  cp_async_wait<0>();
}

template <typename V, int DP, int MINB, bool PACKED>
bool launch_fused_lane(const Consts<typename LaneOf<V>::R>& C, const uint16_t* cl16,
                       const typename LaneOf<V>::R* Nsrc, typename LaneOf<V>::R* Ndst, typename LaneOf<V>::R* Bdst,
                       const typename LaneOf<V>::R* phi_in, typename LaneOf<V>::R* phi_out, cudaStream_t st,
                       const uint2* ptab = nullptr, int nw = 0, unsigned cpsB = 0) {
  constexpr int WARPS = LBM_PAIR_WARPS;
  constexpr int OUTC = 30 * LaneOf<V>::NL;
  const int nwx = (C.nx + OUTC - 1) / OUTC;
  const int gx = (nwx + WARPS - 1) / WARPS;
  // Rows per warp march.  Long marches amortise the two halo rows and the pipeline fill (about 6 rows' worth); short
  // ones make more CTAs.  The CTAs of a launch run in waves of `slots` (every resident warp takes about as long per row
  // whether the SM is full or not), so a launch takes about ceil(CTAs / slots) x (TY + 6) row times: take the TY that
  // minimises it.  What matters on mid-size grids is that the last wave is full: 2048^2 runs 10-12 % faster with the
  // march length that fits the grid into exactly one wave (41 rows in fp64, 21 in fp32) than with a power of two
  // (profiles/r2_small_grids.md).
  int nsm = 148;
  {
    int dev = 0;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  }
  const long long slots = (long long)nsm * MINB;
  int TY = LBM_PAIR_TY;
  long long best = -1;
  for (int t = LBM_PAIR_TY; t >= 8; t--) {   // marches shorter than 8 rows lost wherever they were tried
    const long long ctas = (long long)gx * ((C.ny + t - 1) / t);
    const long long cost = ((ctas + slots - 1) / slots) * (t + 6);
    if (best < 0 || cost < best) { best = cost; TY = t; }
  }
  // very small grids (less than four warps per SM even then): the march itself is what a launch-bound step waits for
  while (TY > 2 && (long long)nwx * ((C.ny + TY - 1) / TY) < nsm * 4) TY >>= 1;
  const dim3 grid((unsigned)gx, (unsigned)((C.ny + TY - 1) / TY), 1);
  const size_t smem = sizeof(PairRing<V, DP, PACKED>) * WARPS;
  auto kern = Bdst ? k_fused_pair<V, DP, WARPS, MINB, true, PACKED> : k_fused_pair<V, DP, WARPS, MINB, false, PACKED>;
  if (!ensure_smem_attr(reinterpret_cast<const void*>(kern), smem)) return false;
  kern<<<grid, 32 * WARPS, smem, st>>>(C, cl16, Nsrc, Ndst, Bdst, phi_in, phi_out, TY, ptab, nw, cpsB);
  return true;
}

// returns false if the grid does not fit the schedule (odd nx): the caller uses another schedule
inline bool launch_fused_pair(const Consts<double>& C, const uint16_t* cl16, const double* Nsrc, double* Ndst,
                              double* Bdst, const double* phi_in, double* phi_out, cudaStream_t st) {
  if (C.nx & 1) return false;
  return launch_fused_lane<D2, LBM_PAIR_DP64, LBM_PAIR_MINB64, false>(C, cl16, Nsrc, Ndst, Bdst, phi_in, phi_out, st);
}
inline bool launch_fused_pair(const Consts<float>& C, const uint16_t* cl16, const float* Nsrc, float* Ndst,
                              float* Bdst, const float* phi_in, float* phi_out, cudaStream_t st) {
  if (C.nx & 1) return false;
  if (LBM_PAIR_QUAD && (C.nx & 3) == 0)
    return launch_fused_lane<Q4, LBM_PAIR_DP32, LBM_PAIR_MINBQ, false>(C, cl16, Nsrc, Ndst, Bdst, phi_in, phi_out, st);
  return launch_fused_lane<F2, LBM_PAIR_DP32, LBM_PAIR_MINB32, false>(C, cl16, Nsrc, Ndst, Bdst, phi_in, phi_out, st);
}

// nodes per compacted group of the PACK schedule: the kernel's nodes per lane (4 in fp32 when the quad
// variant is enabled and nx allows it, else 2)
inline int pack_group(int elem_size, int nx) { return (elem_size == 4 && LBM_PACK_QUAD && (nx & 3) == 0) ? 4 : 2; }

// PACK schedule: the same kernel on group-compacted planes (Nsrc / Ndst are the compact buffers)
inline bool launch_fused_pack(const Consts<double>& C, const uint16_t* cl16, const double* Nsrc, double* Ndst,
                              double* Bdst, const double* phi_in, double* phi_out, cudaStream_t st,
                              const uint2* ptab, int nw, unsigned cpsB) {
  return launch_fused_lane<D2, LBM_PAIR_DP64, LBM_PAIR_MINB64, true>(C, cl16, Nsrc, Ndst, Bdst, phi_in, phi_out, st, ptab, nw, cpsB);
}
inline bool launch_fused_pack(const Consts<float>& C, const uint16_t* cl16, const float* Nsrc, float* Ndst,
                              float* Bdst, const float* phi_in, float* phi_out, cudaStream_t st,
                              const uint2* ptab, int nw, unsigned cpsB) {
  if (pack_group(4, C.nx) == 4)
    return launch_fused_lane<Q4, LBM_PAIR_DP32, LBM_PAIR_MINBQ, true>(C, cl16, Nsrc, Ndst, Bdst, phi_in, phi_out, st, ptab, nw, cpsB);
  return launch_fused_lane<F2, LBM_PAIR_DP32, LBM_PAIR_MINB32, true>(C, cl16, Nsrc, Ndst, Bdst, phi_in, phi_out, st, ptab, nw, cpsB);
}

}  // namespace lbm

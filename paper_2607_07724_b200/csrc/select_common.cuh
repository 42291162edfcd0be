// select_common.cuh -- device helpers shared by the selection kernels: the order-preserving
// fp32 <-> uint32 key map and the one-warp top-(2k) selection + sigma (Eq.4 / Eq.9-11,
// L94-109, L307-324; readings G1, G5, G6).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bsa {

// ---- order-preserving fp32 <-> uint32 map (ascending); -0 is folded onto +0 ---------------------
__device__ __forceinline__ uint32_t okey(float x) {
  x += 0.0f;
  const uint32_t u = __float_as_uint(x);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float unkey(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k ^ 0x80000000u) : ~k);
}

constexpr int kMaxCand = 264;  // 2 * k_budget <= 256, plus the rank-2k candidate of the diagnostics

// Tells the producer of keys[] that this warp holds everything it needs in registers: one arrival
// on the shared-memory mbarrier `bar` (0 = nobody is waiting).
__device__ __forceinline__ void release_keys(uint32_t bar, int lane) {
  __syncwarp();
  if (bar != 0u && lane == 0)
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// Keys of the free blocks 1..t-1 are held KPL per lane in registers (entry j of lane l is free index
// j*32+l; 0 pads, it is below every key of a finite score).  Finds the need-th largest key by
// bisection on the bits below the common prefix of the warp's min and max key, then compacts the
// selected entries in index order (ties at the threshold -> lower block index, G6) into cand[] as
// (key << 32) | ~block.  n_free > need.  keys[] is not read again once release_keys() has run.
template <int KPL>
__device__ __forceinline__ void warp_topk_compact(const uint32_t* keys, int n_free, int need,
                                                  unsigned long long* cand, int lane,
                                                  uint32_t release_bar) {
  const unsigned full = 0xffffffffu;
  uint32_t r[KPL];
  uint32_t hi = 0u, lo = 0xffffffffu;
#pragma unroll
  for (int j = 0; j < KPL; ++j) {
    const int i = j * 32 + lane;
    const bool v = i < n_free;
    r[j] = v ? keys[1 + i] : 0u;
    hi = max(hi, r[j]);
    lo = v ? min(lo, r[j]) : lo;
  }
  release_keys(release_bar, lane);
  hi = __reduce_max_sync(full, hi);
  lo = __reduce_min_sync(full, lo);
  uint32_t vth = hi;
  int r_eq = need;                       // all keys equal: the `need` lowest indices win
  const uint32_t diff = hi ^ lo;
  if (diff != 0u) {
    const int top = 31 - __clz(diff);
    uint32_t prefix = (top == 31) ? 0u : (hi & ~((2u << top) - 1u));
    bool exact = false;
    for (int bit = top; bit >= 0; --bit) {
      const uint32_t c = prefix | (1u << bit);
      int cnt = 0;
#pragma unroll
      for (int j = 0; j < KPL; ++j) cnt += (r[j] >= c) ? 1 : 0;
      cnt = __reduce_add_sync(full, cnt);
      if (cnt >= need) prefix = c;
      if (cnt == need) { exact = true; break; }   // {key >= c} is exactly the top `need`
    }
    if (exact) {
      vth = prefix - 1u;                 // key > vth  <=>  key >= c
      r_eq = 0;
    } else {
      vth = prefix;                      // the need-th largest key itself
      int cgt = 0;
#pragma unroll
      for (int j = 0; j < KPL; ++j) cgt += (r[j] > vth) ? 1 : 0;
      cgt = __reduce_add_sync(full, cgt);
      r_eq = need - cgt;
    }
  }
  int base = 0, eq_seen = 0;
  const unsigned lt = (1u << lane) - 1u;
#pragma unroll
  for (int j = 0; j < KPL; ++j) {
    if (j * 32 < n_free) {               // warp-uniform
      const int i = j * 32 + lane;
      const bool valid = i < n_free;
      const bool gt = valid && r[j] > vth;
      const bool eq = valid && r[j] == vth && r_eq > 0;
      const unsigned be = __ballot_sync(full, eq);
      const bool take = gt || (eq && (eq_seen + __popc(be & lt) < r_eq));
      const unsigned bsel = __ballot_sync(full, take);
      if (take)
        cand[base + __popc(bsel & lt)] =
            (static_cast<unsigned long long>(r[j]) << 32) | (0xFFFFFFFFu - static_cast<uint32_t>(1 + i));
      base += __popc(bsel);
      eq_seen += __popc(be);
    }
  }
}

// Same result for n_free beyond the register path (KPL = 128 holds 4096 keys per warp): the keys
// stay in shared memory and every bisection step re-reads them (32 passes of n_free / 32 loads per
// lane -- only tiles with more than 4097 visible blocks take this path: > 256K tokens at block 64).
// keys[] is released only after the compaction.
static __device__ __noinline__ void warp_topk_compact_smem(const uint32_t* keys, int n_free, int need,
                                                           unsigned long long* cand, int lane,
                                                           uint32_t release_bar) {
  const unsigned full = 0xffffffffu;
  uint32_t hi = 0u, lo = 0xffffffffu;
  for (int i = lane; i < n_free; i += 32) {
    const uint32_t v = keys[1 + i];
    hi = max(hi, v);
    lo = min(lo, v);
  }
  hi = __reduce_max_sync(full, hi);
  lo = __reduce_min_sync(full, lo);
  uint32_t vth = hi;
  int r_eq = need;
  const uint32_t diff = hi ^ lo;
  if (diff != 0u) {
    const int top = 31 - __clz(diff);
    uint32_t prefix = (top == 31) ? 0u : (hi & ~((2u << top) - 1u));
    bool exact = false;
    for (int bit = top; bit >= 0; --bit) {
      const uint32_t c = prefix | (1u << bit);
      int cnt = 0;
      for (int i = lane; i < n_free; i += 32) cnt += (keys[1 + i] >= c) ? 1 : 0;
      cnt = __reduce_add_sync(full, cnt);
      if (cnt >= need) prefix = c;
      if (cnt == need) { exact = true; break; }
    }
    if (exact) {
      vth = prefix - 1u;
      r_eq = 0;
    } else {
      vth = prefix;
      int cgt = 0;
      for (int i = lane; i < n_free; i += 32) cgt += (keys[1 + i] > vth) ? 1 : 0;
      cgt = __reduce_add_sync(full, cgt);
      r_eq = need - cgt;
    }
  }
  int base = 0, eq_seen = 0;
  const unsigned lt = (1u << lane) - 1u;
  for (int i0 = 0; i0 < n_free; i0 += 32) {
    const int i = i0 + lane;
    const bool valid = i < n_free;
    const uint32_t v = valid ? keys[1 + i] : 0u;
    const bool gt = valid && v > vth;
    const bool eq = valid && v == vth && r_eq > 0;
    const unsigned be = __ballot_sync(full, eq);
    const bool take = gt || (eq && (eq_seen + __popc(be & lt) < r_eq));
    const unsigned bsel = __ballot_sync(full, take);
    if (take)
      cand[base + __popc(bsel & lt)] =
          (static_cast<unsigned long long>(v) << 32) | (0xFFFFFFFFu - static_cast<uint32_t>(1 + i));
    base += __popc(bsel);
    eq_seen += __popc(be);
  }
  release_keys(release_bar, lane);
}

// D.4 per-cell diagnostics (Eq.18; recipe L486-491) of one (tile, head):
//   g  = s~[k-1] - s~[k]       cutoff gap            G = s~[k-1] - s~[rho k]   expansion gap
//   r  = s~[f]   - s~[k]       spread (reading G1)   d2 = min_{j in [f, rho k), j != k-1} s~[j] - s~[j+1]
// defined on tiles with at least rho*k + 1 visible blocks (L493); NaN elsewhere.
struct DiagCell {
  float g, G, r, d2;
};

// One warp.  keys[0..t] = order-preserving keys (okey) of the tile scores of the visible blocks, in
// shared memory.  Writes the first W slots of the sorted row [0, t, free blocks by (score desc, index
// asc)], padded with NB, and returns sigma (Eq.4 / Eq.11; G1, G5).  s3 = 4 words of scratch.
// `release_bar`: mbarrier (shared-memory address, or 0) that receives exactly one arrival as soon as
// keys[] has been consumed, so that the buffer can be refilled while the selection continues.
// `dg` != nullptr: also the diagnostics above (one more candidate, rank rho*k, is selected; `srt` =
// kMaxCand words of per-warp shared memory that receive the sorted keys).
static __device__ float warp_select(const uint32_t* keys, int t, int k, int NB, int W, int32_t* row_out,
                                    unsigned long long* cand, uint32_t* s3, int lane,
                                    uint32_t release_bar = 0u, DiagCell* dg = nullptr,
                                    uint32_t* srt = nullptr) {
  const int f = (t == 0) ? 1 : 2;               // forced: sink, self (Eq.9)
  const int n_free = (t >= 2) ? t - 1 : 0;      // blocks 1 .. t-1
  const int want = 2 * k - f + (dg ? 1 : 0);    // diagnostics read the score at rank rho*k as well
  const int need = want < n_free ? want : n_free;
  if (need > 0) {
    if (n_free <= need) {
      for (int i = lane; i < n_free; i += 32)
        cand[i] = (static_cast<unsigned long long>(keys[1 + i]) << 32) |
                  (0xFFFFFFFFu - static_cast<uint32_t>(1 + i));
      release_keys(release_bar, lane);
    } else if (n_free <= 32 * 8) {
      warp_topk_compact<8>(keys, n_free, need, cand, lane, release_bar);
    } else if (n_free <= 32 * 16) {
      warp_topk_compact<16>(keys, n_free, need, cand, lane, release_bar);
    } else if (n_free <= 32 * 32) {
      warp_topk_compact<32>(keys, n_free, need, cand, lane, release_bar);
    } else if (n_free <= 32 * 64) {
      warp_topk_compact<64>(keys, n_free, need, cand, lane, release_bar);
    } else if (n_free <= 32 * 128) {
      warp_topk_compact<128>(keys, n_free, need, cand, lane, release_bar);
    } else {
      warp_topk_compact_smem(keys, n_free, need, cand, lane, release_bar);
    }
    __syncwarp();
    // order by rank: the (key, ~block) words are distinct, so rank = #{cand > mine} is a permutation
    const int i_hi = k - 1 - f, i_lo = k - f;   // ranks of s~[k-1] and s~[k] in the free list
    const int i_2k = 2 * k - f;                 // rank of s~[rho k] (diagnostics only)
    for (int q = lane; q < need; q += 32) {
      const unsigned long long mine = cand[q];
      int rank = 0;
      for (int u = 0; u < need; ++u) rank += (cand[u] > mine) ? 1 : 0;
      const int slot = f + rank;
      if (slot < W) row_out[slot] = static_cast<int>(0xFFFFFFFFu - static_cast<uint32_t>(mine));
      const uint32_t key = static_cast<uint32_t>(mine >> 32);
      if (rank == 0) s3[0] = key;
      if (rank == i_hi) s3[1] = key;
      if (rank == i_lo) s3[2] = key;
      if (dg) {
        if (rank == i_2k) s3[3] = key;
        srt[rank] = key;
      }
    }
  }
  if (need <= 0) release_keys(release_bar, lane);
  if (lane == 0) {
    row_out[0] = 0;
    if (W > 1) row_out[1] = (t > 0) ? t : NB;
  }
  const int filled = f + need < 2 * k ? f + need : 2 * k;
  for (int slot = filled + lane; slot < W; slot += 32)
    if (slot >= 2) row_out[slot] = NB;
  __syncwarp();
  float sig = 1.0f;  // G5: nothing is dropped
  if (t + 1 > k) {
    const float s_0 = unkey(s3[0]), s_hi = unkey(s3[1]), s_lo = unkey(s3[2]);   // s~[f], s~[k-1], s~[k]
    const float num = s_hi - s_lo, den = s_0 - s_lo;
    sig = (den == 0.0f) ? 0.0f : __fdiv_rn(num, den);                            // L324
  }
  if (dg) {
    const float nan = __int_as_float(0x7fc00000);
    DiagCell c = {nan, nan, nan, nan};
    if (t + 1 >= 2 * k + 1) {                    // rho*k + 1 visible blocks (L493): need == want
      const float s_0 = unkey(s3[0]), s_hi = unkey(s3[1]), s_lo = unkey(s3[2]), s_2k = unkey(s3[3]);
      c.g = s_hi - s_lo;
      c.G = s_hi - s_2k;
      c.r = s_0 - s_lo;
      float mn = INFINITY;                        // secondary spacings, free ranks j | j+1 (A1, L431)
      for (int j = lane; j + 1 < need; j += 32)
        if (j != k - 1 - f) mn = fminf(mn, unkey(srt[j]) - unkey(srt[j + 1]));
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) mn = fminf(mn, __shfl_xor_sync(0xffffffffu, mn, off));
      c.d2 = mn;
    }
    *dg = c;
    __syncwarp();
  }
  return sig;
}

}  // namespace bsa

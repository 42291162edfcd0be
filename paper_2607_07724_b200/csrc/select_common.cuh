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

constexpr int kMaxCand = 256;  // 2 * k_budget <= 256

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

// One warp.  keys[0..t] = order-preserving keys (okey) of the tile scores of the visible blocks, in
// shared memory.  Writes the first W slots of the sorted row [0, t, free blocks by (score desc, index
// asc)], padded with NB, and returns sigma (Eq.4 / Eq.11; G1, G5).  s3 = 3 words of scratch.
// `release_bar`: mbarrier (shared-memory address, or 0) that receives exactly one arrival as soon as
// keys[] has been consumed, so that the buffer can be refilled while the selection continues.
static __device__ float warp_select(const uint32_t* keys, int t, int k, int NB, int W, int32_t* row_out,
                                    unsigned long long* cand, uint32_t* s3, int lane,
                                    uint32_t release_bar = 0u) {
  const int f = (t == 0) ? 1 : 2;               // forced: sink, self (Eq.9)
  const int n_free = (t >= 2) ? t - 1 : 0;      // blocks 1 .. t-1
  const int want = 2 * k - f;
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
    } else {
      warp_topk_compact<128>(keys, n_free, need, cand, lane, release_bar);
    }
    __syncwarp();
    // order by rank: the (key, ~block) words are distinct, so rank = #{cand > mine} is a permutation
    const int i_hi = k - 1 - f, i_lo = k - f;   // ranks of s~[k-1] and s~[k] in the free list
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
    }
  }
  if (need <= 0) release_keys(release_bar, lane);
  if (lane == 0) {
    row_out[0] = 0;
    if (W > 1) row_out[1] = (t > 0) ? t : NB;
  }
  for (int slot = f + need + lane; slot < W; slot += 32)
    if (slot >= 2) row_out[slot] = NB;
  __syncwarp();
  float sig = 1.0f;  // G5: nothing is dropped
  if (t + 1 > k) {
    const float s_0 = unkey(s3[0]), s_hi = unkey(s3[1]), s_lo = unkey(s3[2]);   // s~[f], s~[k-1], s~[k]
    const float num = s_hi - s_lo, den = s_0 - s_lo;
    sig = (den == 0.0f) ? 0.0f : __fdiv_rn(num, den);                            // L324
  }
  return sig;
}

}  // namespace bsa

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

// One warp.  sc[0..t] = tile scores of the visible blocks (shared memory).  Writes the first W slots
// of the sorted row [0, t, free blocks by (score desc, index asc)], padded with NB, and returns sigma.
static __device__ float warp_select(const float* sc, int t, int k, int NB, int W, int32_t* row_out,
                             unsigned long long* cand, int lane) {
  const unsigned full = 0xffffffffu;
  const int f = (t == 0) ? 1 : 2;               // forced: sink, self (Eq.9)
  const int n_free = (t >= 2) ? t - 1 : 0;      // blocks 1 .. t-1
  const int want = 2 * k - f;
  const int need = want < n_free ? want : n_free;
  if (need > 0) {
    const bool all = (n_free <= need);
    uint32_t vth = 0;
    int r_eq = 0;
    if (!all) {
      // largest v with |{key >= v}| >= need  ==  the need-th largest key
      uint32_t prefix = 0;
      for (int bit = 31; bit >= 0; --bit) {
        const uint32_t c = prefix | (1u << bit);
        int cnt = 0;
        for (int i = lane; i < n_free; i += 32) cnt += (okey(sc[1 + i]) >= c) ? 1 : 0;
        cnt = __reduce_add_sync(full, cnt);
        if (cnt >= need) prefix = c;
      }
      vth = prefix;
      int cgt = 0;
      for (int i = lane; i < n_free; i += 32) cgt += (okey(sc[1 + i]) > vth) ? 1 : 0;
      cgt = __reduce_add_sync(full, cgt);
      r_eq = need - cgt;  // ties at the threshold: the r_eq lowest block indices win (G6)
    }
    int base = 0, eq_seen = 0;
    const unsigned lt = (1u << lane) - 1u;
    for (int i0 = 0; i0 < n_free; i0 += 32) {
      const int i = i0 + lane;
      const bool valid = i < n_free;
      const uint32_t key = valid ? okey(sc[1 + i]) : 0u;
      const bool gt = valid && (all || key > vth);
      const bool eq = valid && !all && key == vth;
      const unsigned be = __ballot_sync(full, eq);
      const bool take_eq = eq && (eq_seen + __popc(be & lt) < r_eq);
      const unsigned bsel = __ballot_sync(full, gt || take_eq);
      if (gt || take_eq)
        cand[base + __popc(bsel & lt)] =
            (static_cast<unsigned long long>(key) << 32) | (0xFFFFFFFFu - static_cast<uint32_t>(1 + i));
      base += __popc(bsel);
      eq_seen += __popc(be);
    }
    int P = 1;
    while (P < need) P <<= 1;
    for (int q = need + lane; q < P; q += 32) cand[q] = 0ull;  // sorts last
    __syncwarp();
    // bitonic network, descending: (score desc, block index asc)
    for (int size = 2; size <= P; size <<= 1) {
      for (int stride = size >> 1; stride > 0; stride >>= 1) {
        for (int q = lane; q < (P >> 1); q += 32) {
          const int i = ((q / stride) * (stride << 1)) + (q % stride), j = i + stride;
          const unsigned long long a = cand[i], c = cand[j];
          const bool desc = ((i & size) == 0);
          if (desc ? (a < c) : (a > c)) { cand[i] = c; cand[j] = a; }
        }
        __syncwarp();
      }
    }
  }
  float sig = 1.0f;  // G5: nothing is dropped
  if (t + 1 > k) {
    const float s_hi = unkey(static_cast<uint32_t>(cand[k - 1 - f] >> 32));  // s~[k-1]
    const float s_lo = unkey(static_cast<uint32_t>(cand[k - f] >> 32));      // s~[k]
    const float s_0 = unkey(static_cast<uint32_t>(cand[0] >> 32));           // s~[f]  (G1)
    const float num = s_hi - s_lo, den = s_0 - s_lo;
    sig = (den == 0.0f) ? 0.0f : __fdiv_rn(num, den);                        // L324
  }
  if (lane == 0) {
    row_out[0] = 0;
    if (W > 1) row_out[1] = (t > 0) ? t : NB;
  }
  for (int q = lane; q + 2 < W; q += 32) {
    const int slot = q + 2, fi = slot - f;  // index into the sorted free list
    int v = NB;
    if (t > 0 && fi < need) v = static_cast<int>(0xFFFFFFFFu - static_cast<uint32_t>(cand[fi]));
    row_out[slot] = v;
  }
  return sig;
}

}  // namespace bsa

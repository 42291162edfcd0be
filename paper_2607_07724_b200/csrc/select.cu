// select.cu -- bsa_select: per-(Q-tile, head) block scoring, causal top-k with forced sink / self,
// normalised cutoff margin sigma, head mean, per-layer q-quantile trigger and the shape-uniform
// padded kv_idx (Eq.1-5; A.2-A.9 L296-340; readings G1-G17 in DESIGN.md).
//
// Kernels
//   score_select_kernel : one CTA per (tile t, head h, batch).  Tile scores of the visible blocks
//                         (Eq.3: max over the tile's rows of Eq.1 / Eq.2) are kept in shared memory
//                         only; warp 0 then selects the top-(2k) by a bit-wise bisection on the
//                         order-preserving integer image of the fp32 score (ties -> lower block
//                         index), sorts the survivors with a shared-memory bitonic network, and
//                         emits the sorted prefix into kv_idx plus sigma (Eq.4 / Eq.11).
//   route_kernel        : one CTA per sequence: sigma_bar (Eq.12), device radix-select of the
//                         ceil(qT)-th smallest sigma_bar (Eq.5 / Eq.13), trigger.
//   finalize_kernel     : Eq.14: untriggered tiles keep k entries, the rest becomes the sentinel.
#include <cuda_bf16.h>

#include "bsa_internal.h"

namespace bsa {

namespace {

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
__device__ float warp_select(const float* sc, int t, int k, int NB, int W, int32_t* row_out,
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

// ---- SIMT fp32 scoring + selection ---------------------------------------------------------------
constexpr int kScoreThreads = 256;

template <int D, int BN, bool QUEST>
__global__ void __launch_bounds__(kScoreThreads)
score_select_kernel(const uint16_t* __restrict__ Q, int64_t qsb, int64_t qsh, int64_t qsn,
                    const float* __restrict__ kmean, const uint16_t* __restrict__ kmin,
                    const uint16_t* __restrict__ kmax, int H, int Hkv, int G, int NB, int k, int W,
                    int router, float inv_sqrt_d, int32_t* __restrict__ kv_idx,
                    int32_t* __restrict__ kv_count, float* __restrict__ sigma) {
  constexpr int ROWS = BN / 32;
  constexpr int QSTRIDE = D * 2 + 16;  // bytes; +16 keeps 16-byte row reads conflict free
  extern __shared__ __align__(16) uint8_t sm[];
  uint8_t* qs = sm;                                                   // [BN][QSTRIDE]
  float* sc = reinterpret_cast<float*>(sm + BN * QSTRIDE);           // [NB]
  unsigned long long* cand = reinterpret_cast<unsigned long long*>(sc + ((NB + 1) & ~1));

  const int per_tile = gridDim.y;  // B*H
  const int t = NB - 1 - static_cast<int>(blockIdx.x);  // heaviest tile first
  const int bh = blockIdx.y;
  (void)per_tile;
  const int b = bh / H, h = bh % H, g = h / G;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  // Q tile -> shared memory (bf16, padded rows)
  const uint16_t* qbase = Q + b * qsb + h * qsh + static_cast<int64_t>(t) * BN * qsn;
  for (int i = tid; i < BN * (D / 8); i += kScoreThreads) {
    const int r = i / (D / 8), c = i % (D / 8);
    *reinterpret_cast<uint4*>(qs + r * QSTRIDE + c * 16) =
        *reinterpret_cast<const uint4*>(qbase + static_cast<int64_t>(r) * qsn + c * 8);
  }
  __syncthreads();

  const size_t mrow0 = (static_cast<size_t>(b) * Hkv + g) * NB;
  for (int blk = warp; blk <= t; blk += kScoreThreads / 32) {
    float acc[ROWS];
#pragma unroll
    for (int rr = 0; rr < ROWS; ++rr) acc[rr] = 0.f;
    const size_t mo = (mrow0 + blk) * D;
#pragma unroll 4
    for (int c = 0; c < D; c += 8) {
      float ka[8], kb[8];
      if (QUEST) {
        const uint4 vx = *reinterpret_cast<const uint4*>(kmax + mo + c);
        const uint4 vn = *reinterpret_cast<const uint4*>(kmin + mo + c);
        const uint32_t wx[4] = {vx.x, vx.y, vx.z, vx.w}, wn[4] = {vn.x, vn.y, vn.z, vn.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          ka[2 * i] = __uint_as_float(wx[i] << 16);
          ka[2 * i + 1] = __uint_as_float(wx[i] & 0xFFFF0000u);
          kb[2 * i] = __uint_as_float(wn[i] << 16);
          kb[2 * i + 1] = __uint_as_float(wn[i] & 0xFFFF0000u);
        }
      } else {
        const float4 a0 = *reinterpret_cast<const float4*>(kmean + mo + c);
        const float4 a1 = *reinterpret_cast<const float4*>(kmean + mo + c + 4);
        ka[0] = a0.x; ka[1] = a0.y; ka[2] = a0.z; ka[3] = a0.w;
        ka[4] = a1.x; ka[5] = a1.y; ka[6] = a1.z; ka[7] = a1.w;
      }
#pragma unroll
      for (int rr = 0; rr < ROWS; ++rr) {
        const uint4 qv = *reinterpret_cast<const uint4*>(qs + (lane + 32 * rr) * QSTRIDE + c * 2);
        const uint32_t qw[4] = {qv.x, qv.y, qv.z, qv.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const float q0 = __uint_as_float(qw[i] << 16), q1 = __uint_as_float(qw[i] & 0xFFFF0000u);
          if (QUEST) {  // Eq.2: sum_c max(q_c Kmax_c, q_c Kmin_c); the products are exact in fp32
            acc[rr] += fmaxf(q0 * ka[2 * i], q0 * kb[2 * i]);
            acc[rr] += fmaxf(q1 * ka[2 * i + 1], q1 * kb[2 * i + 1]);
          } else {      // Eq.1: q . kbar
            acc[rr] = fmaf(q0, ka[2 * i], acc[rr]);
            acc[rr] = fmaf(q1, ka[2 * i + 1], acc[rr]);
          }
        }
      }
    }
    float mx = acc[0];
#pragma unroll
    for (int rr = 1; rr < ROWS; ++rr) mx = fmaxf(mx, acc[rr]);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, off));
    if (lane == 0) sc[blk] = QUEST ? mx : mx * inv_sqrt_d;  // Eq.3 tile max (scale is monotone, G8)
  }
  __syncthreads();

  if (warp == 0) {
    const int64_t row = (static_cast<int64_t>(b) * H + h) * NB + t;
    const float sig = warp_select(sc, t, k, NB, W, kv_idx + row * W, cand, lane);
    if (lane == 0) {
      sigma[row] = sig;
      if (!router) kv_count[row] = (k < t + 1) ? k : t + 1;
    }
  }
}

// ---- sigma_bar, quantile, trigger ---------------------------------------------------------------
constexpr int kRouteThreads = 1024;

__global__ void __launch_bounds__(kRouteThreads)
route_kernel(const float* __restrict__ sigma, int H, int T, int router, long long m,
             float* __restrict__ sigma_bar, uint8_t* __restrict__ trigger, float* __restrict__ tau) {
  extern __shared__ uint32_t rk[];  // keys[T], then hist[256], then 2 scratch words
  uint32_t* keys = rk;
  uint32_t* hist = rk + T;
  uint32_t* scratch = hist + 256;
  const int b = blockIdx.x, tid = threadIdx.x;
  for (int t = tid; t < T; t += kRouteThreads) {
    float acc = 0.0f;
    for (int h = 0; h < H; ++h) acc = acc + sigma[(static_cast<size_t>(b) * H + h) * T + t];  // Eq.12
    const float sb = __fdiv_rn(acc, static_cast<float>(H));
    sigma_bar[static_cast<size_t>(b) * T + t] = sb;
    keys[t] = okey(sb);
  }
  __syncthreads();
  if (!router || m <= 0) {
    for (int t = tid; t < T; t += kRouteThreads) trigger[static_cast<size_t>(b) * T + t] = 0;
    if (tid == 0 && tau) tau[b] = -1.0f;
    return;
  }
  // MSB-first 8-bit radix select of the m-th smallest key (1-indexed order statistic, G3)
  uint32_t prefix = 0, mask = 0;
  uint32_t remaining = static_cast<uint32_t>(m);
  for (int shift = 24; shift >= 0; shift -= 8) {
    if (tid < 256) hist[tid] = 0;
    __syncthreads();
    for (int t = tid; t < T; t += kRouteThreads) {
      const uint32_t kk = keys[t];
      if ((kk & mask) == prefix) atomicAdd(&hist[(kk >> shift) & 255u], 1u);
    }
    __syncthreads();
    if (tid == 0) {
      uint32_t cum = 0, d = 0;
      for (; d < 256; ++d) {
        if (cum + hist[d] >= remaining) break;
        cum += hist[d];
      }
      scratch[0] = d;
      scratch[1] = remaining - cum;
    }
    __syncthreads();
    prefix |= scratch[0] << shift;
    mask |= 255u << shift;
    remaining = scratch[1];
    __syncthreads();
  }
  for (int t = tid; t < T; t += kRouteThreads)
    trigger[static_cast<size_t>(b) * T + t] = (keys[t] <= prefix) ? 1 : 0;  // sigma_bar <= tau (Eq.5)
  if (tid == 0 && tau) tau[b] = unkey(prefix);
}

// ---- Eq.14 for the router policies: W = 2k ------------------------------------------------------
__global__ void finalize_kernel(const uint8_t* __restrict__ trigger, int H, int T, int NB, int k,
                                int32_t* __restrict__ kv_idx, int32_t* __restrict__ kv_count,
                                long long rows) {
  const long long i = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  const long long row = i / k;
  const int j = static_cast<int>(i % k);
  if (row >= rows) return;
  const int t = static_cast<int>(row % T);
  const long long b = row / (static_cast<long long>(T) * H);
  const bool trig = trigger[b * T + t] != 0;
  if (!trig) kv_idx[row * (2 * k) + k + j] = NB;
  if (j == 0) {
    const int budget = trig ? 2 * k : k;
    kv_count[row] = budget < t + 1 ? budget : t + 1;
  }
}

template <int D, int BN, bool QUEST>
bsa_status run_score(const Dims& S, const void* Q, const char* meta, const MetaLayout& L, int k, int W,
                     int router, int32_t* kv_idx, int32_t* kv_count, float* sigma,
                     cudaStream_t stream) {
  const size_t smem = static_cast<size_t>(BN) * (D * 2 + 16) + ((S.NB + 1) & ~1) * 4 + kMaxCand * 8;
  auto kern = score_select_kernel<D, BN, QUEST>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       static_cast<int>(smem));
  if (e != cudaSuccess) return fail(BSA_ERR_CUDA, "select: smem attribute: %s", cudaGetErrorString(e));
  dim3 grid(S.NB, S.B * S.H);
  const float inv_sqrt_d = static_cast<float>(1.0 / sqrt(static_cast<double>(S.d)));
  kern<<<grid, kScoreThreads, smem, stream>>>(
      static_cast<const uint16_t*>(Q), S.qsb, S.qsh, S.qsn,
      reinterpret_cast<const float*>(meta + L.off_mean),
      reinterpret_cast<const uint16_t*>(meta + L.off_min),
      reinterpret_cast<const uint16_t*>(meta + L.off_max), S.H, S.Hkv, S.G, S.NB, k, W, router,
      inv_sqrt_d, kv_idx, kv_count, sigma);
  return check_launch("score_select_kernel");
}

}  // namespace

bsa_status launch_select(const Dims& S, const void* Q, const void* meta, int policy, int k, int W,
                         long long m_route, int32_t* kv_idx, int32_t* kv_count, float* sigma,
                         float* sigma_bar, uint8_t* trigger, float* tau, cudaStream_t stream) {
  const MetaLayout L = meta_layout(S);
  const char* mp = static_cast<const char*>(meta);
  const bool quest = (policy == BSA_POLICY_QUEST || policy == BSA_POLICY_ROUTER_QUEST);
  const int router = (policy == BSA_POLICY_ROUTER || policy == BSA_POLICY_ROUTER_QUEST) ? 1 : 0;
  if (S.B * S.H > 65535) return fail(BSA_ERR_UNSUPPORTED, "select: batch*heads > 65535");
  bsa_status st = BSA_ERR_UNSUPPORTED;
#define BSA_SC(DD, BB)                                                                              \
  if (S.d == DD && S.Bn == BB)                                                                      \
    st = quest ? run_score<DD, BB, true>(S, Q, mp, L, k, W, router, kv_idx, kv_count, sigma, stream) \
               : run_score<DD, BB, false>(S, Q, mp, L, k, W, router, kv_idx, kv_count, sigma, stream);
  BSA_SC(64, 64) BSA_SC(128, 64) BSA_SC(256, 64) BSA_SC(64, 128) BSA_SC(128, 128) BSA_SC(256, 128)
#undef BSA_SC
  if (st == BSA_ERR_UNSUPPORTED)
    return fail(BSA_ERR_UNSUPPORTED, "select: unsupported head_dim %d / block %d", S.d, S.Bn);
  if (st != BSA_OK) return st;

  const size_t rsmem = (static_cast<size_t>(S.NB) + 256 + 2) * 4;
  route_kernel<<<S.B, kRouteThreads, rsmem, stream>>>(sigma, S.H, S.NB, router, m_route, sigma_bar,
                                                      trigger, tau);
  st = check_launch("route_kernel");
  if (st != BSA_OK) return st;
  if (router) {
    const long long rows = static_cast<long long>(S.B) * S.H * S.NB;
    const long long total = rows * k;
    const int threads = 256;
    finalize_kernel<<<static_cast<unsigned>((total + threads - 1) / threads), threads, 0, stream>>>(
        trigger, S.H, S.NB, S.NB, k, kv_idx, kv_count, rows);
    st = check_launch("finalize_kernel");
  }
  return st;
}

}  // namespace bsa

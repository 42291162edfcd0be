// select.cu -- bsa_select: per-(Q-tile, head) block scoring, causal top-k with forced sink / self,
// normalised cutoff margin sigma, head mean, per-layer q-quantile trigger and the shape-uniform
// padded kv_idx (Eq.1-5; A.2-A.9 L296-340; readings G1-G17 in DESIGN.md).
//
// Kernels
//   score_tc_kernel (score_tc.cuh) : tensor-core tile scores (Eq.1-3), top-(2k) and sigma (Eq.4 /
//                         Eq.11) per (tile, head); writes all 2k / k slots of kv_idx and sigma.
//   route_kernel        : one CTA per sequence: sigma_bar (Eq.12), device radix-select of the
//                         ceil(qT)-th smallest sigma_bar (Eq.5 / Eq.13), trigger.
//   finalize_kernel     : Eq.14: untriggered tiles keep k entries, the rest becomes the sentinel.
#include <cuda_bf16.h>

#include "bsa_internal.h"
#include "select_common.cuh"
#include "sm100_ptx.cuh"

namespace bsa {

namespace {

// ---- sigma_bar, quantile, trigger ---------------------------------------------------------------
constexpr int kRouteThreads = 1024;

__global__ void __launch_bounds__(kRouteThreads)
route_kernel(const float* __restrict__ sigma, int H, int T, int router, long long m,
             float* __restrict__ sigma_bar, uint8_t* __restrict__ trigger, float* __restrict__ tau) {
  griddep_launch();   // a dependent attention launch may start its prologue now (it waits for our completion)
  extern __shared__ uint32_t rk[];  // keys[T], then hist[256], then 2 scratch words
  uint32_t* keys = rk;
  uint32_t* hist = rk + T;
  uint32_t* scratch = hist + 256;
  const int b = blockIdx.x, tid = threadIdx.x;
  for (int t = tid; t < T; t += kRouteThreads) {
    float acc = 0.0f;
#pragma unroll 8
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
    if (tid < 32) {
      // warp 0 locates the digit: 8 bins per lane, warp-inclusive scan of the lane sums, then the
      // one lane whose range crosses `remaining` walks its 8 bins
      uint32_t v[8], sum = 0;
#pragma unroll
      for (int d = 0; d < 8; ++d) {
        v[d] = hist[tid * 8 + d];
        sum += v[d];
      }
      uint32_t incl = sum;
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) {
        const uint32_t up = __shfl_up_sync(0xffffffffu, incl, off);
        if (tid >= off) incl += up;
      }
      const unsigned hit = __ballot_sync(0xffffffffu, incl >= remaining);
      if (tid == __ffs(hit) - 1) {
        uint32_t cum = incl - sum;
        int d = 0;
        for (; d < 7; ++d) {
          if (cum + v[d] >= remaining) break;
          cum += v[d];
        }
        scratch[0] = static_cast<uint32_t>(tid * 8 + d);
        scratch[1] = remaining - cum;
      }
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
  griddep_launch();
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

}  // namespace

bsa_status launch_select(const Dims& S, const void* Q, const void* meta, int policy, int k, int W,
                         long long m_route, int32_t* kv_idx, int32_t* kv_count, float* sigma,
                         float* sigma_bar, uint8_t* trigger, float* tau, const SelectDiag& dg,
                         cudaStream_t stream) {
  const bool quest = (policy == BSA_POLICY_QUEST || policy == BSA_POLICY_ROUTER_QUEST);
  const int router = (policy == BSA_POLICY_ROUTER || policy == BSA_POLICY_ROUTER_QUEST) ? 1 : 0;
  bsa_status st = quest ? launch_score_tc_quest(S, Q, meta, k, W, router, kv_idx, kv_count, sigma, dg, stream)
                        : launch_score_tc_mean(S, Q, meta, k, W, router, kv_idx, kv_count, sigma, dg, stream);
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
    if (st != BSA_OK) return st;
  }
  if (dg.g && dg.summary) st = launch_diag_summary(S, k, router && m_route > 0, tau, dg, stream);
  return st;
}

}  // namespace bsa

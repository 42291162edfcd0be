// diag.cu -- per-layer aggregation of the D.4 diagnostics (App. D.4, Eq.18,
// assumptions (A1)/(A2) L431-432, Remark 1 L480, Proposition 1) from the per-cell quantities the
// selection kernel emits on chip (select_common.cuh: g, G, r, d2; score_tc.cuh: rough).
//
// One CTA per sequence.  Population = the cells (t, h) with at least rho*k + 1 visible blocks (L493:
// "masked to causally-valid tiles with >= rho k + 1 visible blocks"), i.e. t >= 2k; n = H * (T - 2k).
//   summary[0]  n                     number of cells
//   summary[1]  r_bar                 mean_t r_t                                  (A2)
//   summary[2]  CV(r)                 sqrt(Var_t r_t) / r_bar, population variance (A2) -- proxy of beta
//   summary[3]  sigma_(q)             the threshold the router uses (tau of Eq.5);  NaN for non-router
//   summary[4]  gamma_q               sigma_(q) * r_bar                            (Proposition 1)
//   summary[5]  m_q(beta)             fraction of cells with g in gamma_q [1-beta, 1+beta], beta = CV(r)
//   summary[6]  Delta_2 10 % quantile of d2 (order statistic ceil(p n - 1e-9), as reading G3)  (A1)
//   summary[7]  Delta_2 median
//   summary[8]  tau_hat               sqrt( sum rough / (2 * #pairs) ) over ALL (t, h): E[(s_{i+1,b} -
//                                     s_{i,b})^2] = 2 tau^2 for adjacent rows i, i+1 of a tile (step 3)
//   summary[9]  fraction of cells with g == 0 (the "atom" of L501)
//   summary[10] g_q^+                 40th percentile of g on {g > 0}               (L501)
//   summary[11] g_q^+ / tau_hat
// Sums run in double in a fixed order (thread-strided partials, then a shared-memory tree), so the
// result does not depend on scheduling.
#include "bsa_internal.h"
#include "select_common.cuh"

namespace bsa {

namespace {

constexpr int kDiagThreads = 1024;

__device__ double cta_sum(double v, double* red) {
  const int tid = threadIdx.x;
  red[tid] = v;
  __syncthreads();
  for (int s = kDiagThreads / 2; s > 0; s >>= 1) {
    if (tid < s) red[tid] += red[tid + s];
    __syncthreads();
  }
  const double r = red[0];
  __syncthreads();
  return r;
}

// m-th smallest (1-indexed) of the keys key(i), i in [0, total), restricted to the cells with use(i).
// MSB-first 8-bit radix select; every thread returns the key.
template <class Key, class Use>
__device__ uint32_t cta_select(int total, long long m, Key key, Use use, uint32_t* hist, uint32_t* scratch) {
  const int tid = threadIdx.x;
  uint32_t prefix = 0, mask = 0;
  uint32_t remaining = static_cast<uint32_t>(m);
  for (int shift = 24; shift >= 0; shift -= 8) {
    if (tid < 256) hist[tid] = 0;
    __syncthreads();
    for (int i = tid; i < total; i += kDiagThreads) {
      if (!use(i)) continue;
      const uint32_t kk = key(i);
      if ((kk & mask) == prefix) atomicAdd(&hist[(kk >> shift) & 255u], 1u);
    }
    __syncthreads();
    if (tid == 0) {
      uint32_t cum = 0;
      int d = 0;
      for (; d < 255; ++d) {
        if (cum + hist[d] >= remaining) break;
        cum += hist[d];
      }
      scratch[0] = static_cast<uint32_t>(d);
      scratch[1] = remaining - cum;
    }
    __syncthreads();
    prefix |= scratch[0] << shift;
    mask |= 255u << shift;
    remaining = scratch[1];
    __syncthreads();
  }
  return prefix;
}

__device__ __forceinline__ long long order_index(double p, long long n) {  // ceil(p n - 1e-9) in [1, n]
  long long m = static_cast<long long>(ceil(p * static_cast<double>(n) - 1e-9));
  return m < 1 ? 1 : (m > n ? n : m);
}

__global__ void __launch_bounds__(kDiagThreads)
diag_summary_kernel(const float* __restrict__ g, const float* __restrict__ r, const float* __restrict__ d2,
                    const float* __restrict__ rough, const float* __restrict__ tau, int H, int T, int k,
                    int Bn, int router, float* __restrict__ summary) {
  __shared__ double red[kDiagThreads];
  __shared__ uint32_t hist[256];
  __shared__ uint32_t scratch[2];
  const int b = blockIdx.x, tid = threadIdx.x;
  const size_t base = static_cast<size_t>(b) * H * T;
  g += base; r += base; d2 += base; rough += base;
  float* out = summary + static_cast<size_t>(b) * BSA_DIAG_SUMMARY_LEN;
  const int total = H * T;
  const int t_min = 2 * k;                       // cells with >= rho k + 1 visible blocks
  const long long n = (T > t_min) ? static_cast<long long>(H) * (T - t_min) : 0;
  auto valid = [&](int i) { return (i % T) >= t_min; };
  const float nanf_ = __int_as_float(0x7fc00000);

  // tau_hat over all cells: pairs of adjacent rows per (t, h) = (t + 1) * (Bn - 1)
  double rs = 0.0;
  for (int i = tid; i < total; i += kDiagThreads) rs += static_cast<double>(rough[i]);
  rs = cta_sum(rs, red);
  const double pairs = static_cast<double>(H) * (static_cast<double>(T) * (T + 1) / 2.0) * (Bn - 1);
  const double tau_hat = sqrt(rs / (2.0 * pairs));

  if (n == 0) {
    if (tid == 0) {
      for (int i = 0; i < BSA_DIAG_SUMMARY_LEN; ++i) out[i] = nanf_;
      out[0] = 0.0f;
      out[8] = static_cast<float>(tau_hat);
    }
    return;
  }
  double acc = 0.0;
  for (int i = tid; i < total; i += kDiagThreads)
    if (valid(i)) acc += static_cast<double>(r[i]);
  const double r_bar = cta_sum(acc, red) / static_cast<double>(n);
  acc = 0.0;
  for (int i = tid; i < total; i += kDiagThreads)
    if (valid(i)) {
      const double dv = static_cast<double>(r[i]) - r_bar;
      acc += dv * dv;
    }
  const double var = cta_sum(acc, red) / static_cast<double>(n);
  const double cv = sqrt(var) / r_bar;
  const double sigma_q = router ? static_cast<double>(tau[b]) : nan("");
  const double gamma = sigma_q * r_bar;
  const double lo = gamma * (1.0 - cv), hi = gamma * (1.0 + cv);
  double in_band = 0.0, zero = 0.0, pos = 0.0;
  for (int i = tid; i < total; i += kDiagThreads)
    if (valid(i)) {
      const double gv = static_cast<double>(g[i]);
      in_band += (router && gv >= lo && gv <= hi) ? 1.0 : 0.0;
      zero += (gv == 0.0) ? 1.0 : 0.0;
      pos += (gv > 0.0) ? 1.0 : 0.0;
    }
  in_band = cta_sum(in_band, red);
  zero = cta_sum(zero, red);
  pos = cta_sum(pos, red);
  const uint32_t k10 = cta_select(total, order_index(0.10, n), [&](int i) { return okey(d2[i]); }, valid, hist, scratch);
  const uint32_t k50 = cta_select(total, order_index(0.50, n), [&](int i) { return okey(d2[i]); }, valid, hist, scratch);
  const long long n_pos = static_cast<long long>(pos);
  float gq = nanf_;
  if (n_pos > 0) {
    const uint32_t kg = cta_select(total, order_index(0.40, n_pos), [&](int i) { return okey(g[i]); },
                                   [&](int i) { return valid(i) && g[i] > 0.0f; }, hist, scratch);
    gq = unkey(kg);
  }
  if (tid == 0) {
    out[0] = static_cast<float>(n);
    out[1] = static_cast<float>(r_bar);
    out[2] = static_cast<float>(cv);
    out[3] = router ? tau[b] : nanf_;
    out[4] = static_cast<float>(gamma);
    out[5] = router ? static_cast<float>(in_band / static_cast<double>(n)) : nanf_;
    out[6] = unkey(k10);
    out[7] = unkey(k50);
    out[8] = static_cast<float>(tau_hat);
    out[9] = static_cast<float>(zero / static_cast<double>(n));
    out[10] = gq;
    out[11] = static_cast<float>(static_cast<double>(gq) / tau_hat);
    for (int i = 12; i < BSA_DIAG_SUMMARY_LEN; ++i) out[i] = 0.0f;
  }
}

}  // namespace

bsa_status launch_diag_summary(const Dims& S, int k, int router, const float* tau, const SelectDiag& dg,
                               cudaStream_t stream) {
  diag_summary_kernel<<<S.B, kDiagThreads, 0, stream>>>(dg.g, dg.r, dg.d2, dg.rough, tau, S.H, S.NB, k, S.Bn,
                                                        router, dg.summary);
  return check_launch("diag_summary_kernel");
}

}  // namespace bsa

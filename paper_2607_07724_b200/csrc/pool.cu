// pool.cu -- bsa_build_block_meta: per-KV-block key pooling (Eq.1 / Eq.6 L74, L293 for the
// mean; Eq.2 L78-80 for the element-wise min / max).
//
// HBM-bound: K is read exactly once with 128-bit non-allocating loads; one CTA per (batch, KV head,
// block).  The block sum is accumulated in fp64 (exact for bf16 inputs, hence order independent) and
// rounded once, so kmean is the correctly rounded fp32 mean.  Besides kmean / kmin / kmax the kernel
// writes the exact 3-way bf16 split of kmean (hi + mid + lo == kmean) used by tensor-core scoring.
#include <cuda_bf16.h>

#include "bsa_internal.h"

namespace bsa {

namespace {

__device__ __forceinline__ uint4 ld_stream(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ float bf_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf_hi(uint32_t w) { return __uint_as_float(w & 0xFFFF0000u); }
__device__ __forceinline__ uint16_t f2bf_exact(float f) {  // f is exactly representable in bf16
  return static_cast<uint16_t>(__float_as_uint(f) >> 16);
}
__device__ __forceinline__ uint16_t f2bf_rn(float f) {
  return __bfloat16_as_ushort(__float2bfloat16_rn(f));
}

// Error-free fp32 addition (Knuth TwoSum): s + e == a + b exactly.
__device__ __forceinline__ void two_sum(float a, float b, float& s, float& e) {
  s = __fadd_rn(a, b);
  const float bb = __fsub_rn(s, a);
  e = __fadd_rn(__fsub_rn(a, __fsub_rn(s, bb)), __fsub_rn(b, bb));
}
__device__ __forceinline__ uint32_t bf2_min(uint32_t a, uint32_t b) {
  uint32_t r;
  asm("min.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
  return r;
}
__device__ __forceinline__ uint32_t bf2_max(uint32_t a, uint32_t b) {
  uint32_t r;
  asm("max.bf16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
  return r;
}

constexpr int kPasses = 8;  // key rows per thread: 8 x 16 B = 128 B in flight per thread

// One CTA of BN*D/64 threads per (batch, KV head, block).  Thread (r0, c8) owns 8 adjacent
// columns of rows r0, r0 + RPP, ..., all 8 loads issued before the first use.  The column sum is
// exact: a TwoSum chain in fp32 carries the running sum, and the (almost always zero) rounding
// errors of the chain are detected with one OR; only a thread that saw a non-zero error re-adds
// its 8 rows in fp64.  Partial sums are then combined across threads in fp64 (exact for bf16
// inputs), so the mean is the correctly rounded fp32 mean whatever the order -- without paying an
// fp32->fp64 conversion (XU pipe, quarter rate) per element.
template <int D, int BN>
__global__ void __launch_bounds__(BN* D / 64, 768 / (BN * D / 64)) pool_kernel(const uint16_t* __restrict__ K, int64_t ksb,
                                                         int64_t ksh, int64_t ksn, int NB, int Hkv,
                                                         int kinds, float* __restrict__ kmean,
                                                         uint16_t* __restrict__ kmin,
                                                         uint16_t* __restrict__ kmax,
                                                         uint16_t* __restrict__ ksplit,
                                                         size_t plane_elems) {
  constexpr int kThreads = BN * D / 64;
  constexpr int TPR = D / 8;            // threads per key row (8 bf16 = 16 B each)
  constexpr int RPP = kThreads / TPR;   // rows per pass
  static_assert(RPP * kPasses == BN, "thread count must give exactly kPasses rows per thread");
  const int blk = blockIdx.x, g = blockIdx.y, b = blockIdx.z;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int c8 = tid % TPR, r0 = tid / TPR;

  const uint16_t* base = K + b * ksb + g * ksh + static_cast<int64_t>(blk) * BN * ksn + c8 * 8;
  uint4 v[kPasses];
#pragma unroll
  for (int p = 0; p < kPasses; ++p)
    v[p] = ld_stream(reinterpret_cast<const uint4*>(base + static_cast<int64_t>(r0 + p * RPP) * ksn));

  float hi[8];
  uint32_t mn2[4], mx2[4];
  {
    const uint32_t w[4] = {v[0].x, v[0].y, v[0].z, v[0].w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      hi[2 * i] = bf_lo(w[i]);
      hi[2 * i + 1] = bf_hi(w[i]);
      mn2[i] = w[i];
      mx2[i] = w[i];
    }
  }
  uint32_t err_bits = 0;
#pragma unroll
  for (int p = 1; p < kPasses; ++p) {
    const uint32_t w[4] = {v[p].x, v[p].y, v[p].z, v[p].w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      float e0, e1;
      two_sum(hi[2 * i], bf_lo(w[i]), hi[2 * i], e0);
      two_sum(hi[2 * i + 1], bf_hi(w[i]), hi[2 * i + 1], e1);
      err_bits |= __float_as_uint(e0) | __float_as_uint(e1);
      mn2[i] = bf2_min(mn2[i], w[i]);
      mx2[i] = bf2_max(mx2[i], w[i]);
    }
  }
  double sum[8];
  if ((err_bits << 1) != 0) {  // some fp32 add was inexact (an error of -0 does not count): redo in fp64
#pragma unroll
    for (int i = 0; i < 8; ++i) sum[i] = 0.0;
#pragma unroll
    for (int p = 0; p < kPasses; ++p) {
      const uint32_t w[4] = {v[p].x, v[p].y, v[p].z, v[p].w};
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        sum[2 * i] += static_cast<double>(bf_lo(w[i]));
        sum[2 * i + 1] += static_cast<double>(bf_hi(w[i]));
      }
    }
  } else {
#pragma unroll
    for (int i = 0; i < 8; ++i) sum[i] = static_cast<double>(hi[i]);
  }
  float mn[8], mx[8];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    mn[2 * i] = bf_lo(mn2[i]);
    mn[2 * i + 1] = bf_hi(mn2[i]);
    mx[2 * i] = bf_lo(mx2[i]);
    mx[2 * i + 1] = bf_hi(mx2[i]);
  }
  // rows that live in the same warp (lanes that differ by a multiple of TPR)
#pragma unroll
  for (int off = 16; off >= TPR; off >>= 1) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      sum[i] += __shfl_xor_sync(0xffffffffu, sum[i], off);
      mn[i] = fminf(mn[i], __shfl_xor_sync(0xffffffffu, mn[i], off));
      mx[i] = fmaxf(mx[i], __shfl_xor_sync(0xffffffffu, mx[i], off));
    }
  }
  constexpr int NW = kThreads / 32;
  constexpr int CW = (TPR <= 32) ? 1 : TPR / 32;   // warps that cover one key row
  constexpr int NR = NW / CW;                       // partial results per column
  __shared__ double s_sum[NR][D];
  __shared__ uint16_t s_mn[NR][D], s_mx[NR][D];
  constexpr int LPW = (TPR < 32) ? TPR : 32;  // distinct column groups per warp
  if (lane < LPW) {
    const int col = c8 * 8;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      s_sum[warp / CW][col + i] = sum[i];
      s_mn[warp / CW][col + i] = f2bf_exact(mn[i]);
      s_mx[warp / CW][col + i] = f2bf_exact(mx[i]);
    }
  }
  __syncthreads();
  for (int c = tid; c < D; c += kThreads) {
    double s = 0.0;
    float lo = INFINITY, hv = -INFINITY;
#pragma unroll
    for (int w = 0; w < NR; ++w) {
      s += s_sum[w][c];
      lo = fminf(lo, __uint_as_float(static_cast<uint32_t>(s_mn[w][c]) << 16));
      hv = fmaxf(hv, __uint_as_float(static_cast<uint32_t>(s_mx[w][c]) << 16));
    }
    const size_t o = ((static_cast<size_t>(b) * Hkv + g) * NB + blk) * D + c;
    if (kinds & BSA_META_MEAN) {
      const float mean = static_cast<float>(s / static_cast<double>(BN));  // Eq.1, rounded once
      kmean[o] = mean;
      const uint16_t h1 = f2bf_rn(mean);
      const float r1 = mean - __uint_as_float(static_cast<uint32_t>(h1) << 16);
      const uint16_t h2 = f2bf_rn(r1);
      const float r2 = r1 - __uint_as_float(static_cast<uint32_t>(h2) << 16);
      const uint16_t h3 = f2bf_rn(r2);
      ksplit[o] = h1;
      ksplit[plane_elems + o] = h2;
      ksplit[2 * plane_elems + o] = h3;
    }
    if (kinds & BSA_META_MINMAX) {
      kmin[o] = f2bf_exact(lo);
      kmax[o] = f2bf_exact(hv);
    }
  }
}

template <int D, int BN>
void launch(const Dims& S, const void* K, int kinds, char* meta, const MetaLayout& L,
            cudaStream_t stream) {
  dim3 grid(S.NB, S.Hkv, S.B);
  pool_kernel<D, BN><<<grid, BN * D / 64, 0, stream>>>(
      static_cast<const uint16_t*>(K), S.ksb, S.ksh, S.ksn, S.NB, S.Hkv, kinds,
      reinterpret_cast<float*>(meta + L.off_mean), reinterpret_cast<uint16_t*>(meta + L.off_min),
      reinterpret_cast<uint16_t*>(meta + L.off_max), reinterpret_cast<uint16_t*>(meta + L.off_split),
      L.elems);
}

}  // namespace

bsa_status launch_pool(const Dims& S, const void* K, int kinds, void* meta, cudaStream_t stream) {
  const MetaLayout L = meta_layout(S);
  char* m = static_cast<char*>(meta);
#define BSA_POOL_CASE(DD, BB) \
  if (S.d == DD && S.Bn == BB) { launch<DD, BB>(S, K, kinds, m, L, stream); return check_launch("pool_kernel"); }
  BSA_POOL_CASE(64, 64)
  BSA_POOL_CASE(128, 64)
  BSA_POOL_CASE(256, 64)
  BSA_POOL_CASE(64, 128)
  BSA_POOL_CASE(128, 128)
  BSA_POOL_CASE(256, 128)
#undef BSA_POOL_CASE
  return fail(BSA_ERR_UNSUPPORTED, "pool: unsupported head_dim %d / block %d", S.d, S.Bn);
}

}  // namespace bsa

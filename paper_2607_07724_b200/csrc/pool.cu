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

constexpr int kThreads = 256;

template <int D, int BN>
__global__ void __launch_bounds__(kThreads) pool_kernel(const uint16_t* __restrict__ K, int64_t ksb,
                                                        int64_t ksh, int64_t ksn, int NB, int Hkv,
                                                        int kinds, float* __restrict__ kmean,
                                                        uint16_t* __restrict__ kmin,
                                                        uint16_t* __restrict__ kmax,
                                                        uint16_t* __restrict__ ksplit,
                                                        size_t plane_elems) {
  constexpr int TPR = D / 8;            // threads per key row (8 bf16 = 16 B each)
  constexpr int RPP = kThreads / TPR;   // rows per pass
  constexpr int PASSES = BN / RPP;
  static_assert(BN % RPP == 0, "block must be a multiple of the rows per pass");
  const int blk = blockIdx.x, g = blockIdx.y, b = blockIdx.z;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int c8 = tid % TPR, r0 = tid / TPR;

  const uint16_t* base = K + b * ksb + g * ksh + static_cast<int64_t>(blk) * BN * ksn + c8 * 8;
  uint4 v[PASSES];
#pragma unroll
  for (int p = 0; p < PASSES; ++p)
    v[p] = ld_stream(reinterpret_cast<const uint4*>(base + static_cast<int64_t>(r0 + p * RPP) * ksn));

  double sum[8];
  float mn[8], mx[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { sum[i] = 0.0; mn[i] = INFINITY; mx[i] = -INFINITY; }
#pragma unroll
  for (int p = 0; p < PASSES; ++p) {
    const uint32_t w[4] = {v[p].x, v[p].y, v[p].z, v[p].w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      float a = bf_lo(w[i]), c = bf_hi(w[i]);
      sum[2 * i] += static_cast<double>(a);
      sum[2 * i + 1] += static_cast<double>(c);
      mn[2 * i] = fminf(mn[2 * i], a);
      mx[2 * i] = fmaxf(mx[2 * i], a);
      mn[2 * i + 1] = fminf(mn[2 * i + 1], c);
      mx[2 * i + 1] = fmaxf(mx[2 * i + 1], c);
    }
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
  __shared__ double s_sum[NW][D];
  __shared__ float s_mn[NW][D], s_mx[NW][D];
  constexpr int LPW = (TPR < 32) ? TPR : 32;  // distinct column groups per warp
  if (lane < LPW) {
    const int col = (TPR <= 32 ? lane : c8) * 8;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      s_sum[warp][col + i] = sum[i];
      s_mn[warp][col + i] = mn[i];
      s_mx[warp][col + i] = mx[i];
    }
  }
  __syncthreads();
  if (tid < D) {
    double s = 0.0;
    float lo = INFINITY, hi = -INFINITY;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      s += s_sum[w][tid];
      lo = fminf(lo, s_mn[w][tid]);
      hi = fmaxf(hi, s_mx[w][tid]);
    }
    const size_t o = ((static_cast<size_t>(b) * Hkv + g) * NB + blk) * D + tid;
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
      kmax[o] = f2bf_exact(hi);
    }
  }
}

template <int D, int BN>
void launch(const Dims& S, const void* K, int kinds, char* meta, const MetaLayout& L,
            cudaStream_t stream) {
  dim3 grid(S.NB, S.Hkv, S.B);
  pool_kernel<D, BN><<<grid, kThreads, 0, stream>>>(
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

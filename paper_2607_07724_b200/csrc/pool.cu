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

#ifndef BSA_POOL_TPS
#define BSA_POOL_TPS 768
#endif
// packed fp32x2 adds with directed rounding (FADD2.RP / FADD2.RM): one issue slot for both halves of a word
__device__ __forceinline__ float2 fadd2_ru(float2 a, float2 b) {
  float2 d;
  asm("{\n\t.reg .b64 ra, rb, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\t"
      "add.rp.f32x2 rd, ra, rb;\n\tmov.b64 {%0, %1}, rd;\n\t}"
      : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
  return d;
}
__device__ __forceinline__ float2 fadd2_rd(float2 a, float2 b) {
  float2 d;
  asm("{\n\t.reg .b64 ra, rb, rd;\n\tmov.b64 ra, {%2, %3};\n\tmov.b64 rb, {%4, %5};\n\t"
      "add.rm.f32x2 rd, ra, rb;\n\tmov.b64 {%0, %1}, rd;\n\t}"
      : "=f"(d.x), "=f"(d.y) : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
  return d;
}

constexpr int kPasses = 8;  // key rows per thread: 8 x 16 B = 128 B in flight per thread

// CTAs of BN*D/64 threads; thread (r0, c8) owns 8 adjacent columns of rows r0, r0 + RPP, ... of a
// block (8 x 16 B loads).  The per-thread column sums run in fp32 with a two-adds-per-element
// exactness test (see process_block); only a thread whose test fails re-adds its 8 rows in fp64.
// Partial sums are combined across threads in fp64 (exact for bf16 inputs), so the mean is the
// correctly rounded fp32 mean whatever the order -- without an fp32->fp64 conversion (XU pipe,
// quarter rate) per element.  min / max stay packed bf16x2 until the last step.
template <int D, int BN>
struct PoolArgs {
  const uint16_t* K;
  int64_t ksb, ksh, ksn;
  int NB, Hkv, B, kinds;
  int dfull;   // head_dim; a CTA covers D of its columns, starting at blockIdx.y * D
  float* kmean;
  uint16_t *kmin, *kmax, *ksplit;
  size_t plane_elems;
};

// work item w -> (batch b, KV head g, block blk); rows r0 + p*RPP of that block, 8 columns at c8*8
template <int D, int BN>
__device__ __forceinline__ void load_block(const PoolArgs<D, BN>& a, int w, uint4 (&v)[kPasses]) {
  constexpr int kThreads = BN * D / 64, TPR = D / 8, RPP = kThreads / TPR;
  const int blk = w % a.NB, g = (w / a.NB) % a.Hkv, b = w / (a.NB * a.Hkv);
  const int c8 = threadIdx.x % TPR, r0 = threadIdx.x / TPR;
  const uint16_t* base = a.K + b * a.ksb + g * a.ksh + static_cast<int64_t>(blk) * BN * a.ksn + c8 * 8 +
                         blockIdx.y * D;
#pragma unroll
  for (int p = 0; p < kPasses; ++p)
    v[p] = ld_stream(reinterpret_cast<const uint4*>(base + static_cast<int64_t>(r0 + p * RPP) * a.ksn));
}

template <int D, int BN>
__device__ __forceinline__ void process_block(const PoolArgs<D, BN>& a, int w, const uint4 (&v)[kPasses]) {
  constexpr int kThreads = BN * D / 64;
  constexpr int TPR = D / 8;            // threads per key row (8 bf16 = 16 B each)
  constexpr int RPP = kThreads / TPR;   // rows per pass
  static_assert(RPP * kPasses == BN, "thread count must give exactly kPasses rows per thread");
  const int blk = w % a.NB, g = (w / a.NB) % a.Hkv, b = w / (a.NB * a.Hkv);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int c8 = tid % TPR;
  const int NB = a.NB, Hkv = a.Hkv, kinds = a.kinds;
  float* __restrict__ kmean = a.kmean;
  uint16_t* __restrict__ kmin = a.kmin;
  uint16_t* __restrict__ kmax = a.kmax;
  uint16_t* __restrict__ ksplit = a.ksplit;
  const size_t plane_elems = a.plane_elems;

  // Exactness test that costs two adds per element: the same chain is run once rounding every add
  // up and once rounding it down.  ru >= exact >= rd holds inductively, and the first inexact add
  // opens a gap that later adds can only keep (RU(a' + y) >= a' + y > a + y >= RD(a + y) for
  // a' > a), so ru == rd at the end  <=>  every add was exact  <=>  ru is the exact column sum.
  float ru[8], rd[8];
  uint32_t mn2[4], mx2[4];
  {
    const uint32_t w[4] = {v[0].x, v[0].y, v[0].z, v[0].w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      ru[2 * i] = rd[2 * i] = bf_lo(w[i]);
      ru[2 * i + 1] = rd[2 * i + 1] = bf_hi(w[i]);
      mn2[i] = w[i];
      mx2[i] = w[i];
    }
  }
#pragma unroll
  for (int p = 1; p < kPasses; ++p) {
    const uint32_t w[4] = {v[p].x, v[p].y, v[p].z, v[p].w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float2 x = make_float2(bf_lo(w[i]), bf_hi(w[i]));
      const float2 u = fadd2_ru(make_float2(ru[2 * i], ru[2 * i + 1]), x);
      const float2 dn = fadd2_rd(make_float2(rd[2 * i], rd[2 * i + 1]), x);
      ru[2 * i] = u.x;
      ru[2 * i + 1] = u.y;
      rd[2 * i] = dn.x;
      rd[2 * i + 1] = dn.y;
      mn2[i] = bf2_min(mn2[i], w[i]);
      mx2[i] = bf2_max(mx2[i], w[i]);
    }
  }
  bool exact = true;
#pragma unroll
  for (int i = 0; i < 8; ++i) exact = exact && (ru[i] == rd[i]);
  double sum[8];
  if (!exact) {  // some fp32 add was inexact: redo this thread's rows in fp64
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
    for (int i = 0; i < 8; ++i) sum[i] = static_cast<double>(ru[i]);
  }
  // rows that live in the same warp (lanes that differ by a multiple of TPR)
#pragma unroll
  for (int off = 16; off >= TPR; off >>= 1) {
#pragma unroll
    for (int i = 0; i < 8; ++i) sum[i] += __shfl_xor_sync(0xffffffffu, sum[i], off);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      mn2[i] = bf2_min(mn2[i], __shfl_xor_sync(0xffffffffu, mn2[i], off));
      mx2[i] = bf2_max(mx2[i], __shfl_xor_sync(0xffffffffu, mx2[i], off));
    }
  }
  constexpr int NW = kThreads / 32;
  constexpr int CW = (TPR <= 32) ? 1 : TPR / 32;   // warps that cover one key row
  constexpr int NR = NW / CW;                       // partial results per column
  __shared__ double s_sum[NR][D];
  __shared__ uint32_t s_mn[NR][D / 2], s_mx[NR][D / 2];  // bf16x2
  constexpr int LPW = (TPR < 32) ? TPR : 32;  // distinct column groups per warp
  if (lane < LPW) {
    const int col = c8 * 8;
#pragma unroll
    for (int i = 0; i < 8; ++i) s_sum[warp / CW][col + i] = sum[i];
    *reinterpret_cast<uint4*>(&s_mn[warp / CW][col / 2]) = make_uint4(mn2[0], mn2[1], mn2[2], mn2[3]);
    *reinterpret_cast<uint4*>(&s_mx[warp / CW][col / 2]) = make_uint4(mx2[0], mx2[1], mx2[2], mx2[3]);
  }
  __syncthreads();
  for (int c = tid; c < D; c += kThreads) {
    double s = 0.0;
    float lo = INFINITY, hv = -INFINITY;
#pragma unroll
    for (int w = 0; w < NR; ++w) {
      s += s_sum[w][c];
      const uint32_t wn = s_mn[w][c >> 1], wx = s_mx[w][c >> 1];
      lo = fminf(lo, (c & 1) ? bf_hi(wn) : bf_lo(wn));
      hv = fmaxf(hv, (c & 1) ? bf_hi(wx) : bf_lo(wx));
    }
    const size_t o = ((static_cast<size_t>(b) * Hkv + g) * NB + blk) * a.dfull + blockIdx.y * D + c;
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
__global__ void __launch_bounds__(BN* D / 64, BSA_POOL_TPS / (BN * D / 64)) pool_kernel(const PoolArgs<D, BN> a) {
  uint4 v[kPasses];
  load_block<D, BN>(a, static_cast<int>(blockIdx.x), v);
  process_block<D, BN>(a, static_cast<int>(blockIdx.x), v);
}

template <int D, int BN>
void launch(const Dims& S, const void* K, int kinds, char* meta, const MetaLayout& L,
            cudaStream_t stream) {
  PoolArgs<D, BN> a;
  a.K = static_cast<const uint16_t*>(K);
  a.ksb = S.ksb; a.ksh = S.ksh; a.ksn = S.ksn;
  a.NB = S.NB; a.Hkv = S.Hkv; a.B = S.B; a.kinds = kinds;
  a.dfull = S.d;
  a.kmean = reinterpret_cast<float*>(meta + L.off_mean);
  a.kmin = reinterpret_cast<uint16_t*>(meta + L.off_min);
  a.kmax = reinterpret_cast<uint16_t*>(meta + L.off_max);
  a.ksplit = reinterpret_cast<uint16_t*>(meta + L.off_split);
  a.plane_elems = L.elems;
  constexpr int kThreads = BN * D / 64;
  const int total = S.NB * S.Hkv * S.B;
  // one block per CTA: with ~6 CTAs resident per SM their load and reduce phases interleave; a
  // persistent register-double-buffered variant measured 25 % slower (fewer warps to hide the adds)
  // head_dim 256 runs as two 128-column halves (blockIdx.y): 512-thread CTAs at 128 registers left one
  // CTA of 16 warps per SM (ncu r02: 22.8 % occupancy, 3.1 TB/s); the halves are the d = 128 kernel
  pool_kernel<D, BN><<<dim3(total, S.d / D), kThreads, 0, stream>>>(a);
}

}  // namespace

bsa_status launch_pool(const Dims& S, const void* K, int kinds, void* meta, cudaStream_t stream) {
  const MetaLayout L = meta_layout(S);
  char* m = static_cast<char*>(meta);
#define BSA_POOL_CASE(DD, BB) \
  if (S.d == DD && S.Bn == BB) { launch<DD, BB>(S, K, kinds, m, L, stream); return check_launch("pool_kernel"); }
  BSA_POOL_CASE(64, 64)
  BSA_POOL_CASE(128, 64)
  if (S.d == 256 && S.Bn == 64) { launch<128, 64>(S, K, kinds, m, L, stream); return check_launch("pool_kernel"); }
  BSA_POOL_CASE(64, 128)
  BSA_POOL_CASE(128, 128)
  if (S.d == 256 && S.Bn == 128) { launch<128, 128>(S, K, kinds, m, L, stream); return check_launch("pool_kernel"); }
#undef BSA_POOL_CASE
  return fail(BSA_ERR_UNSUPPORTED, "pool: unsupported head_dim %d / block %d", S.d, S.Bn);
}

}  // namespace bsa

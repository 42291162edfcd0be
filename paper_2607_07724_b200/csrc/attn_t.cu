// attn_t.cu -- sparse attention for 64-token blocks and head_dim 128 in the TRANSPOSED formulation
// (PAPER.md L43-47 softmax definition, L131 / A.10 L342 iteration over kv_idx).
//
// Why: a (Q tile, head) problem has 64 query rows, so S = Q K^T is a UMMA with M = 64, which runs the
// tensor pipe at half rate (sm100_ptx.cuh table: M=64,N=64 32 clk, M=64,N=128 64 clk per K=16 step).  Here
// the KEYS are the M dimension instead, two selected blocks at a time:
//     S^T[128 keys, 64 queries]  = [K_a; K_b] . Q^T        M = 128, N = 64, K = d      (48 clk per step)
//     O^T[128 d,    64 queries] += [V_a; V_b]^T . P^T      M = 128, N = 64, K = 128 keys (48 clk per step)
// i.e. 768 clk of tensor pipe per 128 keys instead of 1024.  Consequences of having the keys on the TMEM
// lanes (thread = key) instead of the queries:
//   * the softmax reference maximum m_ref[q] lives in shared memory and is only a REFERENCE (lazy
//     rescale): p = 2^(s*scale - m_ref[q]).  A CTA-wide vote (bar.red.or) per iteration asks whether any
//     logit exceeds its reference by more than 2^8; only then are the true column maxima reduced across
//     lanes (64 redux per warp + a shared-memory exchange), O^T and the partial sums rescaled;
//   * the row sums l[q] = sum_keys p are kept as per-lane PARTIAL sums in spare TMEM columns (64 columns:
//     tcgen05.ld / add / tcgen05.st per iteration) and reduced across the 128 lanes once per tile;
//   * P^T is written [key][query] -- 128 contiguous bytes per thread -- which is exactly the MN-major B
//     operand of the second product; V tiles [key][d] are its MN-major A operand, unchanged from TMA;
//   * the epilogue transposes O^T through shared memory.
// An odd number of selected blocks is padded with a masked dummy half (no loads, p = 0).
//
// One CTA per (tile, head) and ONE CTA per SM (a 128-key iteration moves 64 KB of K / V; hiding the TMA
// latency needs ~3 iterations in flight, which two CTAs x 113 KB cannot hold -- measured: 2.3 ms at C2
// with two CTAs and 5 ring units each, against 1.5 ms for the M = 64 kernel).  12 warps:
//   0-7  softmax: warp w owns TMEM lanes 32 (w % 4) .. +31 (keys) and query columns 32 (w / 4) .. +31
//   8    TMA producer of the K ring (6 units), 9 TMA producer of the V ring (5 units)
//   10   QK issue (one iteration ahead of the softmax, S^T double buffered), 11 PV issue
// P^T is double buffered, so the softmax of iteration j+1 does not wait for PV(j).  K and V have separate
// rings of 16 KB units, each with a single producer and a single in-order consumer (see attn.cu on why):
// a K unit is one 64-column slab of BOTH blocks (rows 0-63 = block a, 64-127 = block b: the M = 128
// A operand needs them adjacent), a V unit is one block.
#include <cuda_bf16.h>

#include "bsa_internal.h"
#include "sm100_ptx.cuh"
#include "tmap.h"

namespace bsa {

namespace {

constexpr int TD = 128;                 // head_dim
constexpr int TB = 64;                  // block = Q tile rows
constexpr int kTThreads = 384;
constexpr int kTSoft = 256;              // softmax threads
constexpr int kTMaxW = 256;
constexpr int UNIT = 16384;             // ring unit
constexpr int NKU = 6, NVU = 5;         // K / V ring units
constexpr int T_Q_BYTES = TB * TD * 2;  // 16 KB
constexpr int T_P_BYTES = 128 * TB * 2; // P^T [128 keys][64 queries] bf16 = 16 KB
constexpr int T_SMEM = T_Q_BYTES + 2 * T_P_BYTES + (NKU + NVU) * UNIT + 1024;
static_assert(T_SMEM <= 232448, "one CTA per SM");
// TMEM columns: S^T double buffered [0,64) [64,128); O^T [128,192); partial row sums [192,256)
constexpr uint32_t S_COL = 0, O_COL = 128, L_COL = 192, T_TMEM_COLS = 256;

struct TParams {
  const int32_t* kv_idx;
  const int32_t* kv_count;
  uint16_t* O;
  float* lse;
  int W, B, H, G, N, NB;
  int64_t qsb, qsh, qsn;
  float scale_log2;
};

struct alignas(16) TCtl {
  float mref[TB];        // reference maxima (log2 units); 1 / l in the epilogue
  uint64_t q_full, p_full[2], o_done[2];
  uint64_t s_full[2], s_free[2];
  uint64_t k_full[NKU], k_empty[NKU], v_full[NVU], v_empty[NVU];
  uint32_t tmem_base;
  int32_t n_valid;
  uint16_t list[kTMaxW];
};
static_assert(sizeof(TCtl) <= 1024, "TCtl must fit the 1 KB bookkeeping area");
// Scratch of the slow path inside the P^T buffer about to be written (free once PV(j-1) is done):
//   float wmax[4][64] at byte 0 (per-warp column maxima), float alpha[64] at byte 1024

__device__ __forceinline__ void bar_sm() { asm volatile("bar.sync 1, 256;" ::: "memory"); }
__device__ __forceinline__ bool bar_or(bool pred) {   // barrier 2 over the 256 softmax threads + OR
  uint32_t r;
  asm volatile(
      "{\n\t.reg .pred p, q;\n\tsetp.ne.b32 p, %1, 0;\n\t"
      "barrier.cta.red.or.pred q, 2, 256, p;\n\tselp.u32 %0, 1, 0, q;\n\t}"
      : "=r"(r) : "r"(static_cast<uint32_t>(pred)) : "memory");
  return r != 0;
}
__device__ __forceinline__ uint32_t fkey(float x) {   // order-preserving float -> uint (ascending)
  const uint32_t u = __float_as_uint(x);
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float funkey(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k ^ 0x80000000u) : ~k);
}
// 32x32b.x16: thread i of warp w <- TMEM lane 32*(w%4)+i, 16 consecutive columns
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
      "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
      "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
      : "memory");
}

// ---- softmax warps (0-7): thread = (key lane kl, 32-query half cg) of the 128-key iteration ----------
__device__ __forceinline__ void t_softmax(const TParams& p, TCtl* ctl, uint8_t* p_s, uint8_t* ring_s,
                                          uint32_t tmem, int n_blk, int tq, int b, int h) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int quad = warp & 3, cg = warp >> 2;               // TMEM lane quadrant, query-column half
  const int kl = quad * 32 + lane, half = kl >> 6, kk = kl & 63;
  const int qb = cg * 32;                                   // first query column of this thread
  const uint32_t lane_base = static_cast<uint32_t>(quad * 32) << 16;
  const float sc = p.scale_log2;
  const int n_it = (n_blk + 1) >> 1;
  const float ninf = -INFINITY;

  {   // partial row sums start at zero
    uint32_t z[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) z[i] = 0u;
    tmem_st16(tmem + lane_base + L_COL + qb, z);
    tmem_st16(tmem + lane_base + L_COL + qb + 16, z);
    tmem_st_wait();
  }
  if (tid < TB) ctl->mref[tid] = ninf;
  bar_sm();

  for (int j = 0; j < n_it; ++j) {
    const bool has_b = 2 * j + 1 < n_blk;
    const int my_blk = half ? (has_b ? ctl->list[2 * j + 1] : -1) : ctl->list[2 * j];
    const bool dummy = my_blk < 0;                        // padded half: no keys
    const bool diag = my_blk == tq;                       // causal mask inside the self block
    const uint32_t tS = tmem + lane_base + S_COL + (j & 1) * 64 + qb;
    uint8_t* pbuf = p_s + (j & 1) * T_P_BYTES;
    float* wmax = reinterpret_cast<float*>(pbuf);         // [4 quadrants][64]  slow-path scratch
    float* alpha = reinterpret_cast<float*>(pbuf + 1024); // [64]
    mbar_wait(smem_u32(&ctl->s_full[j & 1]), (j >> 1) & 1);
    tc_fence_after();

    // ---- optimistic pass: p = 2^(s*scale - m_ref) with the current references, and the largest
    // exponent seen; the P^T row stays in registers until the vote has passed ------------------------
    uint32_t pk[16];
    float tmax = ninf;
    auto compute_p = [&]() {
      uint32_t x0[16], x1[16];
      tmem_ld16(tS, x0);
      tmem_ld16(tS + 16, x1);
      tmem_ld_wait();
      tmax = ninf;
#pragma unroll
      for (int i4 = 0; i4 < 32; i4 += 4) {
        const float4 mr = *reinterpret_cast<const float4*>(&ctl->mref[qb + i4]);
        const float m4[4] = {mr.x, mr.y, mr.z, mr.w};
        float e4[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const int q = qb + i4 + e;
          const uint32_t xv = (i4 + e < 16) ? x0[(i4 + e) & 15] : x1[(i4 + e) & 15];
          const float t = fmaf(__uint_as_float(xv), sc, -m4[e]);
          const bool masked = diag && kk > q;
          tmax = masked ? tmax : fmaxf(tmax, t);
          e4[e] = masked ? 0.0f : ex2_approx(t);
        }
        pk[i4 >> 1] = pack_bf16x2(e4[0], e4[1]);
        pk[(i4 >> 1) + 1] = pack_bf16x2(e4[2], e4[3]);
      }
    };
#ifdef T_ABL_NOSOFTMAX
#pragma unroll
    for (int i = 0; i < 16; ++i) pk[i] = 0x3c003c00u;
    const bool slow = false;
    if (j == 0 && tid < TB) ctl->mref[tid] = 0.0f;
#else
    if (j > 0 && !dummy) compute_p();                     // j == 0: no reference yet, always slow
    const bool slow = (j == 0) ? true : bar_or(tmax > 8.0f);
#endif
    if (slow) {
      // ---- slow path: true column maxima -> new references, rescale O^T and the partial sums ------
      if (j > 0) {                                        // every earlier PV done: O^T and P^T scratch are ours
        mbar_wait(smem_u32(&ctl->o_done[(j - 1) & 1]), ((j - 1) >> 1) & 1);
        tc_fence_after();
      }
      {
        uint32_t x0[16], x1[16];
        tmem_ld16(tS, x0);
        tmem_ld16(tS + 16, x1);
        tmem_ld_wait();
        uint32_t mine = 0u;
#pragma unroll
        for (int i = 0; i < 32; ++i) {
          const int q = qb + i;
          const uint32_t xv = (i < 16) ? x0[i & 15] : x1[i & 15];
          const float v = (dummy || (diag && kk > q)) ? ninf : __uint_as_float(xv) * sc;
          const uint32_t mx = __reduce_max_sync(0xffffffffu, fkey(v));
          if (lane == i) mine = mx;
        }
        wmax[quad * TB + qb + lane] = funkey(mine);
      }
      bar_sm();
      if (tid < TB) {
        const float m_old = ctl->mref[tid];
        const float m_new = fmaxf(fmaxf(m_old, fmaxf(wmax[tid], wmax[TB + tid])),
                                  fmaxf(wmax[2 * TB + tid], wmax[3 * TB + tid]));
        alpha[tid] = (m_old == ninf) ? 0.0f : ex2_approx(m_old - m_new);
        ctl->mref[tid] = m_new;
      }
      bar_sm();
      if (j > 0) {
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          uint32_t o[16], l[16];
          tmem_ld16(tmem + lane_base + O_COL + qb + c * 16, o);
          tmem_ld16(tmem + lane_base + L_COL + qb + c * 16, l);
          tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 16; ++i) {
            const float a = alpha[qb + c * 16 + i];
            o[i] = __float_as_uint(__uint_as_float(o[i]) * a);
            l[i] = __float_as_uint(__uint_as_float(l[i]) * a);
          }
          tmem_st16(tmem + lane_base + O_COL + qb + c * 16, o);
          tmem_st16(tmem + lane_base + L_COL + qb + c * 16, l);
        }
        tmem_st_wait();
      }
      bar_sm();   // wmax / alpha scratch is read by everyone before P^T overwrites it
      if (!dummy) compute_p();                            // with the new references
    }
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(smem_u32(&ctl->s_free[j & 1]));   // S^T(j) has been read
    if (j >= 2) {                                                 // PV(j-2) done: this P^T buffer is ours
      mbar_wait(smem_u32(&ctl->o_done[j & 1]), ((j >> 1) & 1) ^ 1);
      tc_fence_after();
    }
    if (!dummy) {
      // P^T row `kl`, queries qb .. qb+31 = 64 B: MN-major B operand, 128B swizzle (chunk c at c ^ (row & 7))
      uint8_t* prow = pbuf + kl * 128;
#pragma unroll
      for (int c = 0; c < 4; ++c)
        *reinterpret_cast<uint4*>(prow + (((cg * 4 + c) ^ (kl & 7)) << 4)) =
            make_uint4(pk[4 * c], pk[4 * c + 1], pk[4 * c + 2], pk[4 * c + 3]);
    }
    fence_proxy_async_smem();
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(smem_u32(&ctl->p_full[j & 1]));
    // partial row sums of the bf16-rounded p (what the numerator uses), under the PV product
#ifndef T_ABL_NOLSUM
    if (!dummy) {
      uint32_t l0[16], l1[16];
      tmem_ld16(tmem + lane_base + L_COL + qb, l0);
      tmem_ld16(tmem + lane_base + L_COL + qb + 16, l1);
      tmem_ld_wait();
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const uint32_t w0 = pk[i], w1 = pk[8 + i];
        l0[2 * i] = __float_as_uint(__uint_as_float(l0[2 * i]) + __uint_as_float(w0 << 16));
        l0[2 * i + 1] = __float_as_uint(__uint_as_float(l0[2 * i + 1]) + __uint_as_float(w0 & 0xFFFF0000u));
        l1[2 * i] = __float_as_uint(__uint_as_float(l1[2 * i]) + __uint_as_float(w1 << 16));
        l1[2 * i + 1] = __float_as_uint(__uint_as_float(l1[2 * i + 1]) + __uint_as_float(w1 & 0xFFFF0000u));
      }
      tmem_st16(tmem + lane_base + L_COL + qb, l0);
      tmem_st16(tmem + lane_base + L_COL + qb + 16, l1);
      tmem_st_wait();
    }
#endif
  }

  // ---- epilogue -----------------------------------------------------------------------------------
  mbar_wait(smem_u32(&ctl->o_done[(n_it - 1) & 1]), ((n_it - 1) >> 1) & 1);
  if (n_it >= 2) mbar_wait(smem_u32(&ctl->o_done[n_it & 1]), ((n_it - 2) >> 1) & 1);
  tc_fence_after();
  float* scr = reinterpret_cast<float*>(ring_s);          // [128 lanes][65]: the rings are idle now
  {
    uint32_t l0[16], l1[16];
    tmem_ld16(tmem + lane_base + L_COL + qb, l0);
    tmem_ld16(tmem + lane_base + L_COL + qb + 16, l1);
    tmem_ld_wait();
#pragma unroll
    for (int i = 0; i < 16; ++i) {
      scr[kl * 65 + qb + i] = __uint_as_float(l0[i]);
      scr[kl * 65 + qb + 16 + i] = __uint_as_float(l1[i]);
    }
  }
  bar_sm();
  const int q0 = tq * TB;
  if (tid < TB) {
    float l = 0.0f;
    for (int r = 0; r < 128; ++r) l += scr[r * 65 + tid];
    const int qrow = q0 + tid;
    if (p.lse && qrow < p.N)
      p.lse[(static_cast<int64_t>(b) * p.H + h) * p.N + qrow] = (ctl->mref[tid] + log2f(l)) * 0.6931471805599453f;
    ctl->mref[tid] = 1.0f / l;
  }
  bar_sm();
  uint16_t* stage = reinterpret_cast<uint16_t*>(p_s);     // O tile [64 queries][128 d] bf16 (d = TMEM lane)
  {
    uint32_t o0[16], o1[16];
    tmem_ld16(tmem + lane_base + O_COL + qb, o0);
    tmem_ld16(tmem + lane_base + O_COL + qb + 16, o1);
    tmem_ld_wait();
#pragma unroll
    for (int i = 0; i < 32; ++i) {
      const int q = qb + i;
      const float v = __uint_as_float(i < 16 ? o0[i & 15] : o1[i & 15]) * ctl->mref[q];
      stage[q * TD + kl] = __bfloat16_as_ushort(__float2bfloat16_rn(v));
    }
  }
  tc_fence_before();
  bar_sm();
  {   // 64 rows x 256 B: four threads per row, 64 B (4 x 16 B) each
    const int r = tid >> 2, part = tid & 3, qrow = q0 + r;
    if (qrow < p.N) {
      const uint4* src = reinterpret_cast<const uint4*>(stage + r * TD + part * 32);
      uint4* dst = reinterpret_cast<uint4*>(p.O + b * p.qsb + h * p.qsh + static_cast<int64_t>(qrow) * p.qsn + part * 32);
#pragma unroll
      for (int c = 0; c < 4; ++c) dst[c] = src[c];
    }
  }
}

__global__ void __launch_bounds__(kTThreads, 1)
attn_t_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
              const __grid_constant__ CUtensorMap tmV, const TParams p) {
  extern __shared__ __align__(1024) uint8_t smem[];
  uint8_t* q_s = smem;
  uint8_t* p_s = smem + T_Q_BYTES;
  uint8_t* ring_s = p_s + 2 * T_P_BYTES;             // K units, then V units
  TCtl* ctl = reinterpret_cast<TCtl*>(ring_s + (NKU + NVU) * UNIT);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  int wi = static_cast<int>(blockIdx.x);             // same work order as attn.cu
  const int hi = wi % p.G;
  wi /= p.G;
  const int tq = p.NB - 1 - wi % p.NB;
  wi /= p.NB;
  const int Hkv = p.H / p.G;
  const int g = wi % Hkv, b = wi / Hkv, h = g * p.G + hi;
  const int q0 = tq * TB;
  if ((smem_u32(smem) & 1023u) != 0) __trap();

  if (warp == 8) {
    if (lane == 0) {
      mbar_init(smem_u32(&ctl->q_full), 1);
      for (int i = 0; i < 2; ++i) {
        mbar_init(smem_u32(&ctl->p_full[i]), 8);
        mbar_init(smem_u32(&ctl->o_done[i]), 1);
        mbar_init(smem_u32(&ctl->s_full[i]), 1);
        mbar_init(smem_u32(&ctl->s_free[i]), 8);
      }
      for (int s = 0; s < NKU; ++s) {
        mbar_init(smem_u32(&ctl->k_full[s]), 1);
        mbar_init(smem_u32(&ctl->k_empty[s]), 1);
      }
      for (int s = 0; s < NVU; ++s) {
        mbar_init(smem_u32(&ctl->v_full[s]), 1);
        mbar_init(smem_u32(&ctl->v_empty[s]), 1);
      }
      fence_mbar_init();
      mbar_arrive_expect_tx(smem_u32(&ctl->q_full), T_Q_BYTES);
      tma_load_5d(smem_u32(q_s), &tmQ, smem_u32(&ctl->q_full), 0, q0, 0, h, b);
      tma_prefetch_desc(&tmK);
      tma_prefetch_desc(&tmV);
    }
    __syncwarp();
    tmem_alloc<T_TMEM_COLS>(smem_u32(&ctl->tmem_base));
  }
  if (warp == 0) {
    // compact the valid entries of this kv_idx row (sentinel, blocks > t and duplicates skipped)
    const int64_t row = (static_cast<int64_t>(b) * p.H + h) * p.NB + tq;
    int cnt = p.kv_count ? p.kv_count[row] : p.W;
    cnt = cnt < 0 ? 0 : (cnt > p.W ? p.W : cnt);
    const int32_t* src = p.kv_idx + row * p.W;
    const unsigned lt = (1u << lane) - 1u;
    int base = 0;
    for (int i0 = 0; i0 < cnt; i0 += 32) {
      const int i = i0 + lane;
      const int blk = (i < cnt) ? src[i] : -1;
      bool ok = (blk >= 0) && (blk < p.NB) && (blk <= tq);
      const unsigned same = __match_any_sync(0xffffffffu, ok ? blk : -1 - lane);
      if (same & lt) ok = false;
      if (i0 > 0 && ok) {
        for (int u = 0; u < base; ++u)
          if (ctl->list[u] == static_cast<uint16_t>(blk)) { ok = false; break; }
      }
      const unsigned bal = __ballot_sync(0xffffffffu, ok);
      if (ok) ctl->list[base + __popc(bal & lt)] = static_cast<uint16_t>(blk);
      base += __popc(bal);
      __syncwarp();
    }
    if (lane == 0) ctl->n_valid = base;
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = ctl->tmem_base;
  const int n_blk = ctl->n_valid;
  const int n_it = (n_blk + 1) >> 1;

  if (n_it > 0) {
    if (warp == 8) {
      // ---- TMA producer of the K ring: two slab units per iteration; each unit holds block a in rows
      // 0-63 and block b in rows 64-127 ----------------------------------------------------------------
      if (lane == 0) {
        int kseq = 0;
        for (int i = 0; i < n_it; ++i) {
          const int ba = ctl->list[2 * i];
          const int bb = (2 * i + 1 < n_blk) ? ctl->list[2 * i + 1] : -1;
          for (int s = 0; s < 2; ++s, ++kseq) {
            const int slot = kseq % NKU;
            mbar_wait(smem_u32(&ctl->k_empty[slot]), ((kseq / NKU) & 1) ^ 1);
            const uint32_t dst = smem_u32(ring_s + slot * UNIT), bar = smem_u32(&ctl->k_full[slot]);
            mbar_arrive_expect_tx(bar, bb >= 0 ? UNIT : UNIT / 2);
            tma_load_5d(dst, &tmK, bar, 0, ba * TB, s, g, b);
            if (bb >= 0) tma_load_5d(dst + UNIT / 2, &tmK, bar, 0, bb * TB, s, g, b);
          }
        }
      }
    } else if (warp == 9) {
      // ---- TMA producer of the V ring: one unit per selected block ---------------------------------
      if (lane == 0) {
        for (int vseq = 0; vseq < n_blk; ++vseq) {
          const int slot = vseq % NVU;
          mbar_wait(smem_u32(&ctl->v_empty[slot]), ((vseq / NVU) & 1) ^ 1);
          const uint32_t bar = smem_u32(&ctl->v_full[slot]);
          mbar_arrive_expect_tx(bar, UNIT);
          tma_load_5d(smem_u32(ring_s + (NKU + slot) * UNIT), &tmV, bar, 0, ctl->list[vseq] * TB, 0, g, b);
        }
      }
    } else if (warp == 10) {
      // ---- QK issue: S^T(i) = [K_a; K_b] Q^T into S buffer i & 1, one iteration ahead of the softmax --
      if (lane == 0) {
        constexpr uint32_t idesc = umma_idesc_bf16(128, TB, 0, 0);
        const uint32_t q_a = smem_u32(q_s);
        mbar_wait(smem_u32(&ctl->q_full), 0);
        int kseq = 0;
        for (int i = 0; i < n_it; ++i) {
          if (i >= 2) mbar_wait(smem_u32(&ctl->s_free[i & 1]), ((i >> 1) & 1) ^ 1);
          const uint32_t tS = tmem + S_COL + (i & 1) * 64;
          for (int s = 0; s < 2; ++s, ++kseq) {
            const int slot = kseq % NKU;
            mbar_wait(smem_u32(&ctl->k_full[slot]), (kseq / NKU) & 1);
            tc_fence_after();
            const uint32_t k_a = smem_u32(ring_s + slot * UNIT);
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
              const uint64_t ad = umma_smem_desc(k_a + ks * 32, 16, 1024);
              const uint64_t bd = umma_smem_desc(q_a + s * (TB * 128) + ks * 32, 16, 1024);
#ifndef T_ABL_NOMMA
              umma_ss(tS, ad, bd, idesc, (s > 0) || (ks > 0));
#endif
            }
            tc_commit(smem_u32(&ctl->k_empty[slot]));
          }
          tc_commit(smem_u32(&ctl->s_full[i & 1]));
        }
      }
    } else if (warp == 11) {
      // ---- PV issue: O^T += [V_a; V_b]^T P^T (both operands MN-major) ------------------------------
      if (lane == 0) {
        constexpr uint32_t idesc = umma_idesc_bf16(128, TB, 1, 1);
        const uint32_t tO = tmem + O_COL;
        int vseq = 0;
        for (int jj = 0; jj < n_it; ++jj) {
          const uint32_t p_a = smem_u32(p_s + (jj & 1) * T_P_BYTES);
          mbar_wait(smem_u32(&ctl->p_full[jj & 1]), (jj >> 1) & 1);
          tc_fence_after();
          for (int u = 0; u < 2; ++u) {
            if (2 * jj + u >= n_blk) break;
            const int slot = vseq % NVU;
            mbar_wait(smem_u32(&ctl->v_full[slot]), (vseq / NVU) & 1);
            tc_fence_after();
            const uint32_t v_a = smem_u32(ring_s + (NKU + slot) * UNIT);
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
              const uint64_t ad = umma_smem_desc(v_a + ks * 2048, TB * 128, 1024);        // d chunks 8 KB apart
              const uint64_t bd = umma_smem_desc(p_a + (u * 4 + ks) * 2048, 16, 1024);
#if !defined(T_ABL_NOMMA) && !defined(T_ABL_NOPV)
              umma_ss(tO, ad, bd, idesc, (jj > 0) || (u > 0) || (ks > 0));
#endif
            }
            tc_commit(smem_u32(&ctl->v_empty[slot]));
            ++vseq;
          }
          tc_commit(smem_u32(&ctl->o_done[jj & 1]));
        }
      }
    } else if (warp < 8) {
      t_softmax(p, ctl, p_s, ring_s, tmem, n_blk, tq, b, h);
    }
  } else if (warp < 4) {
    // nothing attended (possible only with a caller-provided kv_idx): zeros, lse = -inf
    mbar_wait(smem_u32(&ctl->q_full), 0);
    if (tid < TB && q0 + tid < p.N) {
      uint16_t* orow = p.O + b * p.qsb + h * p.qsh + static_cast<int64_t>(q0 + tid) * p.qsn;
      for (int c = 0; c < TD; c += 8) *reinterpret_cast<uint4*>(orow + c) = make_uint4(0, 0, 0, 0);
      if (p.lse) p.lse[(static_cast<int64_t>(b) * p.H + h) * p.N + q0 + tid] = -INFINITY;
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 8) tmem_dealloc<T_TMEM_COLS>(tmem);
}

}  // namespace

bool attn_t_supported(const Dims& S, int W) { return S.Bn == TB && S.d == TD && W <= kTMaxW; }

bsa_status launch_attn_t(const Dims& S, const void* Q, const void* K, const void* V, const int32_t* kv_idx,
                         const int32_t* kv_count, int W, float scale, void* O, float* lse,
                         cudaStream_t stream) {
  TParams prm;
  prm.kv_idx = kv_idx; prm.kv_count = kv_count;
  prm.O = static_cast<uint16_t*>(O); prm.lse = lse;
  prm.W = W; prm.B = S.B; prm.H = S.H; prm.G = S.G; prm.N = S.N; prm.NB = S.NB;
  prm.qsb = S.qsb; prm.qsh = S.qsh; prm.qsn = S.qsn;
  prm.scale_log2 = scale * 1.4426950408889634f;
  CUtensorMap tq, tk, tv;
  if (!make_tmap_bhnd(&tq, Q, S.B, S.H, S.N, S.d, S.qsb, S.qsh, S.qsn, TB, S.d / 64, 1) ||
      !make_tmap_bhnd(&tk, K, S.B, S.Hkv, S.N, S.d, S.ksb, S.ksh, S.ksn, TB, 1, 1) ||
      !make_tmap_bhnd(&tv, V, S.B, S.Hkv, S.N, S.d, S.ksb, S.ksh, S.ksn, TB, S.d / 64, 1))
    return fail(BSA_ERR_CUDA, "attn_t: cuTensorMapEncodeTiled failed");
  cudaError_t e = cudaFuncSetAttribute(attn_t_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, T_SMEM);
  if (e != cudaSuccess) return fail(BSA_ERR_CUDA, "attn_t: smem attribute: %s", cudaGetErrorString(e));
  const unsigned grid = static_cast<unsigned>(S.NB) * S.B * S.H;
  attn_t_kernel<<<grid, kTThreads, T_SMEM, stream>>>(tq, tk, tv, prm);
  return check_launch("attn_t_kernel");
}

}  // namespace bsa

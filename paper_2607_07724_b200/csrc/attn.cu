// attn.cu -- bsa_sparse_attn_fwd / bsa_dense_attn_fwd: exact online-softmax attention over the K/V
// blocks listed in kv_idx (PAPER.md L43-47 softmax definition; L131, A.10 L342 iteration over
// kv_idx with a single-compare sentinel skip), and the dense causal kernel of the same design
// (L45, L156) used as the "x dense" denominator.
//
// Two kernels:
//   attn64p_kernel<D>        sparse attention at 64-token blocks from kv_idx rows of up to 128 entries -- the
//                            paper's configuration.  Persistent: 2 x #SM CTAs walk the (tile, head) items; Q, S,
//                            P and O all live in TMEM (two half-lane planes), only K / V pass through shared
//                            memory.  Described at its definition below.
//   attn_kernel<BM,D,SPARSE> one CTA per (Q tile, head, batch): dense attention (BM = 128), sparse attention at
//                            128-token blocks, bitmap lists, rows wider than 128 entries, and the A/B reference
//                            of the persistent kernel (BSA_ATTN_PERSISTENT=0).  7 warps:
//   warps 0-3  softmax: tcgen05.ld of S, fp32 online softmax in base 2, P (bf16) -> shared memory
//              (BM = 128) or into TMEM (BM = 64: PV then takes its A operand from TMEM), lazy rescale of the
//              O accumulator in TMEM, final normalisation and store
//   warp 4     TMA producer: Q once (BM = 128; for BM = 64 the softmax warps put Q into TMEM), then K and V
//              64-key sub-blocks through a ring of stages; the row coordinate of each load is
//              kv_idx * block ("gather" = ordinary tiled TMA loads)
//   warp 5     one thread issues tcgen05.mma: S = Q K^T into TMEM (SS form, both K-major, 128B swizzle; BM = 64:
//              TS form, A = Q from TMEM) and, for BM = 128 with d <= 128, O += P V (V is the MN-major B operand)
//   warp 6     BM = 64 and d = 256: a second thread issues the O += P V MMAs (own V ring, see below)
// Q tile rows: sparse = one selection tile (BM = block), dense = 128.  For BM = 64 the accumulator
// rows live in lanes 0-15 (or, with a lane offset of 16 in the address, 16-31) of each TMEM sub-partition.
#include <cuda_bf16.h>
#include <stdlib.h>

#include <atomic>
#include <type_traits>

#include "bsa_internal.h"
#include "sm100_ptx.cuh"
#include "tmap.h"

namespace bsa {

namespace {

constexpr int BN = 64;                 // keys per pipeline stage / per S tile
constexpr int kThreads = 224;          // warps 0-3 softmax, 4 TMA, 5 MMA issuer (QK), 6 PV issuer (BM = 64)
constexpr int kMaxW = 256;             // widest kv_idx row staged in shared memory

// Measured alternatives that did NOT help on B200 (C2 sparse attention; 1.81 ms with one issuing
// thread, 1.53 ms with two): two 64-key sub-blocks per iteration (2.27 ms: the K/V ring shrinks to
// 1.25 iterations), eight softmax warps splitting the columns of each row (1.90 ms: the pair barrier
// costs more than the shorter exp2 chain saves), a double-buffered P tile (1.85 ms with one issuing
// thread, 1.60 vs 1.53 ms with two), K:V slot splits 3:2 / 2:3 and K running 1 / 2 / 3 iterations
// ahead (all 1.53-1.55 ms), and the transposed PV product O^T += V^T P^T (M = d = 128, N = 64: 48 clk
// per MMA against 64 for M = 64, N = 128, see sm100_ptx.cuh; parity green but 1.80 ms -- the O
// accumulator then has d on lanes, so the lazy rescale needs a CTA-wide vote every iteration and the
// epilogue a transpose through shared memory).  Ablation of the same kernel: TMA gather alone
// 0.96 ms (19 TB/s = 64 B/clk/SM, the SM's L2 port), gather + softmax without MMAs 1.42 ms, UMMA
// M=64 floor 1.02 ms (8 x 32 + 4 x 64 clk per block with two CTAs interleaved on the pipe).
template <int BM, int D>
struct Cfg {
  static constexpr int kOcc = (D <= 128) ? 2 : 1;  // CTAs per SM this kernel is sized for
  static constexpr int Q_BYTES = BM * D * 2;
  static constexpr int P_BYTES = BM * BN * 2;
  // BM = 64: P never touches shared memory.  The softmax writes P(j) (bf16 pairs) over the first 32 columns
  // of the S buffer it has just read, and PV takes its A operand from TMEM (tcgen05.mma TS form).  The
  // kernel is bound by shared-memory bandwidth (TMA fill 32 KB + UMMA operand reads 56 KB + P 8 KB per
  // 64 keys at 128 B/clk/SM ~ the measured 1.5 ms at C2): this removes the P store and the A reads of PV
  // (16 of 96 KB), the generic->async proxy fence and the wait for PV(j-1) from the softmax chain, and
  // frees 8 KB for a sixth K/V stage.
  static constexpr bool kPTmem = (BM == 64);
  static constexpr int kPSmem = kPTmem ? 0 : P_BYTES;
  // BM = 64, round 2b: Q lives in TMEM too.  A UMMA M = 64 accumulator occupies lanes 0-15 of each 32-lane
  // quadrant; probed on B200: the D address of tcgen05.mma may carry a lane offset of 16, the accumulator then
  // occupies lanes 16-31, and a TMEM A operand must sit in the SAME half as D (offset 0 with 16: "misaligned
  // address").  So TMEM is two independent half-lane planes and the 256 columns hold twice what they held:
  //   plane 0 (lane offset 0) : O [0, D)      | P(0) [D, D+32)        | P(1) [D+32, D+64)
  //   plane 1 (lane offset 16): Q [0, D/2)    | S(0) [D/2, D/2+64)    | S(1) [D/2+64, D/2+128)
  // QK = TS form with A = Q in plane 1 (no Q tile in shared memory: 16 KB fewer operand reads per block, no
  // exposed shared-memory latency of the A operand, one more ring stage); P no longer aliases S, so QK(j+2)
  // waits for softmax(j) to have READ S(j) instead of for PV(j).
#ifndef BSA_Q_TMEM
#define BSA_Q_TMEM 1
#endif
  static constexpr bool kQTmem = (BM == 64) && (BSA_Q_TMEM != 0);
  static constexpr int kQSmem = kQTmem ? 0 : Q_BYTES;
  static constexpr int KV_BYTES = BN * D * 2;
  static constexpr int kBudget = (kOcc == 2 ? 115712 : 231424) - 1024;  // barriers + list live in 1 KB
  static constexpr int kNSraw = (kBudget - kQSmem - kPSmem) / KV_BYTES;
  static constexpr int NS = kNSraw > 8 ? 8 : kNSraw;
  static constexpr int SMEM = kQSmem + kPSmem + NS * KV_BYTES + 1024;
  // TMEM without kQTmem: S is double buffered -- columns [0,64) and [64,128) -- so that QK(j+1) can be
  // issued and retire while the softmax warps still work on S(j); O occupies columns [128, 128+D).
  static constexpr int S_COL = kQTmem ? D / 2 : 0;       // S(i) at S_COL + (i & 1) * BN
  static constexpr int O_COL = kQTmem ? 0 : 2 * BN;
  static constexpr int P_COL = kQTmem ? D : 0;           // P(j) at P_COL + (j & 1) * kPStride
  static constexpr int kPStride = kQTmem ? 32 : BN;      // (aliased over S(j) without kQTmem)
  static constexpr uint32_t kSLane = kQTmem ? 16u : 0u;  // lane offset of the Q / S plane
  static constexpr int kColsUsed = kQTmem ? (D + 64 > D / 2 + 128 ? D + 64 : D / 2 + 128) : O_COL + D;
  static constexpr uint32_t TMEM_COLS = (kColsUsed <= 256) ? 256 : 512;
  static_assert(NS >= 2 && ((BM != 64 && kOcc != 1) || NS >= 4), "not enough shared memory for a K/V ring");
};

struct Params {
  const int32_t* kv_idx;    // [B,H,T,W] or nullptr (dense, bitmap)
  const int32_t* kv_count;  // [B,H,T] or nullptr
  const uint32_t* bitmap;   // [B,H,T,nbw] block bitmap per (tile, head) (rowsel.cu), or nullptr
  int nbw;
  const uint16_t* Q;        // BM = 64: the softmax warps copy the Q tile from global memory into TMEM
  uint16_t* O;
  float* lse;
  int W, B, H, G, N, Bn, NB, NT;
  int pdl;                  // launched with programmatic stream serialization (bsa_select_attn_fwd)
  int64_t qsb, qsh, qsn;
  float scale_log2;
};

// bookkeeping block at the end of dynamic shared memory
struct alignas(8) Ctl {
  uint64_t q_full, p_full[2];      // per P buffer (BM = 128 uses buffer 0 only)
  uint64_t s_full[2], s_free[2];   // per S buffer
  uint64_t o_done[2];              // PV(j) done, per P buffer
  uint64_t kv_full[8], kv_empty[8];
  uint32_t tmem_base;
  int32_t n_valid;
  union {
    uint16_t list[kMaxW];       // kv_idx mode: the compacted row
    uint32_t bmw[kMaxW / 2];    // bitmap mode: the row's words, masked to blocks <= t (N_B <= 4096)
  };
};

// Walks the set bits of a bitmap row in ascending order; block_at(n) must be called with non-decreasing n.
struct BitCursor {
  const uint32_t* w;
  int wi, idx, blk;
  uint32_t cur;
  __device__ __forceinline__ void init(const uint32_t* words) {
    w = words; wi = 0; idx = -1; blk = -1; cur = words[0];
  }
  __device__ __forceinline__ int block_at(int n) {
    while (idx < n) {
      while (cur == 0u) cur = w[++wi];
      blk = wi * 32 + __ffs(cur) - 1;
      cur &= cur - 1u;
      ++idx;
    }
    return blk;
  }
};
static_assert(sizeof(Ctl) <= 1024, "Ctl must fit the 1 KB bookkeeping area");

#ifdef BSA_TRACE
// Debug builds only (-DBSA_TRACE): clock64 stamps of one CTA, read back with bsa_debug_trace().
// g_tr[role][iteration][stamp]: role 0 = softmax warp 0, 1 = QK thread, 2 = PV thread.
__device__ long long g_tr[4][32][8];   // role 3, slot 0: CTA-level stamps
#define TR(role, it, k) do { if (trace_on && (it) < 32) g_tr[role][it][k] = clock64(); } while (0)
#define TRW4(k) do { if (blockIdx.x == gridDim.x / 2 && threadIdx.x == 128) g_tr[3][2][k] = clock64(); } while (0)
#else
#define TRW4(k) do { } while (0)
#define TR(role, it, k) do { } while (0)
#endif

// ---- softmax warps, BM = 128 (dense; sparse with 128-token blocks) -------------------------------
// Thread r owns accumulator row r (TMEM lane r, 32x32b loads).  Logits stay unscaled in registers;
// the softmax scale is folded into one FFMA per element: p = 2^(s*scale_log2 - m).
template <int D, bool SPARSE, class KeyStart>
__device__ __forceinline__ void softmax_m128(const Params& p, Ctl* ctl, uint8_t* p_s, uint32_t tmem,
                                             int n_it, int q0, int b, int h, KeyStart key_start) {
  using C = Cfg<128, D>;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int r = tid, qrow = q0 + r;
  const uint32_t lane_base = static_cast<uint32_t>(warp * 32) << 16;
  const uint32_t tS = tmem + lane_base, tO = tmem + lane_base + C::O_COL;
  const float sc = p.scale_log2;
  float m = -INFINITY, l = 0.f;
  for (int j = 0; j < n_it; ++j) {
    const int k0 = key_start(j);
    mbar_wait(smem_u32(&ctl->s_full[j & 1]), (j >> 1) & 1);
    tc_fence_after();
    uint32_t sa[32], sb[32];
    tmem_ld32(tS + (j & 1) * BN, sa);
    tmem_ld32(tS + (j & 1) * BN + 32, sb);
    tmem_ld_wait();
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(smem_u32(&ctl->s_free[j & 1]));

    float x[64];
#pragma unroll
    for (int c = 0; c < 32; ++c) {
      x[c] = __uint_as_float(sa[c]);
      x[c + 32] = __uint_as_float(sb[c]);
    }
    if (k0 + BN - 1 > q0) {  // only blocks touching the diagonal need the causal mask
#pragma unroll
      for (int c = 0; c < 64; ++c) x[c] = (k0 + c <= qrow) ? x[c] : -INFINITY;
    }
    float mx = fmaxf(x[0], x[1]);
#pragma unroll
    for (int c = 2; c < 64; c += 2) mx = fmax3(mx, x[c], x[c + 1]);
    float m_new = fmaxf(m, mx * sc);
    // lazy rescale: keep the stale reference max unless some row of this warp grew by > 2^8
    const bool any = __any_sync(0xffffffffu, m_new - m > 8.0f);
    if (!any) m_new = m;
    const float alpha = ex2_approx(m - m_new);
    // packed fp32x2 FMA / ADD (FFMA2, FADD2): half the issue slots for the argument and the row sum
    float2 sum2a = make_float2(0.f, 0.f), sum2b = make_float2(0.f, 0.f);
    const float2 sc2 = make_float2(sc, sc), nm2 = make_float2(-m_new, -m_new);
    uint32_t pk[32];
#pragma unroll
    for (int c = 0; c < 64; c += 4) {
      const float2 t0 = ffma2(make_float2(x[c], x[c + 1]), sc2, nm2);
      const float2 t1 = ffma2(make_float2(x[c + 2], x[c + 3]), sc2, nm2);
      const float2 e0 = make_float2(ex2_approx(t0.x), ex2_approx(t0.y));
      const float2 e1 = make_float2(ex2_approx(t1.x), ex2_approx(t1.y));
      sum2a = fadd2(sum2a, e0);
      sum2b = fadd2(sum2b, e1);
      pk[c >> 1] = pack_bf16x2(e0.x, e0.y);
      pk[(c >> 1) + 1] = pack_bf16x2(e1.x, e1.y);
    }
    l = l * alpha + ((sum2a.x + sum2a.y) + (sum2b.x + sum2b.y));
    m = m_new;

    if (j > 0) {
      mbar_wait(smem_u32(&ctl->o_done[0]), (j - 1) & 1);  // PV(j-1) done: P and O are ours
      tc_fence_after();
      if (any) {
#pragma unroll
        for (int c0 = 0; c0 < D; c0 += 32) {
          uint32_t o[32];
          tmem_ld32(tO + c0, o);
          tmem_ld_wait();
#pragma unroll
          for (int c = 0; c < 32; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha);
          tmem_st32(tO + c0, o);
        }
        tmem_st_wait();
      }
    }
    uint8_t* prow = p_s + r * 128;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      uint4 v = make_uint4(pk[4 * c], pk[4 * c + 1], pk[4 * c + 2], pk[4 * c + 3]);
      *reinterpret_cast<uint4*>(prow + ((c ^ (r & 7)) << 4)) = v;
    }
    fence_proxy_async_smem();
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(smem_u32(&ctl->p_full[0]));
  }
  // ---- epilogue: O / l -> bf16 -> global ---------------------------------------------------------
  mbar_wait(smem_u32(&ctl->o_done[0]), (n_it - 1) & 1);
  tc_fence_after();
  const float inv_l = 1.0f / l;
  const bool store = qrow < p.N;
  uint16_t* orow = p.O + b * p.qsb + h * p.qsh + static_cast<int64_t>(qrow) * p.qsn;
#pragma unroll
  for (int c0 = 0; c0 < D; c0 += 32) {
    uint32_t o[32];
    tmem_ld32(tO + c0, o);
    tmem_ld_wait();
    if (store) {
#pragma unroll
      for (int c = 0; c < 32; c += 8) {
        uint4 v;
        v.x = pack_bf16x2(__uint_as_float(o[c]) * inv_l, __uint_as_float(o[c + 1]) * inv_l);
        v.y = pack_bf16x2(__uint_as_float(o[c + 2]) * inv_l, __uint_as_float(o[c + 3]) * inv_l);
        v.z = pack_bf16x2(__uint_as_float(o[c + 4]) * inv_l, __uint_as_float(o[c + 5]) * inv_l);
        v.w = pack_bf16x2(__uint_as_float(o[c + 6]) * inv_l, __uint_as_float(o[c + 7]) * inv_l);
        *reinterpret_cast<uint4*>(orow + c0 + c) = v;
      }
    }
  }
  if (store && p.lse)
    p.lse[(static_cast<int64_t>(b) * p.H + h) * p.N + qrow] = (m + log2f(l)) * 0.6931471805599453f;
  tc_fence_before();
}

// ---- softmax warps, BM = 64 (sparse, 64-token blocks) -------------------------------------------
// A UMMA M = 64 accumulator keeps row r in TMEM lane 32*(r/16) + r%16, i.e. only 16 of the 32 lanes
// of each warp's quadrant.  A 32x32b load would leave half the threads idle through the whole
// softmax; the 16x256b shape instead spreads the 16 lanes x 64 columns over all 32 threads: thread
// t owns rows rA = 16w + t/4 and rB = rA + 8, and in every 8-column group the two columns
// 2(t%4), 2(t%4)+1.  Row max = in-thread max + two quad shuffles; the row sum stays a per-thread
// partial until the epilogue.
// Epilogue helper for the BM = 64 fragment layout: thread q = lane % 4 of a quad holds, for every 8-column group,
// the word (two bf16) at columns 2q, 2q+1.  Two shuffle rounds turn the words w0..w3 of four consecutive groups
// g0..g0+3 into the complete 16 bytes of group g0 + q, so that a row leaves as 64 contiguous bytes per quad and
// store instruction instead of 16 (32 four-byte stores per thread kept the store path busy for ~2000 clk).
__device__ __forceinline__ uint4 quad_gather(uint32_t w0, uint32_t w1, uint32_t w2, uint32_t w3, int q) {
  const bool odd = (q & 1) != 0, hi = (q & 2) != 0;
  const uint32_t r01 = __shfl_xor_sync(0xffffffffu, odd ? w0 : w1, 1);
  const uint32_t r23 = __shfl_xor_sync(0xffffffffu, odd ? w2 : w3, 1);
  const uint32_t ax = odd ? r01 : w0, ay = odd ? w1 : r01;   // even q: group g0 (+2: bx, by), odd q: group g0 + 1 (+3)
  const uint32_t bx = odd ? r23 : w2, by = odd ? w3 : r23;
  const uint32_t rx = __shfl_xor_sync(0xffffffffu, hi ? ax : bx, 2);
  const uint32_t ry = __shfl_xor_sync(0xffffffffu, hi ? ay : by, 2);
  return hi ? make_uint4(rx, ry, bx, by) : make_uint4(ax, ay, rx, ry);
}

// Q tile rows of this thread (rA, rB of the fragment layout below), loaded at kernel entry so that the
// global-memory latency runs under the CTA's setup: qr[c][2g] / qr[c][2g+1] = the element pair
// 64c + 8g + 2(t%4) of row rA / rB.
template <int D>
__device__ __forceinline__ void load_q_m64(const Params& p, int q0, int b, int h, uint32_t (&qr)[D / 64][16]) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int rA = warp * 16 + (lane >> 2);
  const uint16_t* qbase = p.Q + b * p.qsb + h * p.qsh + 2 * (lane & 3);
  const uint16_t* qA = qbase + static_cast<int64_t>(q0 + rA) * p.qsn;
  const uint16_t* qB = qA + 8 * p.qsn;
#pragma unroll
  for (int c = 0; c < D / 64; ++c) {
#pragma unroll
    for (int g = 0; g < 8; ++g) {
      qr[c][2 * g] = __ldg(reinterpret_cast<const uint32_t*>(qA + 64 * c + 8 * g));
      qr[c][2 * g + 1] = __ldg(reinterpret_cast<const uint32_t*>(qB + 64 * c + 8 * g));
    }
  }
}

template <int D, bool SPARSE, class KeyStart>
__device__ __forceinline__ void softmax_m64(const Params& p, Ctl* ctl, uint8_t* p_s, uint32_t tmem,
                                            int n_it, int q0, int b, int h, KeyStart key_start,
                                            const uint32_t (&qr)[D / 64][16]) {
  using C = Cfg<64, D>;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int quad = lane & 3;
  const int rA = warp * 16 + (lane >> 2), rB = rA + 8;
  const int qrA = q0 + rA, qrB = q0 + rB;
  const uint32_t lane_base = static_cast<uint32_t>(warp * 32) << 16;
  const uint32_t tS = tmem + lane_base + (C::kSLane << 16) + C::S_COL;   // S(j) at tS + (j & 1) * BN
  const uint32_t tO = tmem + lane_base + C::O_COL;
  const uint32_t tP = tmem + lane_base + C::P_COL;                       // P(j) at tP + (j & 1) * kPStride
  const float sc = p.scale_log2;
  float mA = -INFINITY, mB = -INFINITY, lA = 0.f, lB = 0.f;
#ifdef BSA_TRACE
  const bool trace_on = blockIdx.x == gridDim.x / 2 && tid == 0;
#endif
  if constexpr (C::kQTmem) {
    // Q tile -> TMEM plane 1, columns [0, D/2): the A-operand image (word c of a row = elements 2c, 2c+1).
    // The 16x128b store takes, per 8-element group g, the pair 8g + 2(t%4) of row rA and of row rB.
    const uint32_t tQ = tmem + lane_base + (C::kSLane << 16);
#pragma unroll
    for (int c = 0; c < D / 64; ++c) tmem_st16x128_x8(tQ + 32 * c, qr[c]);
    tmem_st_wait();
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(smem_u32(&ctl->q_full));
  }
  TR(3, 0, 2);
  for (int j = 0; j < n_it; ++j) {
    const int k0 = key_start(j);
    TR(0, j, 0);
    if (C::kQTmem && j >= 2) {
      // S(j) ready, and PV(j-2) done so that P(j) may later overwrite P(j-2): one poll for both
      mbar_wait2_warp(smem_u32(&ctl->s_full[j & 1]), (j >> 1) & 1, smem_u32(&ctl->o_done[j & 1]),
                      ((j - 2) >> 1) & 1);
    } else {
      mbar_wait(smem_u32(&ctl->s_full[j & 1]), (j >> 1) & 1);
    }
    tc_fence_after();
    TR(0, j, 1);
    uint32_t s[32];
    tmem_ld16x256_x8(tS + (j & 1) * BN, s);
    tmem_ld_wait();
    TR(0, j, 2);
    tc_fence_before();
    __syncwarp();
    if constexpr (C::kQTmem) {
      if (lane == 0) mbar_arrive(smem_u32(&ctl->s_free[j & 1]));   // QK(j+2) may overwrite S(j)
    }
    // (without kQTmem no s_free arrival: the S buffer also carries P(j); QK(j+2) waits for PV(j) instead)

    float xa[16], xb[16];
#pragma unroll
    for (int g = 0; g < 8; ++g) {
      xa[2 * g] = __uint_as_float(s[4 * g]);
      xa[2 * g + 1] = __uint_as_float(s[4 * g + 1]);
      xb[2 * g] = __uint_as_float(s[4 * g + 2]);
      xb[2 * g + 1] = __uint_as_float(s[4 * g + 3]);
    }
    if (k0 + BN - 1 > q0) {
#pragma unroll
      for (int g = 0; g < 8; ++g) {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int key = k0 + 8 * g + 2 * quad + e;
          xa[2 * g + e] = (key <= qrA) ? xa[2 * g + e] : -INFINITY;
          xb[2 * g + e] = (key <= qrB) ? xb[2 * g + e] : -INFINITY;
        }
      }
    }
    float mxA = fmaxf(xa[0], xa[1]), mxB = fmaxf(xb[0], xb[1]);
#pragma unroll
    for (int c = 2; c < 16; c += 2) {
      mxA = fmax3(mxA, xa[c], xa[c + 1]);
      mxB = fmax3(mxB, xb[c], xb[c + 1]);
    }
    // lazy rescale: keep the stale reference maxima unless some row of this warp grew by > 2^8.
    // The test only needs each thread's partial maximum (a row exceeds iff one of its four threads
    // does), so the quad shuffles and the alphas are off the common path.
    const bool any = __any_sync(0xffffffffu, (fmaf(mxA, sc, -mA) > 8.0f) || (fmaf(mxB, sc, -mB) > 8.0f));
    float mA_new = mA, mB_new = mB, alphaA = 1.0f, alphaB = 1.0f;
    if (any) {
      mxA = fmaxf(mxA, __shfl_xor_sync(0xffffffffu, mxA, 1));
      mxB = fmaxf(mxB, __shfl_xor_sync(0xffffffffu, mxB, 1));
      mxA = fmaxf(mxA, __shfl_xor_sync(0xffffffffu, mxA, 2));
      mxB = fmaxf(mxB, __shfl_xor_sync(0xffffffffu, mxB, 2));
      mA_new = fmaxf(mA, mxA * sc);
      mB_new = fmaxf(mB, mxB * sc);
      alphaA = ex2_approx(mA - mA_new);
      alphaB = ex2_approx(mB - mB_new);
    }
    // packed fp32x2 FMA / ADD: half the issue slots of the scalar form for the argument and the sum
    float2 sumA2 = make_float2(0.f, 0.f), sumB2 = make_float2(0.f, 0.f);
    const float2 sc2 = make_float2(sc, sc);
    const float2 nmA = make_float2(-mA_new, -mA_new), nmB = make_float2(-mB_new, -mB_new);
    uint32_t pa[8], pb[8];
#pragma unroll
    for (int g = 0; g < 8; ++g) {
      const float2 ta = ffma2(make_float2(xa[2 * g], xa[2 * g + 1]), sc2, nmA);
      const float2 tb = ffma2(make_float2(xb[2 * g], xb[2 * g + 1]), sc2, nmB);
#if defined(BSA_ABL) && BSA_ABL == 1
      const float2 ea = make_float2(ex2_approx(ta.x), fmaf(ta.y, 0.001f, 0.5f));
      const float2 eb = make_float2(ex2_approx(tb.x), fmaf(tb.y, 0.001f, 0.5f));
#elif defined(BSA_ABL) && BSA_ABL == 2
      const float2 ea = make_float2(fmaf(ta.x, 0.001f, 0.5f), fmaf(ta.y, 0.001f, 0.5f));
      const float2 eb = make_float2(fmaf(tb.x, 0.001f, 0.5f), fmaf(tb.y, 0.001f, 0.5f));
#else
      const float2 ea = make_float2(ex2_approx(ta.x), ex2_approx(ta.y));
      const float2 eb = make_float2(ex2_approx(tb.x), ex2_approx(tb.y));
#endif
      sumA2 = fadd2(sumA2, ea);
      sumB2 = fadd2(sumB2, eb);
      pa[g] = pack_bf16x2(ea.x, ea.y);
      pb[g] = pack_bf16x2(eb.x, eb.y);
    }
    lA = lA * alphaA + (sumA2.x + sumA2.y);
    lB = lB * alphaB + (sumB2.x + sumB2.y);
    mA = mA_new;
    mB = mB_new;
    TR(0, j, 3);

    if (any && j > 0) {
      // the rare rescale touches O: every earlier PV must be done (they complete in order)
      mbar_wait(smem_u32(&ctl->o_done[(j - 1) & 1]), ((j - 1) >> 1) & 1);
      tc_fence_after();
      {
#pragma unroll
        for (int c0 = 0; c0 < D; c0 += 64) {
          uint32_t o[32];
          tmem_ld16x256_x8(tO + c0, o);
          tmem_ld_wait();
#pragma unroll
          for (int g = 0; g < 8; ++g) {
            o[4 * g] = __float_as_uint(__uint_as_float(o[4 * g]) * alphaA);
            o[4 * g + 1] = __float_as_uint(__uint_as_float(o[4 * g + 1]) * alphaA);
            o[4 * g + 2] = __float_as_uint(__uint_as_float(o[4 * g + 2]) * alphaB);
            o[4 * g + 3] = __float_as_uint(__uint_as_float(o[4 * g + 3]) * alphaB);
          }
          tmem_st16x256_x8(tO + c0, o);
        }
        tmem_st_wait();
      }
    }
    // P(j) -> TMEM, over columns [0, 32) of the S buffer just read: the 16x128b store writes, per 8-key
    // group g, the bf16 pair of row rA to (lane t/4, column 4g + t%4) and that of rB to lane t/4 + 8 --
    // the A-operand image of the accumulator fragment (sm100_ptx.cuh).
    {
      uint32_t pr[16];
#pragma unroll
      for (int g = 0; g < 8; ++g) {
        pr[2 * g] = pa[g];
        pr[2 * g + 1] = pb[g];
      }
      // (kQTmem: P has its own two buffers in plane 0; that PV(j-2) has consumed the one P(j) goes to was
      // checked together with s_full at the top of the iteration)
      tmem_st16x128_x8(tP + (j & 1) * C::kPStride, pr);
      tmem_st_wait();
    }
    TR(0, j, 4);
    tc_fence_before();
    __syncwarp();
    // per-buffer barrier: the softmax may publish P(j+1) before the PV thread has even looked at P(j)
    if (lane == 0) mbar_arrive(smem_u32(&ctl->p_full[j & 1]));
  }
  // ---- epilogue: O / l -> bf16 -> global ---------------------------------------------------------
  TR(3, 0, 3);
  mbar_wait(smem_u32(&ctl->o_done[(n_it - 1) & 1]), ((n_it - 1) >> 1) & 1);
  tc_fence_after();
  TR(3, 0, 4);
  lA += __shfl_xor_sync(0xffffffffu, lA, 1);
  lB += __shfl_xor_sync(0xffffffffu, lB, 1);
  lA += __shfl_xor_sync(0xffffffffu, lA, 2);
  lB += __shfl_xor_sync(0xffffffffu, lB, 2);
  const float invA = 1.0f / lA, invB = 1.0f / lB;
  const bool stA = qrA < p.N, stB = qrB < p.N;
  uint16_t* obase = p.O + b * p.qsb + h * p.qsh + 2 * quad;
  uint16_t* orowA = obase + static_cast<int64_t>(qrA) * p.qsn;
  uint16_t* orowB = obase + static_cast<int64_t>(qrB) * p.qsn;
#pragma unroll
  for (int c0 = 0; c0 < D; c0 += 64) {
    uint32_t o[32];
    tmem_ld16x256_x8(tO + c0, o);
    tmem_ld_wait();
#pragma unroll
    for (int g = 0; g < 8; ++g) {
      const uint32_t va = pack_bf16x2(__uint_as_float(o[4 * g]) * invA, __uint_as_float(o[4 * g + 1]) * invA);
      const uint32_t vb = pack_bf16x2(__uint_as_float(o[4 * g + 2]) * invB, __uint_as_float(o[4 * g + 3]) * invB);
      if (stA) *reinterpret_cast<uint32_t*>(orowA + c0 + 8 * g) = va;
      if (stB) *reinterpret_cast<uint32_t*>(orowB + c0 + 8 * g) = vb;
    }
  }
  if (p.lse && quad == 0) {
    float* lse = p.lse + (static_cast<int64_t>(b) * p.H + h) * p.N;
    if (stA) lse[qrA] = (mA + log2f(lA)) * 0.6931471805599453f;
    if (stB) lse[qrB] = (mB + log2f(lB)) * 0.6931471805599453f;
  }
  TR(3, 0, 5);
  tc_fence_before();
}

template <int BM, int D, bool SPARSE>
__global__ void __launch_bounds__(kThreads, Cfg<BM, D>::kOcc)
attn_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
            const __grid_constant__ CUtensorMap tmV, const Params p) {
  using C = Cfg<BM, D>;
  extern __shared__ __align__(1024) uint8_t smem[];
  uint8_t* q_s = smem;
  uint8_t* p_s = smem + C::kQSmem;
  uint8_t* kv_s = p_s + C::kPSmem;
  Ctl* ctl = reinterpret_cast<Ctl*>(kv_s + C::NS * C::KV_BYTES);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  // work item order: (batch, KV head) outermost so that the CTAs in flight at any moment gather
  // from ONE KV head's K/V (N*d*4 bytes: 67 MB at 128K, d=128 -- resident in the 126 MB L2) instead
  // of all of them; inside a KV head the heaviest (largest tile index) tiles go first, and the G
  // query heads of the group run side by side.
  int wi = static_cast<int>(blockIdx.x);
  const int hi = wi % p.G;
  wi /= p.G;
  const int tq = p.NT - 1 - wi % p.NT;
  wi /= p.NT;
  const int Hkv = p.H / p.G;
  const int g = wi % Hkv, b = wi / Hkv, h = g * p.G + hi;
  const int q0 = tq * BM;  // first query row of this tile

  if ((smem_u32(smem) & 1023u) != 0) __trap();
#ifdef BSA_TRACE
  const bool trace_on = blockIdx.x == gridDim.x / 2 && tid == 0;
#endif
  TR(3, 0, 0);   // CTA-level stamps (entry, setup done, Q in TMEM, loop end, last PV seen, stored)

  uint32_t qreg[BM == 64 ? D / 64 : 1][16];
  constexpr bool kListFirst = SPARSE && BM == 64 && C::kQTmem;   // warp 0 requests its kv_idx row first
  if constexpr (BM == 64 && C::kQTmem) {
    if (warp < 4 && !(kListFirst && warp == 0 && !p.pdl && p.bitmap == nullptr))
      load_q_m64<D>(p, q0, b, h, qreg);   // in flight during the setup below
  }

  // ---- setup ---------------------------------------------------------------------------------
  // Early start (sparse list mode with split rings): the producer thread reads the first entry of the row
  // itself and, if it is a visible block (then it is also the first entry of the compacted list), loads
  // K(0) and V(0) before the list compaction and the CTA barrier -- the first QK no longer waits for a
  // TMA round trip after the setup.  Slot 0 of each ring is used; the dedupe bitmap lives in the last slot.
  constexpr bool kEarly = SPARSE && ((BM == 64) || (C::kOcc == 1)) && C::NS >= 4;
  bool early = false;
  if (warp == 4) {
    int e_blk = -1, e_cnt = 0;
    if (kEarly && lane == 0 && p.bitmap == nullptr) {
      if (p.pdl) griddep_wait();
      const int64_t row = (static_cast<int64_t>(b) * p.H + h) * p.NT + tq;
      e_blk = __ldg(p.kv_idx + row * p.W);
      e_cnt = p.kv_count ? __ldg(p.kv_count + row) : p.W;
    }
    if (lane == 0) {
      mbar_init(smem_u32(&ctl->q_full), C::kQTmem ? 4 : 1);
      for (int i = 0; i < 2; ++i) {
        mbar_init(smem_u32(&ctl->s_full[i]), 1);
        mbar_init(smem_u32(&ctl->s_free[i]), 4);
      }
      for (int i = 0; i < 2; ++i) {
        mbar_init(smem_u32(&ctl->p_full[i]), 4);
        mbar_init(smem_u32(&ctl->o_done[i]), 1);
      }
      for (int s = 0; s < C::NS; ++s) {
        mbar_init(smem_u32(&ctl->kv_full[s]), 1);
        mbar_init(smem_u32(&ctl->kv_empty[s]), 1);
      }
      fence_mbar_init();
      TRW4(0);
      // the Q tile does not depend on the kv_idx row: start it now, under the TMEM allocation and
      // the list compaction below (both ~1 us of latency)
      if constexpr (!C::kQTmem) {
        mbar_arrive_expect_tx(smem_u32(&ctl->q_full), C::Q_BYTES);
        tma_load_5d(smem_u32(q_s), &tmQ, smem_u32(&ctl->q_full), 0, q0, 0, h, b);
      }
      tma_prefetch_desc(&tmK);
      tma_prefetch_desc(&tmV);
      if (kEarly && e_cnt > 0 && e_blk >= 0 && e_blk < p.NB && e_blk <= tq) {
        constexpr int NSK0 = (C::NS + 1) / 2;
        early = true;
        mbar_arrive_expect_tx(smem_u32(&ctl->kv_full[0]), C::KV_BYTES);
        tma_load_5d(smem_u32(kv_s), &tmK, smem_u32(&ctl->kv_full[0]), 0, e_blk * p.Bn, 0, g, b);
        mbar_arrive_expect_tx(smem_u32(&ctl->kv_full[NSK0]), C::KV_BYTES);
        tma_load_5d(smem_u32(kv_s + NSK0 * C::KV_BYTES), &tmV, smem_u32(&ctl->kv_full[NSK0]), 0, e_blk * p.Bn, 0,
                    g, b);
      }
    }
    __syncwarp();
    tmem_alloc<C::TMEM_COLS>(smem_u32(&ctl->tmem_base));
    TRW4(1);
  }
  // kv_idx / kv_count / bitmap come from the selection kernels: under a programmatic dependent launch
  // everything above (barriers, TMEM, the Q tile load) overlapped their tail
  if (SPARSE && warp == 0) griddep_wait();
  if (SPARSE && warp == 0 && p.bitmap != nullptr) {
    // bitmap mode: copy the row's words, masked to the visible blocks (<= t); count the set bits
    const int64_t row = (static_cast<int64_t>(b) * p.H + h) * p.NT + tq;
    const uint32_t* src = p.bitmap + row * p.nbw;
    int cnt = 0;
    for (int i = lane; i < kMaxW / 2; i += 32) {
      uint32_t wv = (i < p.nbw && i * 32 <= tq) ? src[i] : 0u;
      if (i == (tq >> 5) && (tq & 31) != 31) wv &= (2u << (tq & 31)) - 1u;
      ctl->bmw[i] = wv;
      cnt += __popc(wv);
    }
    cnt = __reduce_add_sync(0xffffffffu, cnt);
    if (lane == 0) ctl->n_valid = cnt;
  } else if (SPARSE && warp == 0) {
    // compact the valid entries of this kv_idx row (sentinel >= N_B and blocks > t are skipped, A.10;
    // a block listed more than once is attended once, like the oracle's O11).  The whole row and its
    // count are requested at once (one global-memory latency); duplicates are found with a bitmap of the
    // visible blocks kept in the still unused K/V ring (N_B <= 65535 -> at most 8 KB).
    const int64_t row = (static_cast<int64_t>(b) * p.H + h) * p.NT + tq;
    const int32_t* src = p.kv_idx + row * p.W;
    int blkv[kMaxW / 32];
#pragma unroll
    for (int c = 0; c < kMaxW / 32; ++c) blkv[c] = (c * 32 + lane < p.W) ? __ldg(src + c * 32 + lane) : -1;
    int cnt = p.kv_count ? __ldg(p.kv_count + row) : p.W;
    if constexpr (kListFirst) {
      if (!p.pdl) load_q_m64<D>(p, q0, b, h, qreg);
    }
    TR(3, 1, 0);
    uint32_t* seen = reinterpret_cast<uint32_t*>(kv_s + (C::NS - 1) * C::KV_BYTES);   // last ring slot
    for (int i = lane; i <= (tq >> 5); i += 32) seen[i] = 0u;
    __syncwarp();
    TR(3, 1, 1);
    cnt = cnt < 0 ? 0 : (cnt > p.W ? p.W : cnt);
    TR(3, 1, 2);
    const unsigned lt = (1u << lane) - 1u;
    int base = 0;
#pragma unroll
    for (int c = 0; c < kMaxW / 32; ++c) {
      if (c * 32 < cnt) {
        const int i = c * 32 + lane;
        const int blk = (i < cnt) ? blkv[c] : -1;
        const bool valid = (blk >= 0) && (blk < p.NB) && (blk <= tq);
        // every valid entry marks its block; an entry that finds the mark already set is a duplicate
        bool ok = valid && (atomicOr(&seen[blk >> 5], 1u << (blk & 31)) & (1u << (blk & 31))) == 0u;
        if (__ballot_sync(0xffffffffu, ok) != __ballot_sync(0xffffffffu, valid)) {
          // rare: some duplicate.  Which of two equal entries of this chunk won the atomic is arbitrary, so
          // resolve it by position: the lowest lane of a block wins unless an earlier chunk listed the block.
          const unsigned same = __match_any_sync(0xffffffffu, valid ? blk : -1 - lane);
          ok = valid && !(same & lt);
          if (ok) {
            for (int u = 0; u < base; ++u)
              if (ctl->list[u] == static_cast<uint16_t>(blk)) { ok = false; break; }
          }
        }
        const unsigned bal = __ballot_sync(0xffffffffu, ok);
        if (ok) ctl->list[base + __popc(bal & lt)] = static_cast<uint16_t>(blk);
        base += __popc(bal);
      }
    }
    if (lane == 0) ctl->n_valid = base;
    TR(3, 1, 3);
    fence_proxy_async_smem();   // the ring goes to the TMA (async proxy) after the CTA barrier below
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  TR(3, 0, 1);
  const uint32_t tmem = ctl->tmem_base;

  constexpr int SUBS = SPARSE ? (BM / BN) : 1;  // 64-key sub-blocks per selected block
  int n_it;
  if (SPARSE) {
    n_it = ctl->n_valid * SUBS;
  } else {
    const int last = (q0 + BM < p.N ? q0 + BM : p.N);
    n_it = last / BN;
  }
  const bool use_bm = SPARSE && p.bitmap != nullptr;
  BitCursor cur_a, cur_b;                      // softmax: cur_a; TMA producer: cur_a for K, cur_b for V
  if (use_bm) {
    cur_a.init(ctl->bmw);
    cur_b.init(ctl->bmw);
  }
  auto start_of = [&](BitCursor& cur, int j) -> int {
    if (SPARSE) {
      const int blk = use_bm ? cur.block_at(j / SUBS) : static_cast<int>(ctl->list[j / SUBS]);
      return blk * p.Bn + (j % SUBS) * BN;
    }
    return j * BN;
  };
  auto key_start = [&](int j) -> int { return start_of(cur_a, j); };

  // ---- K/V ring bookkeeping --------------------------------------------------------------------
  // BM = 128, d <= 128 (two CTAs per SM): one thread issues QK(j+1), PV(j) alternately (kAhead = 1)
  // and the K and V tiles share ONE ring, entered in the order that thread consumes them: K(0), then
  // [K(j+1), V(j)].  (Two threads measured 3 % slower there: 1168 -> 1135 TFLOP/s dense at 32K.)
  // BM = 64, and d = 256 (one CTA per SM; dense 1023 -> 1211 TFLOP/s, sparse C5 1014 -> 1145 with two
  // threads): QK and PV are issued by TWO threads and QK runs up to two iterations ahead, so K and V
  // get SEPARATE rings (NSK + NSV = NS slots), each with a single in-order consumer.  Sharing one
  // ring between two consumers is a bug, not an optimisation: a parity wait on a slot's `full`
  // barrier also succeeds when the slot's PREVIOUS occupant (the other thread's tile) has not even
  // landed yet, so the faster thread runs MMAs on stale bytes and releases a slot it does not own
  // (seen as non-deterministic outputs, lost arrivals and launch failures in stress runs).
  constexpr bool kSplit = (BM == 64) || (C::kOcc == 1);
  constexpr int kAhead = kSplit ? 2 : 1;
  constexpr int NSK = kSplit ? (C::NS + 1) / 2 : C::NS;
  constexpr int NSV = kSplit ? C::NS - NSK : C::NS;
  auto pos_k = [&](int i) -> int { return i < kAhead ? i : 2 * i - kAhead; };
  auto pos_v = [&](int j) -> int { const int a = 2 * j + kAhead + 1, t = j + n_it; return a < t ? a : t; };
  auto seq_k = [&](int i) -> int { return kSplit ? i : pos_k(i); };          // index in its ring
  auto seq_v = [&](int j) -> int { return kSplit ? j : pos_v(j); };
  auto slot_k = [&](int i) -> int { return seq_k(i) % NSK; };
  auto slot_v = [&](int j) -> int { return kSplit ? NSK + j % NSV : pos_v(j) % NSV; };

  if (n_it > 0) {
    if (warp == 4) {
      // ---- TMA producer: K(0..kAhead-1), then [K(j+kAhead), V(j)] for j = 0, 1, ... -------------
      if (lane == 0) {
        auto load = [&](const CUtensorMap* tm, int k0, int s, int seq, int ns) {
          mbar_wait(smem_u32(&ctl->kv_empty[s]), ((seq / ns) & 1) ^ 1);
          mbar_arrive_expect_tx(smem_u32(&ctl->kv_full[s]), C::KV_BYTES);
          tma_load_5d(smem_u32(kv_s + s * C::KV_BYTES), tm, smem_u32(&ctl->kv_full[s]), 0, k0, 0, g, b);
        };
        for (int i = early ? 1 : 0; i < kAhead && i < n_it; ++i)
          load(&tmK, start_of(cur_a, i), slot_k(i), seq_k(i), NSK);
        for (int j = 0; j < n_it; ++j) {
          const int i = j + kAhead;
          if (i < n_it) load(&tmK, start_of(cur_a, i), slot_k(i), seq_k(i), NSK);
          if (!(early && j == 0)) load(&tmV, start_of(cur_b, j), slot_v(j), seq_v(j), NSV);
        }
      }
    } else if (warp == 5 || warp == 6) {
      // ---- MMA issue.  QK(i): S(i) = Q K_i^T into S buffer i & 1, ahead of the softmax; PV(jj):
      // O += P(jj) V_jj.  kSplit: issued by two threads (warp 5: QK, warp 6: PV) -- tcgen05.mma
      // issue blocks while the pipe is busy and every mbarrier poll costs a lone thread ~100 clk, so
      // in one thread the waits and the issue of both products added up to the whole iteration
      // (clock64 trace: 420 clk of waits + 1100 clk of issue per 1700-clk iteration).  The two
      // streams share nothing: S vs O in TMEM, own rings, own commits.  Otherwise: one thread,
      // order QK(0) QK(1) PV(0) QK(2) PV(1) ... (measured 4 % faster there).
      if (lane == 0 && (warp == 5 || kSplit)) {
        constexpr uint32_t idesc_qk = umma_idesc_bf16(BM, BN, 0, 0);
        constexpr uint32_t idesc_pv = umma_idesc_bf16(BM, D, 0, 1);
        const uint32_t tS = tmem + (C::kSLane << 16) + C::S_COL, tO = tmem + C::O_COL;
        const uint32_t tQ = tmem + (C::kSLane << 16), tP = tmem + C::P_COL;
        const uint32_t q_a = smem_u32(q_s), p_a = smem_u32(p_s), kv_a = smem_u32(kv_s);
#ifdef BSA_TRACE
        const bool trace_on = blockIdx.x == gridDim.x / 2;
#endif
        auto issue_qk = [&](int i) {
          const int s = slot_k(i);
          TR(1, i, 0);
          mbar_wait(smem_u32(&ctl->kv_full[s]), (seq_k(i) / NSK) & 1);
          TR(1, i, 1);
          if (i >= 2) {
            if (C::kPTmem && !C::kQTmem)   // the S buffer also holds P(i-2): PV(i-2) must have consumed it
              mbar_wait(smem_u32(&ctl->o_done[i & 1]), ((i >> 1) & 1) ^ 1);
            else
              mbar_wait(smem_u32(&ctl->s_free[i & 1]), ((i >> 1) & 1) ^ 1);   // softmax(i-2) read it
          }
          tc_fence_after();
          TR(1, i, 2);
          const uint32_t k_a = kv_a + s * C::KV_BYTES;
#pragma unroll
          for (int ks = 0; ks < D / 16; ++ks) {
            const uint64_t bd = umma_smem_desc(k_a + (ks >> 2) * (BN * 128) + (ks & 3) * 32, 16, 1024);
            if (C::kQTmem) {   // A = Q from TMEM (same half-lane plane as S): 16 elements = 8 columns per K step
              umma_ts(tS + (i & 1) * BN, tQ + ks * 8, bd, idesc_qk, ks > 0);
            } else {
              const uint64_t ad = umma_smem_desc(q_a + (ks >> 2) * (BM * 128) + (ks & 3) * 32, 16, 1024);
              umma_ss(tS + (i & 1) * BN, ad, bd, idesc_qk, ks > 0);
            }
          }
          tc_commit(smem_u32(&ctl->kv_empty[s]));
          tc_commit(smem_u32(&ctl->s_full[i & 1]));
          TR(1, i, 3);
        };
        auto issue_pv = [&](int jj) {
          const int s = slot_v(jj);
          TR(2, jj, 0);
          mbar_wait(smem_u32(&ctl->kv_full[s]), (seq_v(jj) / NSV) & 1);
          TR(2, jj, 1);
          const int pb = C::kPTmem ? (jj & 1) : 0;       // o_done barrier: per S buffer when P lives there
          mbar_wait(smem_u32(&ctl->p_full[pb]), C::kPTmem ? ((jj >> 1) & 1) : (jj & 1));
          tc_fence_after();
          TR(2, jj, 2);
          const uint32_t v_a = kv_a + s * C::KV_BYTES;
#pragma unroll
          for (int ks = 0; ks < BN / 16; ++ks) {
            const uint64_t bd = umma_smem_desc(v_a + ks * 2048, BN * 128, 1024);
            if (C::kPTmem) {   // A = P(jj) from TMEM: 16 keys = 8 columns of bf16 pairs per K step
              umma_ts(tO, tP + (jj & 1) * C::kPStride + ks * 8, bd, idesc_pv, (jj > 0) || (ks > 0));
            } else {
              const uint64_t ad = umma_smem_desc(p_a + ks * 32, 16, 1024);
              umma_ss(tO, ad, bd, idesc_pv, (jj > 0) || (ks > 0));
            }
          }
          tc_commit(smem_u32(&ctl->kv_empty[s]));
          tc_commit(smem_u32(&ctl->o_done[pb]));
          TR(2, jj, 3);
        };
        if (kSplit) {
          if (warp == 5) {
            mbar_wait(smem_u32(&ctl->q_full), 0);
            for (int i = 0; i < n_it; ++i) issue_qk(i);
          } else {
            for (int jj = 0; jj < n_it; ++jj) issue_pv(jj);
          }
        } else {
          mbar_wait(smem_u32(&ctl->q_full), 0);
          issue_qk(0);
          for (int jj = 0; jj < n_it; ++jj) {
            if (jj + 1 < n_it) issue_qk(jj + 1);
            issue_pv(jj);
          }
        }
      }
    } else if (warp < 4) {
      // ---- softmax warps ---------------------------------------------------------------------
      if constexpr (BM == 64) {
        softmax_m64<D, SPARSE>(p, ctl, p_s, tmem, n_it, q0, b, h, key_start, qreg);
      } else {
        softmax_m128<D, SPARSE>(p, ctl, p_s, tmem, n_it, q0, b, h, key_start);
      }
    }
  } else if (warp < 4) {
    // nothing attended (possible only with a caller-provided kv_idx): zeros, lse = -inf
    if constexpr (!C::kQTmem) mbar_wait(smem_u32(&ctl->q_full), 0);   // the Q tile load must land before the CTA may exit
    const bool active = (BM == 128) || (lane < 16);
    const int r = (BM == 128) ? tid : (warp * 16 + (lane & 15));
    const int qrow = q0 + r;
    if (active && qrow < p.N) {
      uint16_t* orow = p.O + b * p.qsb + h * p.qsh + static_cast<int64_t>(qrow) * p.qsn;
      for (int c = 0; c < D; c += 8) *reinterpret_cast<uint4*>(orow + c) = make_uint4(0, 0, 0, 0);
      if (p.lse) p.lse[(static_cast<int64_t>(b) * p.H + h) * p.N + qrow] = -INFINITY;
    }
  }

  // ---- teardown ------------------------------------------------------------------------------
  tc_fence_before();
  __syncthreads();
  TR(3, 0, 6);
  if (warp == 4) tmem_dealloc<C::TMEM_COLS>(tmem);
}


// =================================================================================================
// Persistent variant for 64-token blocks in list mode (round 2c).
//
// A clock64 trace of attn_kernel<64,128,true> at C2 showed ~10.5k clk of every CTA's 51k-86k outside
// the steady-state loop: barrier / TMEM set-up and the kv_idx row (4.4k), the first TMA round trip
// (2.2k), the wait for the last PV (2.0k), the epilogue (1.2k) and the teardown (0.7k) -- and a CTA that
// is not in its loop leaves the tensor pipe to its single co-resident CTA, which alone cannot fill it.
// Here 2 x #SM CTAs stay resident and walk through the (tile, head) items; every role runs ahead across
// item boundaries on its own:
//   warp 7     scheduler + list builder, one item ahead: fetches the next item from a work counter
//              (dynamic: the items' lengths differ by 2x between routed and unrouted tiles), compacts
//              its kv_idx row into list[n & 1]
//   warp 4     TMA producer: keeps the K / V rings full across items
//   warp 5 / 6 QK / PV issue; buffers and mbarrier phases are indexed by a running iteration count
//   warps 0-3  softmax; after the last iteration of an item they fetch the NEXT item's Q tile and put it
//              into TMEM while the last PV drains, so QK(0) of the next item runs under this item's epilogue
// Items with an empty list are written as zeros by the softmax warps and are invisible to the other
// roles' barriers.  Same arithmetic, in the same order, as attn_kernel: outputs are bit-identical.
// =================================================================================================
constexpr int kMaxWP = 128;          // widest kv_idx row of the persistent kernel (two lists fit the 1 KB block)
constexpr int kThreadsP = 256;
constexpr int kCounterSlots = 1024;  // work counters: one per launch in flight (a launch takes slot
                                     // ticket % 1024 and its last CTA clears it)
__device__ unsigned int g_work_counter[kCounterSlots];
__device__ unsigned int g_work_done[kCounterSlots];

struct alignas(8) CtlP {
  uint64_t q_full, o_free;
  uint64_t p_full[2], s_full[2], s_free[2], o_done[2];
  uint64_t list_full[2], list_free[2];
  uint64_t kv_full[8], kv_empty[8];
  uint32_t tmem_base;
  int32_t item[2];             // work item of list buffer b, -1 = no more work
  int32_t n_valid[2];
  int32_t tq[2], kvh[2], bat[2], qh[2];   // the item decoded by the scheduler warp (tile, KV head, batch, head)
  uint16_t list[2][kMaxWP];
};
static_assert(sizeof(CtlP) <= 1024, "CtlP must fit the 1 KB bookkeeping area");

struct ItemP {
  int tq, g, b, h, q0;
};
__device__ __forceinline__ ItemP decode_item(const Params& p, int wi) {
  ItemP it;
  const int hi = wi % p.G;
  wi /= p.G;
  it.tq = p.NT - 1 - wi % p.NT;
  wi /= p.NT;
  const int Hkv = p.H / p.G;
  it.g = wi % Hkv;
  it.b = wi / Hkv;
  it.h = it.g * p.G + hi;
  it.q0 = it.tq * 64;
  return it;
}

__device__ __forceinline__ ItemP read_item(const CtlP* ctl, int buf) {
  ItemP it;
  it.tq = ctl->tq[buf]; it.g = ctl->kvh[buf]; it.b = ctl->bat[buf]; it.h = ctl->qh[buf];
  it.q0 = it.tq * 64;
  return it;
}

template <int D>
__global__ void __launch_bounds__(kThreadsP, Cfg<64, D>::kOcc)
attn64p_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV, const Params p,
               const int n_items, const int cslot) {
  using C = Cfg<64, D>;
  static_assert(C::kQTmem, "the persistent kernel keeps Q in TMEM");
  extern __shared__ __align__(1024) uint8_t smem[];
  uint8_t* kv_s = smem;
  CtlP* ctl = reinterpret_cast<CtlP*>(kv_s + C::NS * C::KV_BYTES);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  constexpr int NSK = (C::NS + 1) / 2, NSV = C::NS - NSK;
  // Q is double buffered in plane 1 (buffer = index of the non-empty item & 1): the second copy sits in the
  // columns the one-item kernel leaves unused, so the next item's tile can be written during this item's loop
  constexpr uint32_t kQ1Col = (D == 256) ? 256 : 192;
  constexpr int kQChunks = D / 32;   // 16-column (32-element) pieces of a Q tile, one per late iteration
  if ((smem_u32(smem) & 1023u) != 0) __trap();

  if (warp == 4) {
    if (lane == 0) {
      mbar_init(smem_u32(&ctl->q_full), 4);
      mbar_init(smem_u32(&ctl->o_free), 4);
      for (int i = 0; i < 2; ++i) {
        mbar_init(smem_u32(&ctl->p_full[i]), 4);
        mbar_init(smem_u32(&ctl->s_full[i]), 1);
        mbar_init(smem_u32(&ctl->s_free[i]), 4);
        mbar_init(smem_u32(&ctl->o_done[i]), 1);
        mbar_init(smem_u32(&ctl->list_full[i]), 1);
        mbar_init(smem_u32(&ctl->list_free[i]), 7);   // 4 softmax warps, producer, QK thread, PV thread
      }
      for (int s = 0; s < C::NS; ++s) {
        mbar_init(smem_u32(&ctl->kv_full[s]), 1);
        mbar_init(smem_u32(&ctl->kv_empty[s]), 1);
      }
      fence_mbar_init();
      tma_prefetch_desc(&tmK);
      tma_prefetch_desc(&tmV);
    }
    __syncwarp();
    tmem_alloc<C::TMEM_COLS>(smem_u32(&ctl->tmem_base));
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = ctl->tmem_base;

  if (warp == 7) {
    // ---- scheduler + list builder, one item ahead of everybody else ------------------------------------
    if (p.pdl) griddep_wait();
    for (int n = 0;; ++n) {
      const int buf = n & 1;
      if (n >= 2) mbar_wait(smem_u32(&ctl->list_free[buf]), ((n - 2) >> 1) & 1);
      int wi = 0;
      if (lane == 0) wi = static_cast<int>(atomicAdd(&g_work_counter[cslot], 1u));
      wi = __shfl_sync(0xffffffffu, wi, 0);
      if (wi >= n_items) {
        if (lane == 0) {
          ctl->item[buf] = -1;
          mbar_arrive(smem_u32(&ctl->list_full[buf]));
        }
        break;
      }
      const ItemP it = decode_item(p, wi);
      const int64_t row = (static_cast<int64_t>(it.b) * p.H + it.h) * p.NT + it.tq;
      const int32_t* src = p.kv_idx + row * p.W;
      int blkv[kMaxWP / 32];
#pragma unroll
      for (int c = 0; c < kMaxWP / 32; ++c) blkv[c] = (c * 32 + lane < p.W) ? __ldg(src + c * 32 + lane) : -1;
      int cnt = p.kv_count ? __ldg(p.kv_count + row) : p.W;
      cnt = cnt < 0 ? 0 : (cnt > p.W ? p.W : cnt);
      const unsigned lt = (1u << lane) - 1u;
      uint16_t* list = ctl->list[buf];
      int base = 0;
#pragma unroll
      for (int c = 0; c < kMaxWP / 32; ++c) {
        if (c * 32 < cnt) {
          const int i = c * 32 + lane;
          const int blk = (i < cnt) ? blkv[c] : -1;
          bool ok = (blk >= 0) && (blk < p.NB) && (blk <= it.tq);
          // a block listed more than once is attended once (O11): lowest position wins
          const unsigned same = __match_any_sync(0xffffffffu, ok ? blk : -1 - lane);
          if (same & lt) ok = false;
          if (c > 0 && ok) {
            for (int u = 0; u < base; ++u)
              if (list[u] == static_cast<uint16_t>(blk)) { ok = false; break; }
          }
          const unsigned bal = __ballot_sync(0xffffffffu, ok);
          if (ok) list[base + __popc(bal & lt)] = static_cast<uint16_t>(blk);
          base += __popc(bal);
          __syncwarp();
        }
      }
      __syncwarp();
      if (lane == 0) {
        ctl->item[buf] = wi;
        ctl->n_valid[buf] = base;
        ctl->tq[buf] = it.tq; ctl->kvh[buf] = it.g; ctl->bat[buf] = it.b; ctl->qh[buf] = it.h;
        mbar_arrive(smem_u32(&ctl->list_full[buf]));
      }
    }
  } else if (warp == 4) {
    // ---- TMA producer: per item K(0), K(1), then [K(j+2), V(j)]; ring positions run across items --------
    if (lane == 0) {
      uint32_t gk = 0, gv = 0;
      auto load = [&](const CUtensorMap* tm, int k0, int s, uint32_t use, const ItemP& it) {
        mbar_wait(smem_u32(&ctl->kv_empty[s]), (use & 1) ^ 1);
        mbar_arrive_expect_tx(smem_u32(&ctl->kv_full[s]), C::KV_BYTES);
        tma_load_5d(smem_u32(kv_s + s * C::KV_BYTES), tm, smem_u32(&ctl->kv_full[s]), 0, k0, 0, it.g, it.b);
      };
      for (int n = 0;; ++n) {
        const int buf = n & 1;
        mbar_wait(smem_u32(&ctl->list_full[buf]), (n >> 1) & 1);
        const int wi = ctl->item[buf];
        if (wi < 0) break;
        const ItemP it = read_item(ctl, buf);
        const int n_it = ctl->n_valid[buf];
        const uint16_t* list = ctl->list[buf];
        auto ldk = [&](int i) { load(&tmK, static_cast<int>(list[i]) * 64, gk % NSK, gk / NSK, it); ++gk; };
        auto ldv = [&](int j) { load(&tmV, static_cast<int>(list[j]) * 64, NSK + gv % NSV, gv / NSV, it); ++gv; };
        for (int i = 0; i < 2 && i < n_it; ++i) ldk(i);
        for (int j = 0; j < n_it; ++j) {
          if (j + 2 < n_it) ldk(j + 2);
          ldv(j);
        }
        mbar_arrive(smem_u32(&ctl->list_free[buf]));
      }
    }
  } else if (warp == 5) {
    // ---- QK issue: S(gi) = Q K^T (TS form, A = Q in TMEM plane 1) into S buffer gi & 1 ----------------------
    if (lane == 0) {
      constexpr uint32_t idesc_qk = umma_idesc_bf16(64, BN, 0, 0);
      const uint32_t tS = tmem + (C::kSLane << 16) + C::S_COL, tQ = tmem + (C::kSLane << 16);
      const uint32_t kv_a = smem_u32(kv_s);
      uint32_t gi = 0, gk = 0, ne = 0;   // running iteration, K ring position, non-empty items so far
      for (int n = 0;; ++n) {
        const int buf = n & 1;
        mbar_wait(smem_u32(&ctl->list_full[buf]), (n >> 1) & 1);
        const int wi = ctl->item[buf];
        const int n_it = ctl->n_valid[buf];
        if (wi < 0) break;
        mbar_arrive(smem_u32(&ctl->list_free[buf]));
        if (n_it == 0) continue;
        mbar_wait(smem_u32(&ctl->q_full), ne & 1);   // this item's Q tile is in TMEM, buffer ne & 1
        const uint32_t tQn = tQ + (ne & 1) * kQ1Col;
        ++ne;
        for (int i = 0; i < n_it; ++i, ++gi, ++gk) {
          const int s = gk % NSK;
          mbar_wait(smem_u32(&ctl->kv_full[s]), (gk / NSK) & 1);
          if (gi >= 2) mbar_wait(smem_u32(&ctl->s_free[gi & 1]), ((gi >> 1) & 1) ^ 1);   // softmax(gi-2) read it
          tc_fence_after();
          const uint32_t k_a = kv_a + s * C::KV_BYTES;
#pragma unroll
          for (int ks = 0; ks < D / 16; ++ks) {
            const uint64_t bd = umma_smem_desc(k_a + (ks >> 2) * (BN * 128) + (ks & 3) * 32, 16, 1024);
            umma_ts(tS + (gi & 1) * BN, tQn + ks * 8, bd, idesc_qk, ks > 0);
          }
          tc_commit(smem_u32(&ctl->kv_empty[s]));
          tc_commit(smem_u32(&ctl->s_full[gi & 1]));
        }
      }
    }
  } else if (warp == 6) {
    // ---- PV issue: O += P(gj) V (TS form, A = P in TMEM plane 0) -----------------------------------------------
    if (lane == 0) {
      constexpr uint32_t idesc_pv = umma_idesc_bf16(64, D, 0, 1);
      const uint32_t tO = tmem + C::O_COL, tP = tmem + C::P_COL;
      const uint32_t kv_a = smem_u32(kv_s);
      uint32_t gj = 0, gv = 0, ne = 0;
      for (int n = 0;; ++n) {
        const int buf = n & 1;
        mbar_wait(smem_u32(&ctl->list_full[buf]), (n >> 1) & 1);
        const int wi = ctl->item[buf];
        const int n_it = ctl->n_valid[buf];
        if (wi < 0) break;
        mbar_arrive(smem_u32(&ctl->list_free[buf]));
        if (n_it == 0) continue;
        if (ne > 0) mbar_wait(smem_u32(&ctl->o_free), (ne - 1) & 1);   // the previous item's epilogue has read O
        ++ne;
        for (int jj = 0; jj < n_it; ++jj, ++gj, ++gv) {
          const int s = NSK + gv % NSV;
          mbar_wait(smem_u32(&ctl->kv_full[s]), (gv / NSV) & 1);
          mbar_wait(smem_u32(&ctl->p_full[gj & 1]), (gj >> 1) & 1);
          tc_fence_after();
          const uint32_t v_a = kv_a + s * C::KV_BYTES;
#pragma unroll
          for (int ks = 0; ks < BN / 16; ++ks) {
            const uint64_t bd = umma_smem_desc(v_a + ks * 2048, BN * 128, 1024);
            umma_ts(tO, tP + (gj & 1) * C::kPStride + ks * 8, bd, idesc_pv, (jj > 0) || (ks > 0));
          }
          tc_commit(smem_u32(&ctl->kv_empty[s]));
          tc_commit(smem_u32(&ctl->o_done[gj & 1]));
        }
      }
    }
  } else if (warp < 4) {
    // ---- softmax warps ------------------------------------------------------------------------------------------
    const int quad = lane & 3;
    const int rA = warp * 16 + (lane >> 2);
    const uint32_t lane_base = static_cast<uint32_t>(warp * 32) << 16;
    const uint32_t tS = tmem + lane_base + (C::kSLane << 16) + C::S_COL;
    const uint32_t tQ = tmem + lane_base + (C::kSLane << 16);
    const uint32_t tO = tmem + lane_base + C::O_COL;
    const uint32_t tP = tmem + lane_base + C::P_COL;
    const float sc = p.scale_log2;
    uint32_t gj = 0, ne = 0;    // running iteration count / non-empty items so far
    bool q_ready = false;       // the current item's Q tile was already put into TMEM during the previous item
    auto post_q = [&]() {
      tmem_st_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctl->q_full));
    };
    auto put_q = [&](const ItemP& it, uint32_t tq_dst) {   // the whole tile at once (first item, short items)
      uint32_t qr[D / 64][16];
      load_q_m64<D>(p, it.q0, it.b, it.h, qr);
#pragma unroll
      for (int c = 0; c < D / 64; ++c) tmem_st16x128_x8(tq_dst + 32 * c, qr[c]);
      post_q();
    };
    for (int n = 0;; ++n) {
      const int buf = n & 1;
      mbar_wait(smem_u32(&ctl->list_full[buf]), (n >> 1) & 1);
      if (ctl->item[buf] < 0) break;
      const int n_it = ctl->n_valid[buf];
      const int q0 = ctl->tq[buf] * 64;
      const uint16_t* list = ctl->list[buf];
#ifdef BSA_TRACE
      const bool trace_on = blockIdx.x == gridDim.x / 2 && tid == 0;
#endif
      TR(0, n, 0);
      if (n_it == 0) {
        // nothing attended (possible only with a caller-provided kv_idx): zeros, lse = -inf
        const ItemP it = read_item(ctl, buf);
        uint16_t* orowA = p.O + it.b * p.qsb + it.h * p.qsh + static_cast<int64_t>(q0 + rA) * p.qsn + 2 * quad;
        uint16_t* orowB = orowA + 8 * p.qsn;
#pragma unroll
        for (int c = 0; c < D; c += 8) {
          *reinterpret_cast<uint32_t*>(orowA + c) = 0u;
          *reinterpret_cast<uint32_t*>(orowB + c) = 0u;
        }
        if (p.lse && quad == 0) {
          float* lse = p.lse + (static_cast<int64_t>(it.b) * p.H + it.h) * p.N + q0 + rA;
          lse[0] = -INFINITY;
          lse[8] = -INFINITY;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctl->list_free[buf]));
        continue;
      }
      if (!q_ready) put_q(read_item(ctl, buf), tQ + (ne & 1) * kQ1Col);
      q_ready = false;
      ++ne;
      const uint32_t tQnext = tQ + (ne & 1) * kQ1Col;   // where the next non-empty item's tile goes
      float mA = -INFINITY, mB = -INFINITY, lA = 0.f, lB = 0.f;

      // One iteration.  PIECE: the iteration also carries a 16-column piece of the NEXT item's Q tile (8 loads
      // at its top, one store at its end) -- the last kQChunks iterations of an item, if the scheduler has
      // posted the next item by then.  Two instances of the body keep the pieces' registers out of the main loop.
      auto iteration = [&](const int j, auto piece_tag, const uint16_t* qnA, const int pc) {
        constexpr bool PIECE = decltype(piece_tag)::value;
        const int k0 = static_cast<int>(list[j]) * 64;
        uint32_t qn[8];
        if constexpr (PIECE) {
          const uint16_t* a = qnA + 32 * pc;
          const uint16_t* bq = a + 8 * p.qsn;
#pragma unroll
          for (int g = 0; g < 4; ++g) {
            qn[2 * g] = __ldg(reinterpret_cast<const uint32_t*>(a + 8 * g));
            qn[2 * g + 1] = __ldg(reinterpret_cast<const uint32_t*>(bq + 8 * g));
          }
        }
        if (gj >= 2) {
          // S(gj) ready, and PV(gj-2) done so that P(gj) may later overwrite P(gj-2): one poll for both
          mbar_wait2_warp(smem_u32(&ctl->s_full[gj & 1]), (gj >> 1) & 1, smem_u32(&ctl->o_done[gj & 1]),
                          ((gj - 2) >> 1) & 1);
        } else {
          mbar_wait(smem_u32(&ctl->s_full[gj & 1]), (gj >> 1) & 1);
        }
        tc_fence_after();
        uint32_t s[32];
        tmem_ld16x256_x8(tS + (gj & 1) * BN, s);
        tmem_ld_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctl->s_free[gj & 1]));   // QK(gj+2) may overwrite S(gj)

        float xa[16], xb[16];
#pragma unroll
        for (int g = 0; g < 8; ++g) {
          xa[2 * g] = __uint_as_float(s[4 * g]);
          xa[2 * g + 1] = __uint_as_float(s[4 * g + 1]);
          xb[2 * g] = __uint_as_float(s[4 * g + 2]);
          xb[2 * g + 1] = __uint_as_float(s[4 * g + 3]);
        }
        if (k0 + BN - 1 > q0) {
          const int qrA = q0 + rA, qrB = qrA + 8;
#pragma unroll
          for (int g = 0; g < 8; ++g) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
              const int key = k0 + 8 * g + 2 * quad + e;
              xa[2 * g + e] = (key <= qrA) ? xa[2 * g + e] : -INFINITY;
              xb[2 * g + e] = (key <= qrB) ? xb[2 * g + e] : -INFINITY;
            }
          }
        }
        float mxA = fmaxf(xa[0], xa[1]), mxB = fmaxf(xb[0], xb[1]);
#pragma unroll
        for (int c = 2; c < 16; c += 2) {
          mxA = fmax3(mxA, xa[c], xa[c + 1]);
          mxB = fmax3(mxB, xb[c], xb[c + 1]);
        }
        const bool any = __any_sync(0xffffffffu, (fmaf(mxA, sc, -mA) > 8.0f) || (fmaf(mxB, sc, -mB) > 8.0f));
        float mA_new = mA, mB_new = mB, alphaA = 1.0f, alphaB = 1.0f;
        if (any) {
          mxA = fmaxf(mxA, __shfl_xor_sync(0xffffffffu, mxA, 1));
          mxB = fmaxf(mxB, __shfl_xor_sync(0xffffffffu, mxB, 1));
          mxA = fmaxf(mxA, __shfl_xor_sync(0xffffffffu, mxA, 2));
          mxB = fmaxf(mxB, __shfl_xor_sync(0xffffffffu, mxB, 2));
          mA_new = fmaxf(mA, mxA * sc);
          mB_new = fmaxf(mB, mxB * sc);
          alphaA = ex2_approx(mA - mA_new);
          alphaB = ex2_approx(mB - mB_new);
        }
        float2 sumA2 = make_float2(0.f, 0.f), sumB2 = make_float2(0.f, 0.f);
        const float2 sc2 = make_float2(sc, sc);
        const float2 nmA = make_float2(-mA_new, -mA_new), nmB = make_float2(-mB_new, -mB_new);
        uint32_t pr[16];
#pragma unroll
        for (int g = 0; g < 8; ++g) {
          const float2 ta = ffma2(make_float2(xa[2 * g], xa[2 * g + 1]), sc2, nmA);
          const float2 tb = ffma2(make_float2(xb[2 * g], xb[2 * g + 1]), sc2, nmB);
          const float2 ea = make_float2(ex2_approx(ta.x), ex2_approx(ta.y));
          const float2 eb = make_float2(ex2_approx(tb.x), ex2_approx(tb.y));
          sumA2 = fadd2(sumA2, ea);
          sumB2 = fadd2(sumB2, eb);
          pr[2 * g] = pack_bf16x2(ea.x, ea.y);
          pr[2 * g + 1] = pack_bf16x2(eb.x, eb.y);
        }
        lA = lA * alphaA + (sumA2.x + sumA2.y);
        lB = lB * alphaB + (sumB2.x + sumB2.y);
        mA = mA_new;
        mB = mB_new;

        if (any && j > 0) {
          // the rare rescale touches O: every earlier PV of this item must be done (they complete in order)
          mbar_wait(smem_u32(&ctl->o_done[(gj - 1) & 1]), ((gj - 1) >> 1) & 1);
          tc_fence_after();
#pragma unroll
          for (int c0 = 0; c0 < D; c0 += 64) {
            uint32_t o[32];
            tmem_ld16x256_x8(tO + c0, o);
            tmem_ld_wait();
#pragma unroll
            for (int g = 0; g < 8; ++g) {
              o[4 * g] = __float_as_uint(__uint_as_float(o[4 * g]) * alphaA);
              o[4 * g + 1] = __float_as_uint(__uint_as_float(o[4 * g + 1]) * alphaA);
              o[4 * g + 2] = __float_as_uint(__uint_as_float(o[4 * g + 2]) * alphaB);
              o[4 * g + 3] = __float_as_uint(__uint_as_float(o[4 * g + 3]) * alphaB);
            }
            tmem_st16x256_x8(tO + c0, o);
          }
          tmem_st_wait();
        }
        tmem_st16x128_x8(tP + (gj & 1) * C::kPStride, pr);
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctl->p_full[gj & 1]));
        if constexpr (PIECE) tmem_st16x128_x4(tQnext + 16 * pc, qn);   // completes under the next iteration
        ++gj;
      };

      const int n_main = n_it >= kQChunks ? n_it - kQChunks : n_it;
      int j = 0;
      for (; j < n_main; ++j) {
        if (j == 1) TR(0, n, 1);
        iteration(j, std::false_type{}, nullptr, 0);
      }
      bool pieces = false;
      if (j < n_it) {
        // the last kQChunks iterations: is the next item posted and not empty?
        const int nb = (n + 1) & 1;
        bool have = mbar_try_wait(smem_u32(&ctl->list_full[nb]), ((n + 1) >> 1) & 1);
        have = __all_sync(0xffffffffu, have);
        pieces = have && ctl->item[nb] >= 0 && ctl->n_valid[nb] > 0;
        if (pieces) {
          const ItemP nx = read_item(ctl, nb);
          const uint16_t* qnA =
              p.Q + nx.b * p.qsb + nx.h * p.qsh + static_cast<int64_t>(nx.q0 + rA) * p.qsn + 2 * quad;
          for (int pc = 0; j < n_it; ++j, ++pc) iteration(j, std::true_type{}, qnA, pc);
        } else {
          for (; j < n_it; ++j) iteration(j, std::false_type{}, nullptr, 0);
        }
      }
      // ---- item boundary -----------------------------------------------------------------------------------------
      TR(0, n, 2);
      if (pieces) {
        post_q();           // the pieces are in TMEM: QK(0) of the next item may start now
        q_ready = true;
      } else {
        // not fetched during the loop (short item, or the scheduler was late): fetch it now, while the last PV
        // drains.  The other Q buffer is free: its item's QKs completed before this item's first s_full.
        const int nb = (n + 1) & 1;
        mbar_wait(smem_u32(&ctl->list_full[nb]), ((n + 1) >> 1) & 1);
        if (ctl->item[nb] >= 0 && ctl->n_valid[nb] > 0) {
          put_q(read_item(ctl, nb), tQnext);
          q_ready = true;
        }
      }
      // ---- epilogue: O / l -> bf16 -> global -----------------------------------------------------------------
      TR(0, n, 3);
      mbar_wait(smem_u32(&ctl->o_done[(gj - 1) & 1]), ((gj - 1) >> 1) & 1);
      tc_fence_after();
      TR(0, n, 4);
      lA += __shfl_xor_sync(0xffffffffu, lA, 1);
      lB += __shfl_xor_sync(0xffffffffu, lB, 1);
      lA += __shfl_xor_sync(0xffffffffu, lA, 2);
      lB += __shfl_xor_sync(0xffffffffu, lB, 2);
      const float invA = 1.0f / lA, invB = 1.0f / lB;
#ifdef BSA_TRACE
      if (trace_on && n < 32) g_tr[1][n][0] = clock64();
#endif
      const ItemP it = read_item(ctl, buf);
      uint16_t* orowA = p.O + it.b * p.qsb + it.h * p.qsh + static_cast<int64_t>(q0 + rA) * p.qsn;
      uint16_t* orowB = orowA + 8 * p.qsn;
      // All of O into registers first, then the two arrivals, then the stores: mbarrier.arrive has release
      // semantics, and an arrival AFTER the global stores waited ~800 clk for them (clock64 trace).
      uint32_t o[D / 64][32];
#pragma unroll
      for (int c = 0; c < D / 64; ++c) tmem_ld16x256_x8(tO + 64 * c, o[c]);
      tmem_ld_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(smem_u32(&ctl->o_free));          // the next item's first PV may overwrite O
        mbar_arrive(smem_u32(&ctl->list_free[buf]));  // nothing of this item's list / ctl fields is read below
      }
#ifdef BSA_TRACE
      if (trace_on && n < 32) g_tr[1][n][2] = clock64();
#endif
#pragma unroll
      for (int c = 0; c < D / 64; ++c) {
        uint32_t wa[8], wb[8];
#pragma unroll
        for (int g = 0; g < 8; ++g) {
          wa[g] = pack_bf16x2(__uint_as_float(o[c][4 * g]) * invA, __uint_as_float(o[c][4 * g + 1]) * invA);
          wb[g] = pack_bf16x2(__uint_as_float(o[c][4 * g + 2]) * invB, __uint_as_float(o[c][4 * g + 3]) * invB);
        }
#pragma unroll
        for (int g0 = 0; g0 < 8; g0 += 4) {
          const uint4 va = quad_gather(wa[g0], wa[g0 + 1], wa[g0 + 2], wa[g0 + 3], quad);
          const uint4 vb = quad_gather(wb[g0], wb[g0 + 1], wb[g0 + 2], wb[g0 + 3], quad);
          *reinterpret_cast<uint4*>(orowA + 64 * c + 8 * (g0 + quad)) = va;
          *reinterpret_cast<uint4*>(orowB + 64 * c + 8 * (g0 + quad)) = vb;
        }
      }
#ifdef BSA_TRACE
      if (trace_on && n < 32) g_tr[1][n][5] = clock64();
#endif
      if (p.lse && quad == 0) {
        float* lse = p.lse + (static_cast<int64_t>(it.b) * p.H + it.h) * p.N + q0 + rA;
        lse[0] = (mA + log2f(lA)) * 0.6931471805599453f;
        lse[8] = (mB + log2f(lB)) * 0.6931471805599453f;
      }
#ifdef BSA_TRACE
      TR(0, n, 5);
      if (trace_on && n < 32) g_tr[0][n][6] = n_it;
#endif
    }
  }

  // ---- teardown ------------------------------------------------------------------------------------
  tc_fence_before();
  __syncthreads();
  if (warp == 4) tmem_dealloc<C::TMEM_COLS>(tmem);
  if (tid == 0) {
    // the last CTA of the launch returns the work counter to zero for the launch that takes this slot next
    __threadfence();
    if (atomicAdd(&g_work_done[cslot], 1u) == gridDim.x - 1) {
      g_work_counter[cslot] = 0u;
      g_work_done[cslot] = 0u;
      __threadfence();
    }
  }
}

// ---- host side ---------------------------------------------------------------------------------
template <int BM, int D, bool SPARSE>
bsa_status run(const Dims& S, const void* Q, const void* K, const void* V, const Params& prm,
               cudaStream_t stream) {
  using C = Cfg<BM, D>;
  CUtensorMap tq, tk, tv;
  if (!make_tmap_bhnd(&tq, Q, S.B, S.H, S.N, S.d, S.qsb, S.qsh, S.qsn, BM, S.d / 64, 1) ||
      !make_tmap_bhnd(&tk, K, S.B, S.Hkv, S.N, S.d, S.ksb, S.ksh, S.ksn, BN, S.d / 64, 1) ||
      !make_tmap_bhnd(&tv, V, S.B, S.Hkv, S.N, S.d, S.ksb, S.ksh, S.ksn, BN, S.d / 64, 1))
    return fail(BSA_ERR_CUDA, "attn: cuTensorMapEncodeTiled failed");
  auto kern = attn_kernel<BM, D, SPARSE>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM);
  if (e != cudaSuccess) return fail(BSA_ERR_CUDA, "attn: smem attribute: %s", cudaGetErrorString(e));
  const unsigned grid = static_cast<unsigned>(prm.NT) * prm.B * prm.H;
  if (prm.pdl) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = C::SMEM;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    e = cudaLaunchKernelEx(&cfg, kern, tq, tk, tv, prm);
    if (e != cudaSuccess) return fail(BSA_ERR_CUDA, "attn: cudaLaunchKernelEx: %s", cudaGetErrorString(e));
  } else {
    kern<<<grid, kThreads, C::SMEM, stream>>>(tq, tk, tv, prm);
  }
  return check_launch("attn_kernel");
}


// one ticket sequence for every head_dim instantiation: two launches in flight never share a counter slot
std::atomic<unsigned> g_ticket{0};

template <int D>
bsa_status run_persistent(const Dims& S, const void* K, const void* V, const Params& prm, cudaStream_t stream) {
  using C = Cfg<64, D>;
  CUtensorMap tk, tv;
  if (!make_tmap_bhnd(&tk, K, S.B, S.Hkv, S.N, S.d, S.ksb, S.ksh, S.ksn, BN, S.d / 64, 1) ||
      !make_tmap_bhnd(&tv, V, S.B, S.Hkv, S.N, S.d, S.ksb, S.ksh, S.ksn, BN, S.d / 64, 1))
    return fail(BSA_ERR_CUDA, "attn: cuTensorMapEncodeTiled failed");
  auto kern = attn64p_kernel<D>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM);
  if (e != cudaSuccess) return fail(BSA_ERR_CUDA, "attn: smem attribute: %s", cudaGetErrorString(e));
  const long long items = static_cast<long long>(prm.NT) * prm.B * prm.H;
  const long long slots = static_cast<long long>(sm_count()) * C::kOcc;
  const unsigned grid = static_cast<unsigned>(items < slots ? items : slots);
  const int cslot = static_cast<int>(g_ticket.fetch_add(1u) % kCounterSlots);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(kThreadsP);
  cfg.dynamicSmemBytes = C::SMEM;
  cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = prm.pdl ? 1 : 0;
  e = cudaLaunchKernelEx(&cfg, kern, tk, tv, prm, static_cast<int>(items), cslot);
  if (e != cudaSuccess) return fail(BSA_ERR_CUDA, "attn: cudaLaunchKernelEx: %s", cudaGetErrorString(e));
  return check_launch("attn64p_kernel");
}

}  // namespace

// The transposed kernel of attn_t.cu (keys on the M dimension, M = 128) is parity-green but slower than
// the M = 64 kernel here on B200 (C2: 2.3-2.7 ms against 1.5 ms; ablation in DESIGN.md section 6), so it
// is an opt-in experiment: the environment variable BSA_ATTN_T=1 routes block 64 / head_dim 128 to it.
// BSA_ATTN_PERSISTENT=0 routes block 64 back to the one-CTA-per-item kernel (A/B runs).
static bool attn_persistent_enabled() {
  const char* e = getenv("BSA_ATTN_PERSISTENT");
  return e == nullptr || e[0] != '0';
}

static bool attn_t_enabled() {
  const char* e = getenv("BSA_ATTN_T");
  return e != nullptr && e[0] == '1';
}

bsa_status launch_attn(const Dims& S, const void* Q, const void* K, const void* V,
                       const int32_t* kv_idx, const int32_t* kv_count, int W, bool sparse, float scale,
                       void* O, float* lse, cudaStream_t stream, const uint32_t* bitmap, bool pdl) {
  Params prm;
  prm.pdl = pdl ? 1 : 0;
  prm.kv_idx = kv_idx;
  prm.kv_count = kv_count;
  prm.bitmap = bitmap;
  prm.nbw = (S.NB + 31) / 32;
  if (bitmap && S.NB > 32 * (kMaxW / 2))
    return fail(BSA_ERR_UNSUPPORTED, "bitmap attention: %d blocks per sequence, at most %d", S.NB,
                32 * (kMaxW / 2));
  prm.Q = static_cast<const uint16_t*>(Q);
  prm.O = static_cast<uint16_t*>(O);
  prm.lse = lse;
  prm.W = W;
  prm.B = S.B; prm.H = S.H; prm.G = S.G; prm.N = S.N; prm.Bn = S.Bn; prm.NB = S.NB;
  prm.qsb = S.qsb; prm.qsh = S.qsh; prm.qsn = S.qsn;
  prm.scale_log2 = scale * 1.4426950408889634f;
  if (sparse && !bitmap && attn_t_supported(S, W) && attn_t_enabled())
    return launch_attn_t(S, Q, K, V, kv_idx, kv_count, W, scale, O, lse, stream);
  if (sparse) {
    if (!bitmap && W > kMaxW) return fail(BSA_ERR_UNSUPPORTED, "sparse attn: kv_width %d > %d", W, kMaxW);
    prm.NT = S.NB;
    if (S.Bn == 64 && !bitmap && W <= kMaxWP && attn_persistent_enabled() &&
        static_cast<long long>(S.NB) * S.B * S.H < (1ll << 31)) {
      if (S.d == 64) return run_persistent<64>(S, K, V, prm, stream);
      if (S.d == 128) return run_persistent<128>(S, K, V, prm, stream);
      if (S.d == 256) return run_persistent<256>(S, K, V, prm, stream);
    }
#define BSA_SP(BMM, DD) \
  if (S.Bn == BMM && S.d == DD) return run<BMM, DD, true>(S, Q, K, V, prm, stream);
    BSA_SP(64, 64) BSA_SP(64, 128) BSA_SP(64, 256) BSA_SP(128, 64) BSA_SP(128, 128) BSA_SP(128, 256)
#undef BSA_SP
  } else {
    prm.NT = (S.N + 127) / 128;
    if (S.d == 64) return run<128, 64, false>(S, Q, K, V, prm, stream);
    if (S.d == 128) return run<128, 128, false>(S, Q, K, V, prm, stream);
    if (S.d == 256) return run<128, 256, false>(S, Q, K, V, prm, stream);
  }
  return fail(BSA_ERR_UNSUPPORTED, "attn: unsupported head_dim %d / block %d", S.d, S.Bn);
}

#ifdef BSA_TRACE
extern "C" int bsa_debug_trace(long long* host) {
  return static_cast<int>(cudaMemcpyFromSymbol(host, g_tr, sizeof(g_tr)));
}
#endif

}  // namespace bsa

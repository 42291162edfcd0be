// score_tc.cu -- tensor-core block scoring fused with tile-max, top-(2k) and sigma
// (Eq.1-4; A.2-A.6 L296-324; readings G1, G4-G8 in DESIGN.md).
//
// Work item = (tile t, KV head g, head set) where a head set is up to NH query heads of the GQA
// group.  The product is computed TRANSPOSED so that the tile max (Eq.3) is a per-thread loop:
//     S^T[block, (head, row)] = Pooled[block, :] . Qplanes[(head, row), :]
//   A (M = 128 pooled blocks, K-major)  streamed by TMA from the meta planes through a ring,
//   B (N = heads*BN query rows)         resident in shared memory,
//   D in TMEM, double buffered: lanes = blocks, columns = query rows.
// Quest (Eq.2):  sum_c max(q_c Kmax_c, q_c Kmin_c) = q+ . Kmax + q- . Kmin with q+ = max(q,0),
//   q- = min(q,0); all four operands are bf16-exact, K dimension 2d.
// K-mean (Eq.1): kmean (fp32) = hi + mid + lo exactly (three bf16 planes written by the pooling
//   kernel), K dimension 3d against the same Q chunk; products are exact, accumulation is fp32.
//
// The kernel is PERSISTENT (one CTA per SM, items strided over the grid, heaviest tiles first) and
// software-pipelined across items, because a one-item CTA spends ~10 us in phases that leave the
// tensor pipe idle (Q load 1.7k clk, q+/q- conversion 1.9k, ring warm-up, selection 6-8k) against
// 1-2 us of MMAs at 32K.  Roles (10 warps):
//   W0-3  q+/q- conversion of the item's Q tile, then the per-chunk epilogue: TMEM -> column max
//         per head -> order-preserving key -> score row in shared memory
//   W4    TMA producer: Q tile of the next item as soon as the MMAs of the current one are done,
//         pooled planes through the ring, continuously across items
//   W5    tcgen05.mma issue, accumulators ping-pong across chunks and items
//   W6-9  one warp per head: warp_select (select_common.cuh) of item i while W0-5 already work on
//         item i+1; the score rows are released as soon as the warp holds its keys in registers
//
// This header holds the kernel template; score_tc_quest.cu and score_tc_mean.cu instantiate it for the
// two backbones (two translation units so that the ~30 instantiations compile in parallel).
#pragma once
#include <cuda_bf16.h>

#include "bsa_internal.h"
#include "select_common.cuh"
#include "sm100_ptx.cuh"
#include "tmap.h"

namespace bsa {

namespace {

constexpr int kTcThreads = 320;
constexpr int kABlocks = 128;                 // pooled blocks per MMA (UMMA M)
constexpr int kAStageBytes = kABlocks * 128;  // one [128 blocks x 64 elem] swizzled tile
constexpr int kMaxStages = 6;
constexpr int kSelWarp0 = 6;                  // first selection warp

// NH = query heads of one GQA group scored per work item (UMMA N = NH * BN <= 256; B planes <= 128 KB).
// The host picks the largest NH <= NH_MAX whose shared-memory footprint fits: the score rows take
// NH * N_B * 4 bytes, so long sequences (N_B >= 4096, i.e. 256K tokens at block 64) run with fewer
// heads per item instead of being refused.
template <int D, int BN, bool QUEST>
struct TcShape {
  static constexpr int PLANES_B = QUEST ? 2 : 1;          // q+ | q-   or   q
  static constexpr int PLANES_A = QUEST ? 2 : 3;          // kmax | kmin   or   hi | mid | lo
  static constexpr int DC = D / 64;                        // 64-element K chunks per plane
  static constexpr int HEAD_B_BYTES = BN * D * 2 * PLANES_B;
  static constexpr int NH_N = 256 / BN;                    // UMMA N <= 256; also <= 4 selection warps
  static constexpr int NH_S = (128 * 1024) / HEAD_B_BYTES; // B planes <= 128 KB
  static constexpr int NH_MAX = NH_N < NH_S ? NH_N : NH_S;
};

template <int D, int BN, bool QUEST, int NH_>
struct TcCfg : TcShape<D, BN, QUEST> {
  using S = TcShape<D, BN, QUEST>;
  static constexpr int NH = NH_;
  static constexpr int NROWS = NH * BN;                    // rows of one B chunk tile
  static constexpr int B_CHUNK_BYTES = NROWS * 128;
  static constexpr int B_BYTES = B_CHUNK_BYTES * S::DC * S::PLANES_B;
  static constexpr int KCHUNKS = S::PLANES_A * S::DC;      // A chunks per block chunk
  static constexpr uint32_t TMEM_COLS = (2 * NROWS <= 32) ? 32 : (2 * NROWS <= 64) ? 64
                                        : (2 * NROWS <= 128) ? 128 : (2 * NROWS <= 256) ? 256 : 512;
  static_assert(NH >= 1 && NH <= 4 && NH <= S::NH_MAX, "one selection warp per head, four of them");
};

struct TcParams {
  int32_t* kv_idx;
  int32_t* kv_count;
  float* sigma;
  int B, H, Hkv, G, NB, k, W, router, sets, stages, nbpad, n_items, ncand;
  float inv_sqrt_d;
  // D.4 diagnostics (Eq.18), all [B,H,T] or nullptr (diag == 0)
  int diag;
  float *dg_g, *dg_G, *dg_r, *dg_d2, *dg_rough;
};

struct alignas(8) TcCtl {
  uint64_t q_full, b_ready, b_free, sc_full, sc_free;
  uint64_t a_full[kMaxStages], a_empty[kMaxStages];
  uint64_t acc_full[2], acc_empty[2];
  uint32_t tmem_base;
  uint32_t s3[4 * 4];   // per-warp scratch of warp_select
  float rough[4][4];    // [epilogue warp][head]: sum of squared row-to-row score differences (diag)
};

struct Item {
  int t, b, g, set, h0, nh, n_chunks;
};

// item w -> (tile, batch, KV head, head set); heaviest (largest t) tiles first
template <int NH>
__device__ __forceinline__ Item decode_item(const TcParams& p, int w) {
  Item it;
  const int per_tile = p.B * p.Hkv * p.sets;
  it.t = p.NB - 1 - w / per_tile;
  int rem = w % per_tile;
  it.b = rem / (p.Hkv * p.sets);
  rem %= p.Hkv * p.sets;
  it.g = rem / p.sets;
  it.set = rem % p.sets;
  it.h0 = it.g * p.G + it.set * NH;
  const int left = p.G - it.set * NH;
  it.nh = left < NH ? left : NH;
  it.n_chunks = (it.t + 1 + kABlocks - 1) / kABlocks;
  return it;
}

template <int D, int BN, bool QUEST, int NH, bool DIAG>
__global__ void __launch_bounds__(kTcThreads, 1)
score_tc_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmA,
                const TcParams p) {
  using C = TcCfg<D, BN, QUEST, NH>;
  extern __shared__ __align__(1024) uint8_t smem[];
  uint8_t* b_s = smem;                                   // [PLANES_B][DC][NROWS x 128 B]
  uint8_t* a_s = smem + C::B_BYTES;                      // ring of [128 x 128 B] stages
  uint32_t* sc = reinterpret_cast<uint32_t*>(a_s + p.stages * kAStageBytes);   // [NH][nbpad] okey(score)
  unsigned long long* cand = reinterpret_cast<unsigned long long*>(sc + C::NH * p.nbpad);
  // candidate / sorted-key arrays are sized by the budget (p.ncand >= 2k + 1 entries per head), the sorted
  // keys exist only in diagnostics mode: at N_B = 4096 these bytes decide whether four heads fit
  uint32_t* srt = reinterpret_cast<uint32_t*>(cand + C::NH * p.ncand);    // sorted keys (diag), per head
  TcCtl* ctl = reinterpret_cast<TcCtl*>(srt + (DIAG ? C::NH * p.ncand : 0));

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int w0 = static_cast<int>(blockIdx.x), wstep = static_cast<int>(gridDim.x);

  if ((smem_u32(smem) & 1023u) != 0) __trap();

  if (warp == 5 && lane == 0) {
    mbar_init(smem_u32(&ctl->q_full), 1);
    mbar_init(smem_u32(&ctl->b_ready), 4);
    mbar_init(smem_u32(&ctl->b_free), 1);
    mbar_init(smem_u32(&ctl->sc_full), 4);
    mbar_init(smem_u32(&ctl->sc_free), 4);
    for (int s = 0; s < p.stages; ++s) {
      mbar_init(smem_u32(&ctl->a_full[s]), 1);
      mbar_init(smem_u32(&ctl->a_empty[s]), 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&ctl->acc_full[i]), 1);
      mbar_init(smem_u32(&ctl->acc_empty[i]), 4);
    }
    fence_mbar_init();
  }
  if (warp == 4) {
    if (lane == 0) {
      tma_prefetch_desc(&tmQ);
      tma_prefetch_desc(&tmA);
    }
    __syncwarp();
    tmem_alloc<C::TMEM_COLS>(smem_u32(&ctl->tmem_base));
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = ctl->tmem_base;

  if (warp == 4) {
    // ---- TMA producer ------------------------------------------------------------------------
    if (lane == 0) {
      const int stages = p.stages;
      int li = 0, s = 0;
      uint32_t ph = 0;
      for (int w = w0; w < p.n_items; w += wstep, ++li) {
        const Item im = decode_item<C::NH>(p, w);
        if (li > 0) mbar_wait(smem_u32(&ctl->b_free), (li - 1) & 1);   // MMAs of the previous item done
        mbar_arrive_expect_tx(smem_u32(&ctl->q_full), C::DC * C::B_CHUNK_BYTES);
        for (int c64 = 0; c64 < C::DC; ++c64)
          tma_load_5d(smem_u32(b_s + c64 * C::B_CHUNK_BYTES), &tmQ, smem_u32(&ctl->q_full), 0,
                      im.t * BN, c64, im.h0, im.b);
        if (w + wstep < p.n_items) {   // warm the L2 with the Q tile of this CTA's next item
          const Item nx = decode_item<C::NH>(p, w + wstep);
          for (int c64 = 0; c64 < C::DC; ++c64)
            tma_prefetch_5d(&tmQ, 0, nx.t * BN, c64, nx.h0, nx.b);
        }
        for (int c = 0; c < im.n_chunks; ++c) {
#pragma unroll
          for (int kc = 0; kc < C::KCHUNKS; ++kc) {
            const int pa = kc / C::DC, c64 = kc % C::DC;
            const int mem_plane = QUEST ? (1 - pa) : pa;   // memory order: [kmin, kmax] / [hi, mid, lo]
            mbar_wait(smem_u32(&ctl->a_empty[s]), ph ^ 1u);
            mbar_arrive_expect_tx(smem_u32(&ctl->a_full[s]), kAStageBytes);
            tma_load_5d(smem_u32(a_s + s * kAStageBytes), &tmA, smem_u32(&ctl->a_full[s]), c64 * 64,
                        c * kABlocks, im.g, im.b, mem_plane);
            if (++s == stages) {
              s = 0;
              ph ^= 1u;
            }
          }
        }
      }
    }
  } else if (warp == 5) {
    // ---- MMA issuer --------------------------------------------------------------------------
    // One thread; it must stay cheap: an ncu source view of the first persistent version showed this
    // thread executing ~700 scalar instructions per 16-MMA chunk (runtime `ring % stages`, descriptor
    // rebuilds), i.e. longer than the MMAs it issues, with the tensor pipe 50 % idle.  The ring slot
    // and phase are tracked incrementally and the descriptors are a base plus a small constant.
    {   // the whole warp runs the loop (warp-uniform addresses and descriptors); one lane issues
      const bool leader = elect_one();
      const uint32_t b_a = smem_u32(b_s), a_a = smem_u32(a_s);
      const uint64_t adesc0 = umma_smem_desc(a_a, 16, 1024);
      const uint64_t bdesc0 = umma_smem_desc(b_a, 16, 1024);
      const int stages = p.stages;
      int li = 0, cg = 0, s = 0;
      uint32_t ph = 0;
      for (int w = w0; w < p.n_items; w += wstep, ++li) {
        const Item im = decode_item<C::NH>(p, w);
        const uint32_t idesc = umma_idesc_bf16(kABlocks, im.nh * BN, 0, 0);
        mbar_wait(smem_u32(&ctl->b_ready), li & 1);
        tc_fence_after();
        for (int c = 0; c < im.n_chunks; ++c, ++cg) {
          const int buf = cg & 1;
          if (cg >= 2) {
            mbar_wait(smem_u32(&ctl->acc_empty[buf]), ((cg >> 1) & 1) ^ 1);
            tc_fence_after();
          }
          const uint32_t tD = tmem + buf * C::NROWS;
#pragma unroll
          for (int kc = 0; kc < C::KCHUNKS; ++kc) {
            const int bchunk = QUEST ? kc : (kc % C::DC);
            mbar_wait(smem_u32(&ctl->a_full[s]), ph);
            tc_fence_after();
            const uint64_t ad = adesc0 + static_cast<uint64_t>((s * kAStageBytes) >> 4);
            const uint64_t bd = bdesc0 + static_cast<uint64_t>((bchunk * C::B_CHUNK_BYTES) >> 4);
#pragma unroll
            for (int ks = 0; ks < 4; ++ks)
              if (leader) umma_ss(tD, ad + 2 * ks, bd + 2 * ks, idesc, (kc > 0) || (ks > 0));   // +32 B per K step
            if (leader) tc_commit(smem_u32(&ctl->a_empty[s]));
            __syncwarp();
            if (++s == stages) {
              s = 0;
              ph ^= 1u;
            }
          }
          if (leader) tc_commit(smem_u32(&ctl->acc_full[buf]));
        }
        if (leader) tc_commit(smem_u32(&ctl->b_free));   // every MMA that reads this item's B planes has completed
      }
    }
  } else if (warp < 4) {
    // ---- conversion + epilogue (warps 0-3) ---------------------------------------------------
    const uint32_t lane_base = static_cast<uint32_t>(warp * 32) << 16;
    int li = 0, cg = 0;
    for (int w = w0; w < p.n_items; w += wstep, ++li) {
      const Item im = decode_item<C::NH>(p, w);
      mbar_wait(smem_u32(&ctl->q_full), li & 1);
      if (QUEST) {
        // q+ = max(q, 0) in place, q- = min(q, 0) into plane 1 (element-wise, swizzle preserved)
        constexpr int PLANE = C::DC * C::B_CHUNK_BYTES;
#pragma unroll 4
        for (int i = tid; i < PLANE / 16; i += 128) {
          uint4 v = *reinterpret_cast<uint4*>(b_s + i * 16);
          uint32_t wv[4] = {v.x, v.y, v.z, v.w}, pos[4], neg[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const uint32_t nm = ((wv[j] & 0x80008000u) >> 15) * 0xFFFFu;  // 0xFFFF per negative half
            neg[j] = wv[j] & nm;
            pos[j] = wv[j] & ~nm;
          }
          *reinterpret_cast<uint4*>(b_s + i * 16) = make_uint4(pos[0], pos[1], pos[2], pos[3]);
          *reinterpret_cast<uint4*>(b_s + PLANE + i * 16) = make_uint4(neg[0], neg[1], neg[2], neg[3]);
        }
        fence_proxy_async_smem();
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctl->b_ready));

      // the selection warps must hold the previous item's keys in registers before sc is rewritten
      // (and have read the previous item's rough[] partials, which they do before releasing the keys)
      if (li > 0) mbar_wait(smem_u32(&ctl->sc_free), (li - 1) & 1);
      double rough[4] = {0.0, 0.0, 0.0, 0.0};
      for (int c = 0; c < im.n_chunks; ++c, ++cg) {
        const int buf = cg & 1;
        mbar_wait(smem_u32(&ctl->acc_full[buf]), (cg >> 1) & 1);
        tc_fence_after();
        const int blk = c * kABlocks + warp * 32 + lane;
        const uint32_t tD = tmem + lane_base + buf * C::NROWS;
#pragma unroll(DIAG ? C::NH : 1)
        for (int j = 0; j < (DIAG ? C::NH : im.nh); ++j) {
          if (DIAG && j >= im.nh) break;
          float m0 = -INFINITY, m1 = -INFINITY, m2 = -INFINITY, m3 = -INFINITY;   // four independent chains
          float rs = 0.0f, prev = 0.0f;   // diag: sum of squared differences of adjacent rows' scores
#pragma unroll
          for (int c0 = 0; c0 < BN; c0 += 64) {
            uint32_t ra[32], rb[32];
            tmem_ld32(tD + j * BN + c0, ra);
            tmem_ld32(tD + j * BN + c0 + 32, rb);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; i += 4) {
              m0 = fmax3(m0, __uint_as_float(ra[i]), __uint_as_float(rb[i]));
              m1 = fmax3(m1, __uint_as_float(ra[i + 1]), __uint_as_float(rb[i + 1]));
              m2 = fmax3(m2, __uint_as_float(ra[i + 2]), __uint_as_float(rb[i + 2]));
              m3 = fmax3(m3, __uint_as_float(ra[i + 3]), __uint_as_float(rb[i + 3]));
            }
            if constexpr (DIAG) {   // rows c0 .. c0+63 are ra[0..31], rb[0..31]
              if (c0 > 0) { const float d0 = __uint_as_float(ra[0]) - prev; rs = fmaf(d0, d0, rs); }
#pragma unroll
              for (int i = 0; i < 31; ++i) {
                const float da = __uint_as_float(ra[i + 1]) - __uint_as_float(ra[i]);
                const float db = __uint_as_float(rb[i + 1]) - __uint_as_float(rb[i]);
                rs = fmaf(da, da, rs);
                rs = fmaf(db, db, rs);
              }
              const float dm = __uint_as_float(rb[0]) - __uint_as_float(ra[31]);
              rs = fmaf(dm, dm, rs);
              prev = __uint_as_float(rb[31]);
            }
          }
          const float mx = fmaxf(fmax3(m0, m1, m2), m3);
          if (blk <= im.t) sc[j * p.nbpad + blk] = okey(QUEST ? mx : mx * p.inv_sqrt_d);   // Eq.3 (G8)
          if constexpr (DIAG) rough[j] += (blk <= im.t) ? static_cast<double>(rs) : 0.0;
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctl->acc_empty[buf]));
      }
      if constexpr (DIAG) {   // fixed-order reduction: lanes by shuffle tree, warps summed 0..3 by the consumer
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          double v = rough[j];
#pragma unroll
          for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
          if (lane == 0) ctl->rough[warp][j] = static_cast<float>(v);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(smem_u32(&ctl->sc_full));   // release: the score rows are complete
    }
  } else if (warp >= kSelWarp0) {
    // ---- selection (warps 6-9, one per head) --------------------------------------------------
    const int sw = warp - kSelWarp0;
    int li = 0;
    for (int w = w0; w < p.n_items; w += wstep, ++li) {
      const Item im = decode_item<C::NH>(p, w);
      mbar_wait(smem_u32(&ctl->sc_full), li & 1);
      const uint32_t rel = smem_u32(&ctl->sc_free);
      if (sw < im.nh && sw < C::NH) {
        const int h = im.h0 + sw;
        const int64_t row = (static_cast<int64_t>(im.b) * p.H + h) * p.NB + im.t;
        float rough_sum = 0.0f;
        if constexpr (DIAG)   // read before the keys are released: the epilogue warps rewrite it for the next item
          rough_sum = ((ctl->rough[0][sw] + ctl->rough[1][sw]) + ctl->rough[2][sw]) + ctl->rough[3][sw];
        DiagCell cell;
        const float sig = warp_select(sc + sw * p.nbpad, im.t, p.k, p.NB, p.W, p.kv_idx + row * p.W,
                                      cand + sw * p.ncand, ctl->s3 + sw * 4, lane, rel,
                                      DIAG ? &cell : nullptr, srt + sw * p.ncand);
        if (lane == 0) {
          p.sigma[row] = sig;
          if (!p.router) p.kv_count[row] = (p.k < im.t + 1) ? p.k : im.t + 1;
          if constexpr (DIAG) {
            p.dg_g[row] = cell.g;
            p.dg_G[row] = cell.G;
            p.dg_r[row] = cell.r;
            p.dg_d2[row] = cell.d2;
            // Eq.1 carries 1/sqrt(d) (G8): the K-mean row scores are scaled after the fact
            p.dg_rough[row] = QUEST ? rough_sum : rough_sum * (p.inv_sqrt_d * p.inv_sqrt_d);
          }
        }
        __syncwarp();   // cand / s3 of this warp are reused by the next item
      } else {
        release_keys(rel, lane);
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 4) tmem_dealloc<C::TMEM_COLS>(tmem);
}

struct DiagPtrs {
  float *g, *G, *r, *d2, *rough;   // all nullptr: no diagnostics
};

inline int tc_ncand(int k) { return (2 * k + 1 + 7) & ~7; }   // <= kMaxCand for k <= 128

template <int D, int BN, bool QUEST, int NH>
size_t tc_fixed_smem(int nbpad, int k, bool diag) {
  using C = TcCfg<D, BN, QUEST, NH>;
  const size_t ncand = static_cast<size_t>(tc_ncand(k));
  return static_cast<size_t>(C::B_BYTES) + static_cast<size_t>(NH) * nbpad * 4 +
         static_cast<size_t>(NH) * ncand * 8 + (diag ? static_cast<size_t>(NH) * ncand * 4 : 0) + sizeof(TcCtl);
}
constexpr size_t kTcSmemBudget = 227 * 1024;

template <int D, int BN, bool QUEST, int NH>
bsa_status run_score_tc(const Dims& S, const void* Q, const char* meta, const MetaLayout& L, int k, int W,
                        int router, int32_t* kv_idx, int32_t* kv_count, float* sigma, const DiagPtrs& dg,
                        cudaStream_t stream) {
  using C = TcCfg<D, BN, QUEST, NH>;
  TcParams p;
  p.kv_idx = kv_idx; p.kv_count = kv_count; p.sigma = sigma;
  p.B = S.B; p.H = S.H; p.Hkv = S.Hkv; p.G = S.G; p.NB = S.NB; p.k = k; p.W = W; p.router = router;
  p.sets = (S.G + NH - 1) / NH;
  p.nbpad = (S.NB + 3) & ~3;
  p.inv_sqrt_d = static_cast<float>(1.0 / sqrt(static_cast<double>(S.d)));
  p.diag = dg.g != nullptr;
  p.dg_g = dg.g; p.dg_G = dg.G; p.dg_r = dg.r; p.dg_d2 = dg.d2; p.dg_rough = dg.rough;
  const long long n_items = static_cast<long long>(S.NB) * S.B * S.Hkv * p.sets;
  if (n_items > 0x7fffffffLL) return fail(BSA_ERR_UNSUPPORTED, "select: too many work items");
  p.n_items = static_cast<int>(n_items);
  p.ncand = tc_ncand(k);
  const size_t fixed = tc_fixed_smem<D, BN, QUEST, NH>(p.nbpad, k, p.diag != 0);
  int stages = static_cast<int>((kTcSmemBudget - fixed) / kAStageBytes);
  p.stages = stages > kMaxStages ? kMaxStages : stages;
#ifdef BSA_TC_STAGE_CAP
  if (p.stages > BSA_TC_STAGE_CAP) p.stages = BSA_TC_STAGE_CAP;
#endif
  const size_t smem = fixed + static_cast<size_t>(p.stages) * kAStageBytes;

  CUtensorMap tq, ta;
  if (!make_tmap_bhnd(&tq, Q, S.B, S.H, S.N, S.d, S.qsb, S.qsh, S.qsn, BN, 1, NH))
    return fail(BSA_ERR_CUDA, "select: cuTensorMapEncodeTiled(Q) failed");
  {
    const char* base = meta + (QUEST ? L.off_min : L.off_split);
    const cuuint64_t d2 = static_cast<cuuint64_t>(S.d) * 2;
    cuuint64_t dims[5] = {static_cast<cuuint64_t>(S.d), static_cast<cuuint64_t>(S.NB),
                          static_cast<cuuint64_t>(S.Hkv), static_cast<cuuint64_t>(S.B),
                          static_cast<cuuint64_t>(C::PLANES_A)};
    cuuint64_t strides[4] = {d2, d2 * S.NB, d2 * S.NB * S.Hkv, static_cast<cuuint64_t>(L.elems) * 2};
    cuuint32_t box[5] = {64, kABlocks, 1, 1, 1};
    if (!make_tmap_bf16(&ta, base, 5, dims, strides, box))
      return fail(BSA_ERR_CUDA, "select: cuTensorMapEncodeTiled(meta) failed");
  }
  auto kern = p.diag ? score_tc_kernel<D, BN, QUEST, NH, true> : score_tc_kernel<D, BN, QUEST, NH, false>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       static_cast<int>(smem));
  if (e != cudaSuccess) return fail(BSA_ERR_CUDA, "select: smem attribute: %s", cudaGetErrorString(e));
  const int sms = sm_count();
  const unsigned grid = static_cast<unsigned>(p.n_items < sms ? p.n_items : sms);   // one CTA per SM
  kern<<<grid, kTcThreads, smem, stream>>>(tq, ta, p);
  return check_launch("score_tc_kernel");
}

// Largest NH <= NH_MAX whose footprint leaves at least two A stages; 0 = even one head does not fit.
template <int D, int BN, bool QUEST, int NH>
bsa_status dispatch_nh(const Dims& S, const void* Q, const char* meta, const MetaLayout& L, int k, int W,
                       int router, int32_t* kv_idx, int32_t* kv_count, float* sigma, const DiagPtrs& dg,
                       cudaStream_t stream) {
  const int nbpad = (S.NB + 3) & ~3;
  // fewer heads per item than the GQA group has only cost A-plane re-reads; more never help
  const bool useful = (NH == 1) || (NH - 1 < S.G);
  const bool diag = dg.g != nullptr;
  if (useful && tc_fixed_smem<D, BN, QUEST, NH>(nbpad, k, diag) + 2 * kAStageBytes <= kTcSmemBudget)
    return run_score_tc<D, BN, QUEST, NH>(S, Q, meta, L, k, W, router, kv_idx, kv_count, sigma, dg, stream);
  if constexpr (NH > 1) {
    return dispatch_nh<D, BN, QUEST, NH - 1>(S, Q, meta, L, k, W, router, kv_idx, kv_count, sigma, dg, stream);
  } else {
    return fail(BSA_ERR_UNSUPPORTED,
                "select: %d blocks per sequence need %zu bytes of shared memory per head (limit %zu): "
                "at most %zu blocks fit for head_dim %d / block %d / this backbone",
                S.NB, tc_fixed_smem<D, BN, QUEST, 1>(nbpad, k, diag) + 2 * kAStageBytes, kTcSmemBudget,
                (kTcSmemBudget - tc_fixed_smem<D, BN, QUEST, 1>(0, k, diag) - 2 * kAStageBytes) / 4, S.d, S.Bn);
  }
}

template <bool QUEST>
bsa_status launch_score_tc_backbone(const Dims& S, const void* Q, const void* meta, int k, int W, int router,
                                    int32_t* kv_idx, int32_t* kv_count, float* sigma, const DiagPtrs& dg,
                                    cudaStream_t stream) {
  const MetaLayout L = meta_layout(S);
  const char* mp = static_cast<const char*>(meta);
#define BSA_TC(DD, BB)                                                                                \
  if (S.d == DD && S.Bn == BB)                                                                        \
    return dispatch_nh<DD, BB, QUEST, TcShape<DD, BB, QUEST>::NH_MAX>(S, Q, mp, L, k, W, router, kv_idx, \
                                                                     kv_count, sigma, dg, stream);
  BSA_TC(64, 64) BSA_TC(128, 64) BSA_TC(256, 64) BSA_TC(64, 128) BSA_TC(128, 128) BSA_TC(256, 128)
#undef BSA_TC
  return fail(BSA_ERR_UNSUPPORTED, "select: unsupported head_dim %d / block %d", S.d, S.Bn);
}

}  // namespace

}  // namespace bsa

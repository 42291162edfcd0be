// rowsel.cu -- bsa_select_rows_bitmap: per-ROW block selection scattered into a per-tile bitmap
// (section 4.5 item 1, L269: "A per-row scatter-into-bitmap kernel would close the rest of the
// gap without re-materialising the [B, H, M, N_B] keep tensor; not yet built").  Reading G18:
// every query row ranks the visible blocks by its own row score (Eq.1 / Eq.2, no tile max), blocks 0 and t
// forced (Eq.9), ties -> lower block index (G6), keeps its first min(k_row, t+1) blocks; the bitmap of
// tile t is the union over its rows.
//
// Work item = (tile t, head h), persistent CTAs (one per SM), heaviest tiles first.  The row scores are
// the same transposed tensor-core product as score_tc.cuh with one head per item:
//     S^T[block, row] = Pooled[block, :] . Qplanes[row, :]      (M = 128 blocks, N = BN rows)
// but instead of the column max the epilogue keeps every score: a SEGMENT of up to 512 blocks x BN rows
// of order-preserving keys in shared memory (128 KB).  After each segment every row merges the segment
// into its running top-(k_row - f) list (key, block) -- bisection on the key bits in registers, ties to
// the lower index, exactly warp_topk_compact's rule -- so sequences of any length run in bounded shared
// memory.  At the end the rows' lists are OR-ed into the tile's bitmap with shared-memory atomics.
// Roles (6 warps): W0-3 q+/q- conversion, epilogue and the per-row merges (rows split four ways),
// W4 TMA producer, W5 tcgen05.mma issue.
#include <cuda_bf16.h>

#include "bsa_internal.h"
#include "select_common.cuh"
#include "sm100_ptx.cuh"
#include "tmap.h"

namespace bsa {

namespace {

constexpr int kRsThreads = 192;
constexpr int kRsABlocks = 128;
constexpr int kRsAStage = kRsABlocks * 128;
constexpr int kRsMaxStages = 4;

template <int D, int BN, bool QUEST>
struct RsCfg {
  static constexpr int PLANES_B = QUEST ? 2 : 1;
  static constexpr int PLANES_A = QUEST ? 2 : 3;
  static constexpr int DC = D / 64;
  static constexpr int B_CHUNK_BYTES = BN * 128;
  static constexpr int B_BYTES = B_CHUNK_BYTES * DC * PLANES_B;
  static constexpr int KCHUNKS = PLANES_A * DC;
  static constexpr uint32_t TMEM_COLS = (2 * BN <= 128) ? 128 : 256;
  static constexpr int RPW = BN / 4;   // rows per selection warp
};

struct RsParams {
  uint32_t* bitmap;     // [B, H, T, nbw]
  int32_t* count;       // [B, H, T]
  int B, H, G, NB, k_row, kcap, seg, stages, n_items, nbw;
  float inv_sqrt_d;
};

struct alignas(8) RsCtl {
  uint64_t q_full, b_ready, b_free;
  uint64_t a_full[kRsMaxStages], a_empty[kRsMaxStages];
  uint64_t acc_full[2], acc_empty[2];
  uint32_t tmem_base;
  int32_t cnt;
  int16_t np[128];      // per row: entries in its running list
};

__device__ __forceinline__ void bar128() { asm volatile("bar.sync 1, 128;" ::: "memory"); }

// One warp merges a segment into the running lists of FOUR rows.  Per row: keys[i], i in [j_lo, j_hi), are
// the keys of blocks blk0 + i of this segment (candidates: free blocks only); list[0..np) = the row's current
// top entries (key, block), blocks ascending, all below blk0.  Afterwards list holds the top
// min(kprime, np + n_seg) of the union by (key desc, block asc), blocks ascending, and np4[] the new counts.
// The threshold is found by bisection on the key bits (ties to the lower block, warp_topk_compact's rule);
// the four rows' (compare, redux) chains are independent and overlap their latencies.
template <int KPL>
__device__ __noinline__ void row_merge4(const uint32_t* keys0, int seg, int j_lo, int j_hi, int blk0,
                                        uint2* list0, int kcap, int16_t* np4, int kprime, int lane) {
  const unsigned full = 0xffffffffu;
  constexpr int R = 4;
  uint32_t r[R][KPL], ck[R][2], cb[R][2];
  uint32_t hi[R], lo[R];
  int np[R];
  const int n_seg = j_hi > j_lo ? j_hi - j_lo : 0;
#pragma unroll
  for (int a = 0; a < R; ++a) {
    np[a] = np4[a];
    hi[a] = 0u;
    lo[a] = 0xffffffffu;
#pragma unroll
    for (int j = 0; j < KPL; ++j) {
      const int i = j * 32 + lane;
      const bool v = i >= j_lo && i < j_hi;
      r[a][j] = v ? keys0[a * seg + i] : 0u;
      hi[a] = max(hi[a], r[a][j]);
      lo[a] = v ? min(lo[a], r[a][j]) : lo[a];
    }
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const int i = j * 32 + lane;
      const bool v = i < np[a];
      const uint2 e = v ? list0[a * kcap + i] : make_uint2(0u, 0u);
      ck[a][j] = e.x;
      cb[a][j] = e.y;
      hi[a] = max(hi[a], ck[a][j]);
      lo[a] = v ? min(lo[a], ck[a][j]) : lo[a];
    }
  }
  __syncwarp();
  uint32_t vth[R], prefix[R];
  int r_eq[R], need[R], top[R];
  bool open[R];                          // bisection still running for this row
  int top_max = -1;
#pragma unroll
  for (int a = 0; a < R; ++a) {
    const int total = np[a] + n_seg;
    need[a] = kprime < total ? kprime : total;
    vth[a] = 0u;
    r_eq[a] = 0;
    open[a] = false;
    top[a] = -1;
    prefix[a] = 0u;
    if (need[a] > 0 && need[a] < total) {
      hi[a] = __reduce_max_sync(full, hi[a]);
      lo[a] = __reduce_min_sync(full, lo[a]);
      vth[a] = hi[a];
      r_eq[a] = need[a];
      const uint32_t diff = hi[a] ^ lo[a];
      if (diff != 0u) {
        top[a] = 31 - __clz(diff);
        prefix[a] = (top[a] == 31) ? 0u : (hi[a] & ~((2u << top[a]) - 1u));
        open[a] = true;
        top_max = top[a] > top_max ? top[a] : top_max;
      }
    }
  }
  bool exact[R] = {false, false, false, false};
  for (int bit = top_max; bit >= 0; --bit) {
    int cnt[R];
#pragma unroll
    for (int a = 0; a < R; ++a) {
      const uint32_t c = prefix[a] | (1u << bit);
      int n = (ck[a][0] >= c ? 1 : 0) + (ck[a][1] >= c ? 1 : 0);
#pragma unroll
      for (int j = 0; j < KPL; ++j) n += (r[a][j] >= c) ? 1 : 0;
      cnt[a] = n;
    }
#pragma unroll
    for (int a = 0; a < R; ++a) cnt[a] = __reduce_add_sync(full, cnt[a]);
    bool any_open = false;
#pragma unroll
    for (int a = 0; a < R; ++a) {
      if (open[a] && bit <= top[a]) {
        if (cnt[a] >= need[a]) prefix[a] |= (1u << bit);
        if (cnt[a] == need[a]) { exact[a] = true; open[a] = false; }
      }
      any_open = any_open || open[a];
    }
    if (!any_open) break;
  }
#pragma unroll
  for (int a = 0; a < R; ++a) {
    if (top[a] >= 0) {
      if (exact[a]) {
        vth[a] = prefix[a] - 1u;
        r_eq[a] = 0;
      } else {
        vth[a] = prefix[a];
        int cgt = (ck[a][0] > vth[a] ? 1 : 0) + (ck[a][1] > vth[a] ? 1 : 0);
#pragma unroll
        for (int j = 0; j < KPL; ++j) cgt += (r[a][j] > vth[a]) ? 1 : 0;
        cgt = __reduce_add_sync(full, cgt);
        r_eq[a] = need[a] - cgt;
      }
    }
  }
  const unsigned lt = (1u << lane) - 1u;
#pragma unroll
  for (int a = 0; a < R; ++a) {
    if (need[a] <= 0) {
      if (lane == 0) np4[a] = 0;
      continue;
    }
    uint2* list = list0 + a * kcap;
    int base = 0, eq_seen = 0;
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      if (j * 32 < np[a]) {
        const bool valid = j * 32 + lane < np[a];
        const bool gt = valid && ck[a][j] > vth[a];
        const bool eq = valid && ck[a][j] == vth[a] && r_eq[a] > 0;
        const unsigned be = __ballot_sync(full, eq);
        const bool take = gt || (eq && (eq_seen + __popc(be & lt) < r_eq[a]));
        const unsigned bsel = __ballot_sync(full, take);
        if (take) list[base + __popc(bsel & lt)] = make_uint2(ck[a][j], cb[a][j]);
        base += __popc(bsel);
        eq_seen += __popc(be);
      }
    }
#pragma unroll
    for (int j = 0; j < KPL; ++j) {
      if (j * 32 < j_hi) {
        const int i = j * 32 + lane;
        const bool valid = i >= j_lo && i < j_hi;
        const bool gt = valid && r[a][j] > vth[a];
        const bool eq = valid && r[a][j] == vth[a] && r_eq[a] > 0;
        const unsigned be = __ballot_sync(full, eq);
        const bool take = gt || (eq && (eq_seen + __popc(be & lt) < r_eq[a]));
        const unsigned bsel = __ballot_sync(full, take);
        if (take) list[base + __popc(bsel & lt)] = make_uint2(r[a][j], static_cast<uint32_t>(blk0 + i));
        base += __popc(bsel);
        eq_seen += __popc(be);
      }
    }
    if (lane == 0) np4[a] = static_cast<int16_t>(need[a]);
  }
  __syncwarp();
}

template <int D, int BN, bool QUEST>
__global__ void __launch_bounds__(kRsThreads, 1)
rowsel_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmA,
              const RsParams p) {
  using C = RsCfg<D, BN, QUEST>;
  extern __shared__ __align__(1024) uint8_t smem[];
  uint8_t* b_s = smem;                                                  // [PLANES_B][DC][BN x 128 B]
  uint8_t* a_s = smem + C::B_BYTES;                                     // ring of [128 x 128 B] stages
  uint32_t* sc = reinterpret_cast<uint32_t*>(a_s + p.stages * kRsAStage);   // [BN rows][seg] keys
  uint2* lists = reinterpret_cast<uint2*>(sc + BN * p.seg);             // [BN rows][kcap] (key, block)
  uint32_t* bm = reinterpret_cast<uint32_t*>(lists + BN * p.kcap);      // [nbw] bitmap of this item
  RsCtl* ctl = reinterpret_cast<RsCtl*>(bm + ((p.nbw + 1) & ~1));

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int w0 = static_cast<int>(blockIdx.x), wstep = static_cast<int>(gridDim.x);
  if ((smem_u32(smem) & 1023u) != 0) __trap();

  if (warp == 5 && lane == 0) {
    mbar_init(smem_u32(&ctl->q_full), 1);
    mbar_init(smem_u32(&ctl->b_ready), 4);
    mbar_init(smem_u32(&ctl->b_free), 1);
    for (int s = 0; s < p.stages; ++s) {
      mbar_init(smem_u32(&ctl->a_full[s]), 1);
      mbar_init(smem_u32(&ctl->a_empty[s]), 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&ctl->acc_full[i]), 1);
      mbar_init(smem_u32(&ctl->acc_empty[i]), 4);
    }
    ctl->cnt = 0;
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
  const int per_tile = p.B * p.H;
  const int cps = p.seg / kRsABlocks;                   // chunks per segment

  if (warp == 4) {
    // ---- TMA producer ------------------------------------------------------------------------
    if (lane == 0) {
      int li = 0, s = 0;
      uint32_t ph = 0;
      for (int w = w0; w < p.n_items; w += wstep, ++li) {
        const int t = p.NB - 1 - w / per_tile, rem = w % per_tile, b = rem / p.H, h = rem % p.H;
        const int g = h / p.G, n_chunks = (t + 1 + kRsABlocks - 1) / kRsABlocks;
        if (li > 0) mbar_wait(smem_u32(&ctl->b_free), (li - 1) & 1);
        mbar_arrive_expect_tx(smem_u32(&ctl->q_full), C::DC * C::B_CHUNK_BYTES);
        for (int c64 = 0; c64 < C::DC; ++c64)
          tma_load_5d(smem_u32(b_s + c64 * C::B_CHUNK_BYTES), &tmQ, smem_u32(&ctl->q_full), 0, t * BN, c64, h, b);
        for (int c = 0; c < n_chunks; ++c) {
#pragma unroll
          for (int kc = 0; kc < C::KCHUNKS; ++kc) {
            const int pa = kc / C::DC, c64 = kc % C::DC;
            const int mem_plane = QUEST ? (1 - pa) : pa;
            mbar_wait(smem_u32(&ctl->a_empty[s]), ph ^ 1u);
            mbar_arrive_expect_tx(smem_u32(&ctl->a_full[s]), kRsAStage);
            tma_load_5d(smem_u32(a_s + s * kRsAStage), &tmA, smem_u32(&ctl->a_full[s]), c64 * 64,
                        c * kRsABlocks, g, b, mem_plane);
            if (++s == p.stages) { s = 0; ph ^= 1u; }
          }
        }
      }
    }
  } else if (warp == 5) {
    // ---- MMA issuer (warp-uniform loop, one elected lane issues) ------------------------------
    const bool leader = elect_one();
    const uint64_t adesc0 = umma_smem_desc(smem_u32(a_s), 16, 1024);
    const uint64_t bdesc0 = umma_smem_desc(smem_u32(b_s), 16, 1024);
    constexpr uint32_t idesc = umma_idesc_bf16(kRsABlocks, BN, 0, 0);
    int li = 0, cg = 0, s = 0;
    uint32_t ph = 0;
    for (int w = w0; w < p.n_items; w += wstep, ++li) {
      const int t = p.NB - 1 - w / per_tile, n_chunks = (t + 1 + kRsABlocks - 1) / kRsABlocks;
      mbar_wait(smem_u32(&ctl->b_ready), li & 1);
      tc_fence_after();
      for (int c = 0; c < n_chunks; ++c, ++cg) {
        const int buf = cg & 1;
        if (cg >= 2) {
          mbar_wait(smem_u32(&ctl->acc_empty[buf]), ((cg >> 1) & 1) ^ 1);
          tc_fence_after();
        }
        const uint32_t tD = tmem + buf * BN;
#pragma unroll
        for (int kc = 0; kc < C::KCHUNKS; ++kc) {
          const int bchunk = QUEST ? kc : (kc % C::DC);
          mbar_wait(smem_u32(&ctl->a_full[s]), ph);
          tc_fence_after();
          const uint64_t ad = adesc0 + static_cast<uint64_t>((s * kRsAStage) >> 4);
          const uint64_t bd = bdesc0 + static_cast<uint64_t>((bchunk * C::B_CHUNK_BYTES) >> 4);
#pragma unroll
          for (int ks = 0; ks < 4; ++ks)
            if (leader) umma_ss(tD, ad + 2 * ks, bd + 2 * ks, idesc, (kc > 0) || (ks > 0));
          if (leader) tc_commit(smem_u32(&ctl->a_empty[s]));
          __syncwarp();
          if (++s == p.stages) { s = 0; ph ^= 1u; }
        }
        if (leader) tc_commit(smem_u32(&ctl->acc_full[buf]));
      }
      if (leader) tc_commit(smem_u32(&ctl->b_free));
    }
  } else {
    // ---- conversion, epilogue and per-row merges (warps 0-3) -----------------------------------
    const uint32_t lane_base = static_cast<uint32_t>(warp * 32) << 16;
    int li = 0, cg = 0;
    for (int w = w0; w < p.n_items; w += wstep, ++li) {
      const int t = p.NB - 1 - w / per_tile, rem = w % per_tile, b = rem / p.H, h = rem % p.H;
      const int n_chunks = (t + 1 + kRsABlocks - 1) / kRsABlocks;
      const int f = (t == 0) ? 1 : 2, kprime = p.k_row - f;
      mbar_wait(smem_u32(&ctl->q_full), li & 1);
      if (QUEST) {
        constexpr int PLANE = C::DC * C::B_CHUNK_BYTES;
#pragma unroll 4
        for (int i = tid; i < PLANE / 16; i += 128) {
          uint4 v = *reinterpret_cast<uint4*>(b_s + i * 16);
          uint32_t wv[4] = {v.x, v.y, v.z, v.w}, pos[4], neg[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const uint32_t nm = ((wv[j] & 0x80008000u) >> 15) * 0xFFFFu;
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
      for (int i = tid; i < p.nbw; i += 128) bm[i] = 0u;
      int16_t* np = ctl->np + warp * C::RPW;          // entries in the lists of this warp's rows
      for (int r = lane; r < C::RPW; r += 32) np[r] = 0;
      __syncwarp();

      for (int c = 0; c < n_chunks; ++c, ++cg) {
        const int buf = cg & 1;
        mbar_wait(smem_u32(&ctl->acc_full[buf]), (cg >> 1) & 1);
        tc_fence_after();
        const int blk = c * kRsABlocks + warp * 32 + lane;
        const bool cand = blk >= 1 && blk < t;        // free blocks 1 .. t-1
        const int col = (c % cps) * kRsABlocks + warp * 32 + lane;
        const uint32_t tD = tmem + lane_base + buf * BN;
#pragma unroll
        for (int c0 = 0; c0 < BN; c0 += 32) {
          uint32_t x[32];
          tmem_ld32(tD + c0, x);
          tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            const float s = __uint_as_float(x[i]);
            sc[(c0 + i) * p.seg + col] = cand ? okey(QUEST ? s : s * p.inv_sqrt_d) : 0u;
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&ctl->acc_empty[buf]));
        if ((c % cps) == cps - 1 || c == n_chunks - 1) {
          // a segment is complete: blocks [blk0, blk0 + seg), candidates 1 .. t-1
          const int seg_i = c / cps, blk0 = seg_i * p.seg;
          int j_lo = 1 - blk0, j_hi = t - blk0;
          j_lo = j_lo < 0 ? 0 : j_lo;
          j_hi = j_hi > p.seg ? p.seg : j_hi;
          bar128();
          if (kprime > 0) {
            for (int r = 0; r < C::RPW; r += 4) {       // four rows per call: independent bisection chains
              const int row = warp * C::RPW + r;
              const uint32_t* keys = sc + row * p.seg;
              uint2* list = lists + row * p.kcap;
              if (p.seg == 512) row_merge4<16>(keys, p.seg, j_lo, j_hi, blk0, list, p.kcap, np + r, kprime, lane);
              else if (p.seg == 256) row_merge4<8>(keys, p.seg, j_lo, j_hi, blk0, list, p.kcap, np + r, kprime, lane);
              else row_merge4<4>(keys, p.seg, j_lo, j_hi, blk0, list, p.kcap, np + r, kprime, lane);
            }
          }
          bar128();
        }
      }
      // scatter the rows' lists into the tile's bitmap (Eq.9: sink and self always)
      for (int r = 0; r < C::RPW; ++r) {
        const uint2* list = lists + (warp * C::RPW + r) * p.kcap;
        const int n = np[r];
        for (int i = lane; i < n; i += 32) atomicOr(&bm[list[i].y >> 5], 1u << (list[i].y & 31u));
      }
      if (tid == 0) {
        atomicOr(&bm[0], 1u);
        atomicOr(&bm[t >> 5], 1u << (t & 31));
      }
      bar128();
      const int64_t row = (static_cast<int64_t>(b) * p.H + h) * p.NB + t;
      int pc = 0;
      for (int i = tid; i < p.nbw; i += 128) {
        const uint32_t wv = bm[i];
        p.bitmap[row * p.nbw + i] = wv;
        pc += __popc(wv);
      }
      pc = __reduce_add_sync(0xffffffffu, pc);
      if (lane == 0) atomicAdd(&ctl->cnt, pc);
      bar128();
      if (tid == 0) {
        p.count[row] = ctl->cnt;
        ctl->cnt = 0;
      }
      bar128();   // bm and cnt are reused by the next item
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 4) tmem_dealloc<C::TMEM_COLS>(tmem);
}

template <int D, int BN, bool QUEST>
bsa_status run_rowsel(const Dims& S, const void* Q, const char* meta, const MetaLayout& L, int k_row,
                      uint32_t* bitmap, int32_t* count, cudaStream_t stream) {
  using C = RsCfg<D, BN, QUEST>;
  RsParams p;
  p.bitmap = bitmap; p.count = count;
  p.B = S.B; p.H = S.H; p.G = S.G; p.NB = S.NB; p.k_row = k_row; p.kcap = k_row;
  p.nbw = (S.NB + 31) / 32;
  p.inv_sqrt_d = static_cast<float>(1.0 / sqrt(static_cast<double>(S.d)));
  const long long n_items = static_cast<long long>(S.NB) * S.B * S.H;
  if (n_items > 0x7fffffffLL) return fail(BSA_ERR_UNSUPPORTED, "rows_bitmap: too many work items");
  p.n_items = static_cast<int>(n_items);
  const size_t budget = 227 * 1024;
  size_t fixed = 0;
  p.seg = 0;
  for (int seg = 512; seg >= 128; seg >>= 1) {
    fixed = static_cast<size_t>(C::B_BYTES) + static_cast<size_t>(BN) * seg * 4 +
            static_cast<size_t>(BN) * p.kcap * 8 + static_cast<size_t>((p.nbw + 1) & ~1) * 4 + sizeof(RsCtl);
    if (fixed + (seg > 128 ? 2 : 1) * kRsAStage <= budget) { p.seg = seg; break; }   // last resort: one stage
  }
  if (p.seg == 0)
    return fail(BSA_ERR_UNSUPPORTED, "rows_bitmap: head_dim %d / block %d / k_row %d need %zu bytes of shared "
                "memory (limit %zu)", S.d, S.Bn, k_row, fixed + kRsAStage, budget);
  int stages = static_cast<int>((budget - fixed) / kRsAStage);
  p.stages = stages > kRsMaxStages ? kRsMaxStages : stages;
  const size_t smem = fixed + static_cast<size_t>(p.stages) * kRsAStage;

  CUtensorMap tq, ta;
  if (!make_tmap_bhnd(&tq, Q, S.B, S.H, S.N, S.d, S.qsb, S.qsh, S.qsn, BN, 1, 1))
    return fail(BSA_ERR_CUDA, "rows_bitmap: cuTensorMapEncodeTiled(Q) failed");
  {
    const char* base = meta + (QUEST ? L.off_min : L.off_split);
    const cuuint64_t d2 = static_cast<cuuint64_t>(S.d) * 2;
    cuuint64_t dims[5] = {static_cast<cuuint64_t>(S.d), static_cast<cuuint64_t>(S.NB),
                          static_cast<cuuint64_t>(S.Hkv), static_cast<cuuint64_t>(S.B),
                          static_cast<cuuint64_t>(C::PLANES_A)};
    cuuint64_t strides[4] = {d2, d2 * S.NB, d2 * S.NB * S.Hkv, static_cast<cuuint64_t>(L.elems) * 2};
    cuuint32_t box[5] = {64, kRsABlocks, 1, 1, 1};
    if (!make_tmap_bf16(&ta, base, 5, dims, strides, box))
      return fail(BSA_ERR_CUDA, "rows_bitmap: cuTensorMapEncodeTiled(meta) failed");
  }
  auto kern = rowsel_kernel<D, BN, QUEST>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       static_cast<int>(smem));
  if (e != cudaSuccess) return fail(BSA_ERR_CUDA, "rows_bitmap: smem attribute: %s", cudaGetErrorString(e));
  const int sms = sm_count();
  const unsigned grid = static_cast<unsigned>(p.n_items < sms ? p.n_items : sms);
  kern<<<grid, kRsThreads, smem, stream>>>(tq, ta, p);
  return check_launch("rowsel_kernel");
}

}  // namespace

bsa_status launch_rowsel(const Dims& S, const void* Q, const void* meta, bool quest, int k_row,
                         uint32_t* bitmap, int32_t* count, cudaStream_t stream) {
  const MetaLayout L = meta_layout(S);
  const char* mp = static_cast<const char*>(meta);
#define BSA_RS(DD, BB)                                                                           \
  if (S.d == DD && S.Bn == BB)                                                                   \
    return quest ? run_rowsel<DD, BB, true>(S, Q, mp, L, k_row, bitmap, count, stream)           \
                 : run_rowsel<DD, BB, false>(S, Q, mp, L, k_row, bitmap, count, stream);
  BSA_RS(64, 64) BSA_RS(128, 64) BSA_RS(256, 64) BSA_RS(64, 128) BSA_RS(128, 128) BSA_RS(256, 128)
#undef BSA_RS
  return fail(BSA_ERR_UNSUPPORTED, "rows_bitmap: unsupported head_dim %d / block %d", S.d, S.Bn);
}

}  // namespace bsa

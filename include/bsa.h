/*
 * bsa.h -- C ABI of libbsa: uncertainty-gated block-sparse prefill attention for NVIDIA B200 (sm_100a).
 *
 * The calls follow the problem statement of arxiv/paper_2607_07724 (citations: PAPER.md line + eq.):
 *   bsa_build_block_meta : per-KV-block key pooling          (Eq.1/Eq.6 L74,L293; Eq.2)
 *   bsa_select           : per-(Q-tile, head) block scoring, causal top-k with forced sink/self,
 *                          normalised cutoff margin sigma, head mean, per-layer q-quantile trigger,
 *                          shape-uniform padded kv_idx       (Eq.3-5; A.2-A.9 L296-340)
 *   bsa_sparse_attn_fwd  : exact online-softmax attention over the selected K/V blocks
 *                                                            (L43-47, L131, A.10 L342)
 *   bsa_dense_attn_fwd   : dense causal attention, the "x dense" denominator (L45, L156)
 *
 * Conventions
 *   - Every pointer named Q/K/V/O/meta/kv_idx/kv_count/sigma/sigma_bar/trigger/tau/lse/workspace is a
 *     DEVICE pointer owned by the caller; the library allocates no device memory and keeps no state
 *     between calls.  Two exceptions, both small static device arrays: the scratch of bsa_select_static (see
 *     there) and the work counters of the persistent sparse attention kernel -- a launch takes one of 1024
 *     counter slots and returns it to zero itself; launches that overlap on the GPU use different slots unless
 *     more than 1024 of them are in flight at once.
 *     `shape` is a HOST pointer.  `stream` is a cudaStream_t passed as void*.
 *   - Every call only enqueues work on `stream`; it never synchronises and never touches the
 *     default stream.
 *   - Argument checks run on the host before any launch: BSA_ERR_INVALID_ARG, BSA_ERR_UNSUPPORTED and
 *     BSA_ERR_WORKSPACE_TOO_SMALL mean nothing was enqueued.  BSA_ERR_CUDA reports a failed CUDA call;
 *     when it comes from a kernel launch of a multi-kernel call (bsa_select), the kernels launched
 *     before it stay enqueued and the outputs are partially written.
 *     bsa_last_error() returns a thread-local description of the last failure.
 *   - Tensors are bf16 with the head dimension contiguous; strides are in elements.  Q and O share
 *     strides; K and V share strides.  Pointers and row strides must be 16-byte aligned.
 *   - BLOCK_M == BLOCK_N == shape.block (reading G10).  N_B = Q_t = seqlen / block.
 *   - GQA (reading G7): query head h uses KV head h / (n_q_heads / n_kv_heads).
 *   - Inputs are assumed finite.
 */
#ifndef BSA_H_
#define BSA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  BSA_OK = 0,
  BSA_ERR_INVALID_ARG = 1,        /* NULL pointer, seqlen % block, heads % kv heads, k_budget < 3,
                                     q_frac outside [0,1], misaligned pointer or stride */
  BSA_ERR_UNSUPPORTED = 2,        /* block not in {64,128}, head_dim not in {64,128,256}, not sm_100 */
  BSA_ERR_WORKSPACE_TOO_SMALL = 3,
  BSA_ERR_CUDA = 4                /* a CUDA runtime / driver call failed (see bsa_last_error) */
} bsa_status;

typedef enum {
  BSA_POLICY_TOPK = 0,            /* K-mean backbone (Eq.1), no expansion      (L157) */
  BSA_POLICY_ROUTER = 1,          /* K-mean backbone, sigma router              (L159) */
  BSA_POLICY_QUEST = 2,           /* K-min/K-max backbone (Eq.2), no expansion  (L158) */
  BSA_POLICY_ROUTER_QUEST = 3     /* K-min/K-max backbone, sigma router         (L160) */
} bsa_policy;

enum { BSA_META_MEAN = 1, BSA_META_MINMAX = 2 }; /* bit mask for `kinds` */
enum { BSA_META_SPLIT = 4 };                      /* bsa_block_meta_offset only: the bf16 split planes */
#define BSA_RHO 2                                 /* expansion factor rho (L129) */

typedef struct {
  int32_t batch, seqlen, n_q_heads, n_kv_heads, head_dim, block;
  int64_t q_stride_b, q_stride_h, q_stride_n;     /* Q and O, in elements */
  int64_t kv_stride_b, kv_stride_h, kv_stride_n;  /* K and V, in elements */
} bsa_shape;

/*
 * Block metadata buffer ("meta"), documented so tests can read and write it:
 *   offset 0                      : kmean fp32 [B, Hkv, N_B, d]   (Eq.1: (1/BLOCK_N) sum_j k_j)
 *   offset bsa_block_meta_offset(shape, BSA_META_MINMAX)
 *                                 : kmin  bf16 [B, Hkv, N_B, d]   (Eq.2: element-wise min)
 *   directly after kmin           : kmax  bf16 [B, Hkv, N_B, d]   (Eq.2: element-wise max)
 *   offset bsa_block_meta_offset(shape, BSA_META_SPLIT)
 *                                 : three bf16 planes hi, mid, lo, each [B, Hkv, N_B, d], with
 *                                   hi = bf16_rn(kmean), mid = bf16_rn(kmean - hi),
 *                                   lo = bf16_rn(kmean - hi - mid), so hi + mid + lo == kmean exactly.
 *                                   Written together with kmean (BSA_META_MEAN).  THE K-MEAN POLICIES OF
 *                                   bsa_select READ THESE PLANES (tensor-core operands), not the fp32
 *                                   kmean plane: a caller that overwrites kmean must rewrite the split.
 * The planes have fixed offsets regardless of `kinds`; planes not requested are left untouched.
 * bsa_block_meta_bytes returns the size to allocate (0 on invalid shape).
 */
size_t bsa_block_meta_bytes(const bsa_shape* shape, int kinds);
size_t bsa_block_meta_offset(const bsa_shape* shape, int kind /* BSA_META_MEAN | _MINMAX | _SPLIT */);

/* Pools K once (one pass, 128-bit loads) into `meta`.  kinds: BSA_META_MEAN | BSA_META_MINMAX. */
bsa_status bsa_build_block_meta(const bsa_shape* shape, const void* K, int kinds, void* meta,
                                void* stream);

/* Width W of a kv_idx row: k_budget (TOPK, QUEST) or BSA_RHO * k_budget (router policies). */
int32_t bsa_kv_width(bsa_policy policy, int32_t k_budget);

size_t bsa_select_workspace_bytes(const bsa_shape* shape, bsa_policy policy, int32_t k_budget);

/*
 * Selection.  For every Q-tile t (rows [t*block, (t+1)*block)) and query head h:
 *   tile_score[b] = max_{r in tile} s[r,h,b] for visible blocks b <= t            (Eq.3, reading G4)
 *     s = (q . kmean_b) / sqrt(d)  (TOPK, ROUTER)   |   s = sum_c max(q_c kmax_c, q_c kmin_c) (QUEST*)
 *   blocks 0 and t are forced on top (Eq.9); the rest sorted by score descending, ties -> lower
 *   block index first (reading G6).
 *   sigma[t,h] (Eq.4 / Eq.11, readings G1, G5):
 *       t+1 <= k_budget : 1
 *       else (s~[k-1] - s~[k]) / (s~[f] - s~[k]), f = number of forced blocks; 0 when the
 *       denominator is 0 (L324)
 *   sigma_bar[t] = mean_h sigma[t,h] (Eq.12, fp32 sum in ascending h, then / H)
 *   router policies: m = ceil(q_frac*Q_t - 1e-9); tau = m-th smallest sigma_bar (order statistic,
 *       readings G3, G15); trigger[t] = sigma_bar[t] <= tau; m == 0 -> no trigger, tau = -1.
 *       other policies: trigger = 0, tau = -1; q_frac is ignored.
 *   kv_count[t,h] = min(trigger ? 2k : k, t+1); kv_idx[t,h,0..count) = sorted prefix,
 *       remaining slots = N_B (sentinel)                                          (Eq.14)
 * Outputs: kv_idx [B,Hq,Q_t,W] int32, kv_count [B,Hq,Q_t] int32, sigma [B,Hq,Q_t] fp32 (required);
 *          sigma_bar [B,Q_t] fp32, trigger [B,Q_t] u8, tau [B] fp32 (each may be NULL).
 * `meta` must hold the planes the policy needs (MEAN for TOPK/ROUTER, MINMAX for QUEST policies).
 * Limits: 3 <= k_budget <= 128; N_B <= 8192 and N_B * 4 bytes of score row per head must fit the SM's
 * shared memory beside the query planes (the error text states the largest N_B that fits; block 64 /
 * head_dim 128 reaches N_B = 8192 = 512K tokens with both backbones).
 * sigma_bar / trigger may be NULL only if `workspace` (bsa_select_workspace_bytes, 256-byte aligned
 * use) is given: they are then kept there.
 */
bsa_status bsa_select(const bsa_shape* shape, const void* Q, const void* meta, bsa_policy policy,
                      int32_t k_budget, double q_frac, int32_t* kv_idx, int32_t* kv_count,
                      float* sigma, float* sigma_bar, uint8_t* trigger, float* tau, void* workspace,
                      size_t workspace_bytes, void* stream);

/*
 * bsa_select for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): same selection, same kernels and bit-identical kv_idx / kv_count /
 * sigma / tau as bsa_select, but the per-tile scratch (sigma_bar [B,Q_t] fp32 and trigger [B,Q_t] u8, Eq.12 /
 * Eq.5) lives in a static __device__ array inside the library instead of caller memory.  The call allocates
 * nothing (no cudaMalloc / cudaFree, no allocating library routine) and takes no workspace.
 *   Limit : batch * Q_t <= BSA_STATIC_MAX_TILES; beyond it BSA_ERR_UNSUPPORTED, nothing enqueued.  The other
 *           limits and errors are those of bsa_select.
 *   Cost  : every GPU that loads libbsa holds the array (82 176 bytes) until the process exits.
 *   State : all calls on a device share the one array and it keeps the last call's sigma_bar / trigger; a call
 *           needs none of it zeroed (it overwrites what it reads).  Two bsa_select_static calls that may
 *           overlap on the GPU (different streams, or graphs replayed concurrently) RACE on it: order them.
 *   Set-up: the first call on a device resolves the array's device address (cudaGetSymbolAddress, once per
 *           device, cached); make that first call outside stream capture.
 * sigma_bar and trigger are not returned; callers that want them use bsa_select.
 */
#define BSA_STATIC_MAX_TILES 16384
bsa_status bsa_select_static(const bsa_shape* shape, const void* Q, const void* meta, bsa_policy policy,
                             int32_t k_budget, double q_frac, int32_t* kv_idx, int32_t* kv_count,
                             float* sigma, float* tau, void* stream);

/*
 * D.4 diagnostics (App. D.4; Eq.18; (A1)/(A2) L431-432), computed
 * from the tile scores while they are on chip.  bsa_select_diag = bsa_select with the same arguments and
 * results, plus, per cell (tile t, head h) with at least rho*k + 1 visible blocks (L493; NaN elsewhere),
 * with s~ the sorted list of Eq.10 (forced blocks on top, f of them):
 *   g  [B,Hq,Q_t] = s~[k-1] - s~[k]        cutoff gap
 *   G  [B,Hq,Q_t] = s~[k-1] - s~[rho k]    expansion gap
 *   r  [B,Hq,Q_t] = s~[f]   - s~[k]        spread (so sigma = g / r, reading G1)
 *   d2 [B,Hq,Q_t] = min over ranks j in [f, rho k), j != k-1, of s~[j] - s~[j+1]   (secondary spacing, A1)
 * and for EVERY cell
 *   rough [B,Hq,Q_t] = sum over visible blocks b and adjacent rows i, i+1 of tile t of
 *                      (s[i+1,h,b] - s[i,h,b])^2      (step 3 of the recipe: E = 2 tau^2)
 * and per sequence summary [B, BSA_DIAG_SUMMARY_LEN] fp32 (index: meaning), population = the valid cells:
 *   0 n | 1 r_bar | 2 CV(r) = sqrt(Var r)/r_bar | 3 sigma_(q) = tau of the router (NaN otherwise) |
 *   4 gamma_q = sigma_(q) r_bar | 5 band mass m_q(beta): fraction with g in gamma_q[1-beta,1+beta],
 *   beta = CV(r) (Remark 1) | 6 / 7 10 % / 50 % order statistics of d2 (ceil(p n - 1e-9)-th smallest) |
 *   8 tau_hat = sqrt(sum rough / (2 #pairs)) over all cells | 9 fraction with g == 0 |
 *   10 g_q^+ = 40th percentile of g on {g > 0} (L501) | 11 g_q^+ / tau_hat | 12.. 0
 * All pointers of bsa_diag_out are device pointers owned by the caller and must not be NULL; tau must
 * not be NULL.
 */
#define BSA_DIAG_SUMMARY_LEN 16
typedef struct {
  float *g, *G, *r, *d2, *rough; /* each [B,Hq,Q_t] */
  float* summary;                /* [B, BSA_DIAG_SUMMARY_LEN] */
} bsa_diag_out;

bsa_status bsa_select_diag(const bsa_shape* shape, const void* Q, const void* meta, bsa_policy policy,
                           int32_t k_budget, double q_frac, int32_t* kv_idx, int32_t* kv_count,
                           float* sigma, float* sigma_bar, uint8_t* trigger, float* tau,
                           const bsa_diag_out* diag, void* workspace, size_t workspace_bytes, void* stream);

/*
 * Sparse attention.  For tile t, head h, row i: softmax over keys j <= i of the blocks listed in
 * kv_idx[b,h,t,0..kv_count) (kv_count may be NULL: all W slots are read), scale <= 0 means
 * 1/sqrt(head_dim).  Entries >= N_B (sentinel) or > t are skipped; the block equal to t gets the
 * causal diagonal mask; the order of entries is free; a block listed more than once is attended once.
 * O [B,Hq,N,d] bf16 (Q strides); lse [B,Hq,N] fp32 natural-log-sum-exp of the scaled logits, or NULL.
 */
bsa_status bsa_sparse_attn_fwd(const bsa_shape* shape, const void* Q, const void* K, const void* V,
                               const int32_t* kv_idx, const int32_t* kv_count, int32_t kv_width,
                               float softmax_scale, void* O, float* lse, void* stream);

/*
 * Selection and sparse attention in ONE call (rows 2-6; section 4.5 item 3, L271, names "block-
 * selection fused into the attention kernel for >= 256K" as the next engineering step).  Same arguments and
 * results as bsa_select followed by bsa_sparse_attn_fwd on its kv_idx / kv_count.  What is and is not
 * fused here: the tile scores never exist in HBM in this library (scoring, top-2k and
 * sigma are one kernel), so the call enqueues the same kernels back to back and launches the attention
 * kernel as a programmatic dependent launch -- its prologue (barriers, TMEM allocation, the Q tile load) runs
 * under the tail of the selection kernels and it waits (griddepcontrol.wait) before it reads kv_idx.  It is
 * NOT a single persistent kernel; measured, it equals the two-call path within noise at 128K and 256K.
 */
bsa_status bsa_select_attn_fwd(const bsa_shape* shape, const void* Q, const void* K, const void* V,
                               const void* meta, bsa_policy policy, int32_t k_budget, double q_frac,
                               int32_t* kv_idx, int32_t* kv_count, float* sigma, float* sigma_bar,
                               uint8_t* trigger, float* tau, float softmax_scale, void* O, float* lse,
                               void* workspace, size_t workspace_bytes, void* stream);

/* Dense causal attention with the same kernel design (every visible block). */
bsa_status bsa_dense_attn_fwd(const bsa_shape* shape, const void* Q, const void* K, const void* V,
                              float softmax_scale, void* O, float* lse, void* stream);

/*
 * Ragged batches (SURVEY 8(f).1 "varlen"): n_seqs sequences packed along the token axis, Q / O
 * [Hq, total, d], K / V [Hkv, total, d] with shape.batch = 1 and shape.seqlen = total =
 * cu_seqlens[n_seqs]; cu_seqlens is a HOST array of n_seqs + 1 offsets, cu_seqlens[0] = 0, every length a
 * multiple of shape.block (0 allowed).  Each sequence is an independent problem: its own causal frame,
 * block numbers local to the sequence (0 .. T_i - 1, sentinel T_i) and its own quantile threshold
 * (reading G9).  The calls loop over the sequences on `stream` (one set of launches per sequence).
 * Index and statistics tensors are SEQUENCE-MAJOR, sequence i first token s_i = cu_seqlens[i],
 * first tile t_i = s_i / block, T_i tiles:
 *   kv_idx   : [Hq, T_i, W] at element Hq * W * t_i      kv_count, sigma : [Hq, T_i] at Hq * t_i
 *   sigma_bar, trigger : [T_i] at t_i                    tau : [n_seqs]
 *   lse      : [Hq, N_i] at Hq * s_i
 *   meta     : sequence i at the sum over j < i of bsa_block_meta_bytes(shape with seqlen = N_j, 3)
 *              rounded up to 256 (bsa_block_meta_bytes_varlen returns the total)
 * Errors as for the batch calls; a failing sequence leaves the earlier sequences enqueued.
 */
size_t bsa_block_meta_bytes_varlen(const bsa_shape* shape, const int32_t* cu_seqlens, int32_t n_seqs,
                                   int kinds);
bsa_status bsa_build_block_meta_varlen(const bsa_shape* shape, const int32_t* cu_seqlens, int32_t n_seqs,
                                       const void* K, int kinds, void* meta, void* stream);
bsa_status bsa_select_varlen(const bsa_shape* shape, const int32_t* cu_seqlens, int32_t n_seqs, const void* Q,
                             const void* meta, bsa_policy policy, int32_t k_budget, double q_frac,
                             int32_t* kv_idx, int32_t* kv_count, float* sigma, float* sigma_bar,
                             uint8_t* trigger, float* tau, void* stream);
bsa_status bsa_sparse_attn_fwd_varlen(const bsa_shape* shape, const int32_t* cu_seqlens, int32_t n_seqs,
                                      const void* Q, const void* K, const void* V, const int32_t* kv_idx,
                                      const int32_t* kv_count, int32_t kv_width, float softmax_scale, void* O,
                                      float* lse, void* stream);
bsa_status bsa_dense_attn_fwd_varlen(const bsa_shape* shape, const int32_t* cu_seqlens, int32_t n_seqs,
                                     const void* Q, const void* K, const void* V, float softmax_scale, void* O,
                                     float* lse, void* stream);

/*
 * Per-row selection scattered into a per-tile block bitmap (section 4.5 item 1, L269: "A per-row
 * scatter-into-bitmap kernel would close the rest of the gap without re-materialising the [B, H, M, N_B]
 * keep tensor"; reading G18).  Every query row i of tile t ranks the visible blocks b <= t
 * by its OWN row score (Eq.1 with BSA_POLICY_TOPK, Eq.2 with BSA_POLICY_QUEST; no tile max), blocks 0 and t
 * forced on top (Eq.9), ties -> lower block index (G6), and keeps its first min(k_row, t+1) blocks; the
 * tile's bitmap is the union over its rows and the whole tile attends the union.
 *   bitmap   [B, Hq, Q_t, bsa_bitmap_words(shape)] uint32: bit (b % 32) of word (b / 32) = block b
 *   kv_count [B, Hq, Q_t] int32: number of set bits (between min(k_row, t+1) and min(t+1, 2 + block (k_row-2)))
 * Limits: 3 <= k_row <= 64.  bsa_sparse_attn_fwd_bitmap attends the set blocks of every row (bits above
 * t are ignored; the block equal to t gets the causal mask); N_B <= 4096.
 */
size_t bsa_bitmap_words(const bsa_shape* shape);
bsa_status bsa_select_rows_bitmap(const bsa_shape* shape, const void* Q, const void* meta, bsa_policy policy,
                                  int32_t k_row, uint32_t* bitmap, int32_t* kv_count, void* stream);
bsa_status bsa_sparse_attn_fwd_bitmap(const bsa_shape* shape, const void* Q, const void* K, const void* V,
                                      const uint32_t* bitmap, float softmax_scale, void* O, float* lse,
                                      void* stream);

/* Thread-local, static storage; never NULL. */
const char* bsa_last_error(void);

/* Library version string, e.g. "bsa 0.1 sm_100a". */
const char* bsa_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BSA_H_ */

// api.cu -- the C ABI of libbsa (include/bsa.h): argument validation, meta / workspace layout,
// dispatch to the kernels.  Nothing here touches the device except kernel launches on the caller's
// stream; no device memory is allocated and no state is kept between calls.  The one exception is
// bsa_select_static at the end of the file: its scratch is a file-scope __device__ array whose contents
// survive from call to call.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>

#include <mutex>

#include "bsa_internal.h"

namespace bsa {

static thread_local char g_err[512] = "";

bsa_status fail(bsa_status code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

bsa_status check_launch(const char* what) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(BSA_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
  return BSA_OK;
}

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

MetaLayout meta_layout(const Dims& D) {
  MetaLayout L;
  L.elems = static_cast<size_t>(D.B) * D.Hkv * D.NB * D.d;
  L.off_mean = 0;
  L.off_min = align_up(L.elems * 4, 256);
  L.off_max = L.off_min + L.elems * 2;
  L.off_split = align_up(L.off_max + L.elems * 2, 256);
  L.bytes = L.off_split + 3 * L.elems * 2;
  return L;
}

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// Shape checks shared by every entry point.
static bsa_status make_dims(const bsa_shape* s, Dims* out) {
  if (!s) return fail(BSA_ERR_INVALID_ARG, "shape is NULL");
  if (s->batch < 1 || s->seqlen < 1 || s->n_q_heads < 1 || s->n_kv_heads < 1)
    return fail(BSA_ERR_INVALID_ARG, "batch, seqlen and head counts must be positive");
  if (s->block != 64 && s->block != 128)
    return fail(BSA_ERR_UNSUPPORTED, "block %d not in {64, 128}", s->block);
  if (s->head_dim != 64 && s->head_dim != 128 && s->head_dim != 256)
    return fail(BSA_ERR_UNSUPPORTED, "head_dim %d not in {64, 128, 256}", s->head_dim);
  if (s->seqlen % s->block != 0)
    return fail(BSA_ERR_INVALID_ARG, "seqlen %d is not a multiple of block %d", s->seqlen, s->block);
  if (s->n_q_heads % s->n_kv_heads != 0)
    return fail(BSA_ERR_INVALID_ARG, "n_q_heads %d is not a multiple of n_kv_heads %d", s->n_q_heads,
                s->n_kv_heads);
  if (s->seqlen / s->block > 65535)
    return fail(BSA_ERR_UNSUPPORTED, "more than 65535 blocks per sequence");
  const int64_t st[6] = {s->q_stride_b, s->q_stride_h, s->q_stride_n,
                         s->kv_stride_b, s->kv_stride_h, s->kv_stride_n};
  for (int i = 0; i < 6; ++i)
    if (st[i] < 0 || st[i] % 8 != 0)
      return fail(BSA_ERR_INVALID_ARG, "strides must be non-negative multiples of 8 elements (16 B)");
  if (s->q_stride_n < s->head_dim || s->kv_stride_n < s->head_dim)
    return fail(BSA_ERR_INVALID_ARG, "row stride smaller than head_dim");
  Dims D;
  D.B = s->batch; D.N = s->seqlen; D.H = s->n_q_heads; D.Hkv = s->n_kv_heads; D.d = s->head_dim;
  D.Bn = s->block; D.NB = s->seqlen / s->block; D.G = s->n_q_heads / s->n_kv_heads;
  D.qsb = s->q_stride_b; D.qsh = s->q_stride_h; D.qsn = s->q_stride_n;
  D.ksb = s->kv_stride_b; D.ksh = s->kv_stride_h; D.ksn = s->kv_stride_n;
  *out = D;
  return BSA_OK;
}

static bsa_status check_device() {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(BSA_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
  int major = 0;
  e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  if (e != cudaSuccess) return fail(BSA_ERR_CUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
  if (major != 10) return fail(BSA_ERR_UNSUPPORTED, "device is sm_%d0, libbsa needs sm_100", major);
  return BSA_OK;
}

int sm_count() {
  static int cached[64] = {0};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
  if (cached[dev] == 0) {
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    cached[dev] = n;
  }
  return cached[dev];
}

static bool policy_ok(int p) { return p >= BSA_POLICY_TOPK && p <= BSA_POLICY_ROUTER_QUEST; }
static bool is_router(int p) { return p == BSA_POLICY_ROUTER || p == BSA_POLICY_ROUTER_QUEST; }

}  // namespace bsa

using namespace bsa;

extern "C" {

const char* bsa_last_error(void) { return g_err; }
const char* bsa_version(void) { return "bsa 0.1 sm_100a"; }

size_t bsa_block_meta_bytes(const bsa_shape* shape, int kinds) {
  Dims D;
  if (make_dims(shape, &D) != BSA_OK) return 0;
  if ((kinds & ~(BSA_META_MEAN | BSA_META_MINMAX)) != 0 || kinds == 0) return 0;
  return meta_layout(D).bytes;
}

size_t bsa_block_meta_offset(const bsa_shape* shape, int kind) {
  Dims D;
  if (make_dims(shape, &D) != BSA_OK) return 0;
  const MetaLayout L = meta_layout(D);
  return kind == BSA_META_MINMAX ? L.off_min : kind == BSA_META_SPLIT ? L.off_split : L.off_mean;
}

bsa_status bsa_build_block_meta(const bsa_shape* shape, const void* K, int kinds, void* meta,
                                void* stream) {
  Dims D;
  bsa_status st = make_dims(shape, &D);
  if (st != BSA_OK) return st;
  if (!K || !meta) return fail(BSA_ERR_INVALID_ARG, "K or meta is NULL");
  if ((kinds & ~(BSA_META_MEAN | BSA_META_MINMAX)) != 0 || kinds == 0)
    return fail(BSA_ERR_INVALID_ARG, "kinds must be a non-empty mask of BSA_META_MEAN | BSA_META_MINMAX");
  if (!aligned16(K) || (reinterpret_cast<uintptr_t>(meta) & 255u))
    return fail(BSA_ERR_INVALID_ARG, "K must be 16-byte and meta 256-byte aligned");
  st = check_device();
  if (st != BSA_OK) return st;
  return launch_pool(D, K, kinds, meta, static_cast<cudaStream_t>(stream));
}

int32_t bsa_kv_width(bsa_policy policy, int32_t k_budget) {
  if (!policy_ok(policy) || k_budget < 1) return 0;
  return is_router(policy) ? BSA_RHO * k_budget : k_budget;
}

size_t bsa_select_workspace_bytes(const bsa_shape* shape, bsa_policy policy, int32_t k_budget) {
  Dims D;
  if (make_dims(shape, &D) != BSA_OK || !policy_ok(policy) || k_budget < 3) return 0;
  const size_t bt = static_cast<size_t>(D.B) * D.NB;
  return align_up(bt * 4, 256) + align_up(bt, 256) + 256;
}

static bsa_status select_common(const bsa_shape* shape, const void* Q, const void* meta, bsa_policy policy,
                                int32_t k_budget, double q_frac, int32_t* kv_idx, int32_t* kv_count,
                                float* sigma, float* sigma_bar, uint8_t* trigger, float* tau,
                                const bsa_diag_out* diag, bool want_diag, void* workspace,
                                size_t workspace_bytes, void* stream) {
  Dims D;
  bsa_status st = make_dims(shape, &D);
  if (st != BSA_OK) return st;
  if (!Q || !meta || !kv_idx || !kv_count || !sigma)
    return fail(BSA_ERR_INVALID_ARG, "Q, meta, kv_idx, kv_count and sigma must not be NULL");
  if (!policy_ok(policy)) return fail(BSA_ERR_INVALID_ARG, "unknown policy %d", static_cast<int>(policy));
  if (k_budget < 3) return fail(BSA_ERR_INVALID_ARG, "k_budget %d < 3", k_budget);
  if (k_budget > 128) return fail(BSA_ERR_UNSUPPORTED, "k_budget %d > 128", k_budget);
  if (is_router(policy) && !(q_frac >= 0.0 && q_frac <= 1.0))
    return fail(BSA_ERR_INVALID_ARG, "q_frac %g outside [0, 1]", q_frac);
  if (!aligned16(Q) || (reinterpret_cast<uintptr_t>(meta) & 255u))
    return fail(BSA_ERR_INVALID_ARG, "Q must be 16-byte and meta 256-byte aligned");
  if (D.NB > 8192)
    return fail(BSA_ERR_UNSUPPORTED, "select: %d blocks per sequence, at most 8192 are supported", D.NB);
  SelectDiag dg = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  if (want_diag) {
    if (!diag || !diag->g || !diag->G || !diag->r || !diag->d2 || !diag->rough || !diag->summary || !tau)
      return fail(BSA_ERR_INVALID_ARG, "diagnostics: every bsa_diag_out pointer and tau must be given");
    dg = {diag->g, diag->G, diag->r, diag->d2, diag->rough, diag->summary};
  }
  const size_t need = bsa_select_workspace_bytes(shape, policy, k_budget);
  if ((!sigma_bar || !trigger) && (!workspace || workspace_bytes < need))
    return fail(BSA_ERR_WORKSPACE_TOO_SMALL, "workspace of %zu bytes needed, %zu given", need,
                workspace_bytes);
  st = check_device();
  if (st != BSA_OK) return st;
  const size_t bt = static_cast<size_t>(D.B) * D.NB;
  char* ws = static_cast<char*>(workspace);
  if (ws) ws = reinterpret_cast<char*>(align_up(reinterpret_cast<uintptr_t>(ws), 256));
  if (!sigma_bar) sigma_bar = reinterpret_cast<float*>(ws);
  if (!trigger) trigger = reinterpret_cast<uint8_t*>(ws + align_up(bt * 4, 256));
  long long m = 0;  // O9: m = ceil(q*T - 1e-9), clamped to [0, T]
  if (is_router(policy)) {
    m = static_cast<long long>(ceil(q_frac * static_cast<double>(D.NB) - 1e-9));
    if (m < 0) m = 0;
    if (m > D.NB) m = D.NB;
  }
  const int W = bsa_kv_width(policy, k_budget);
  return launch_select(D, Q, meta, policy, k_budget, W, m, kv_idx, kv_count, sigma, sigma_bar, trigger,
                       tau, dg, static_cast<cudaStream_t>(stream));
}

bsa_status bsa_select(const bsa_shape* shape, const void* Q, const void* meta, bsa_policy policy,
                      int32_t k_budget, double q_frac, int32_t* kv_idx, int32_t* kv_count,
                      float* sigma, float* sigma_bar, uint8_t* trigger, float* tau, void* workspace,
                      size_t workspace_bytes, void* stream) {
  return select_common(shape, Q, meta, policy, k_budget, q_frac, kv_idx, kv_count, sigma, sigma_bar,
                       trigger, tau, nullptr, false, workspace, workspace_bytes, stream);
}

bsa_status bsa_select_diag(const bsa_shape* shape, const void* Q, const void* meta, bsa_policy policy,
                           int32_t k_budget, double q_frac, int32_t* kv_idx, int32_t* kv_count,
                           float* sigma, float* sigma_bar, uint8_t* trigger, float* tau,
                           const bsa_diag_out* diag, void* workspace, size_t workspace_bytes,
                           void* stream) {
  return select_common(shape, Q, meta, policy, k_budget, q_frac, kv_idx, kv_count, sigma, sigma_bar,
                       trigger, tau, diag, true, workspace, workspace_bytes, stream);
}

static bsa_status attn_common(const bsa_shape* shape, const void* Q, const void* K, const void* V,
                              const int32_t* kv_idx, const int32_t* kv_count, int32_t kv_width,
                              bool sparse, float softmax_scale, void* O, float* lse, void* stream,
                              bool pdl = false) {
  Dims D;
  bsa_status st = make_dims(shape, &D);
  if (st != BSA_OK) return st;
  if (!Q || !K || !V || !O) return fail(BSA_ERR_INVALID_ARG, "Q, K, V and O must not be NULL");
  if (sparse && (!kv_idx || kv_width < 1))
    return fail(BSA_ERR_INVALID_ARG, "kv_idx is NULL or kv_width < 1");
  if (!aligned16(Q) || !aligned16(K) || !aligned16(V) || !aligned16(O))
    return fail(BSA_ERR_INVALID_ARG, "Q, K, V and O must be 16-byte aligned");
  st = check_device();
  if (st != BSA_OK) return st;
  const float scale = softmax_scale > 0.f ? softmax_scale
                                          : static_cast<float>(1.0 / sqrt(static_cast<double>(D.d)));
  return launch_attn(D, Q, K, V, kv_idx, kv_count, kv_width, sparse, scale, O, lse,
                     static_cast<cudaStream_t>(stream), nullptr, pdl);
}

bsa_status bsa_sparse_attn_fwd(const bsa_shape* shape, const void* Q, const void* K, const void* V,
                               const int32_t* kv_idx, const int32_t* kv_count, int32_t kv_width,
                               float softmax_scale, void* O, float* lse, void* stream) {
  return attn_common(shape, Q, K, V, kv_idx, kv_count, kv_width, true, softmax_scale, O, lse, stream);
}

bsa_status bsa_select_attn_fwd(const bsa_shape* shape, const void* Q, const void* K, const void* V,
                               const void* meta, bsa_policy policy, int32_t k_budget, double q_frac,
                               int32_t* kv_idx, int32_t* kv_count, float* sigma, float* sigma_bar,
                               uint8_t* trigger, float* tau, float softmax_scale, void* O, float* lse,
                               void* workspace, size_t workspace_bytes, void* stream) {
  // every argument of the attention half is checked before the selection is enqueued
  Dims D;
  bsa_status st = make_dims(shape, &D);
  if (st != BSA_OK) return st;
  if (!K || !V || !O) return fail(BSA_ERR_INVALID_ARG, "K, V and O must not be NULL");
  if (!aligned16(K) || !aligned16(V) || !aligned16(O))
    return fail(BSA_ERR_INVALID_ARG, "K, V and O must be 16-byte aligned");
  st = select_common(shape, Q, meta, policy, k_budget, q_frac, kv_idx, kv_count, sigma, sigma_bar, trigger,
                     tau, nullptr, false, workspace, workspace_bytes, stream);
  if (st != BSA_OK) return st;
  return attn_common(shape, Q, K, V, kv_idx, kv_count, bsa_kv_width(policy, k_budget), true, softmax_scale,
                     O, lse, stream, /*pdl=*/true);
}

bsa_status bsa_dense_attn_fwd(const bsa_shape* shape, const void* Q, const void* K, const void* V,
                              float softmax_scale, void* O, float* lse, void* stream) {
  return attn_common(shape, Q, K, V, nullptr, nullptr, 0, false, softmax_scale, O, lse, stream);
}

/* ---- ragged batches (SURVEY 8(f).1 "varlen") ------------------------------------------------------
 * A loop over the sequences on the caller's stream; every sequence is an independent batch-1 problem
 * (own causal frame, own block numbering, own quantile -- reading G9). */
static bsa_status varlen_check(const bsa_shape* shape, const int32_t* cu, int32_t n_seqs) {
  if (!shape || !cu) return fail(BSA_ERR_INVALID_ARG, "shape or cu_seqlens is NULL");
  if (n_seqs < 1) return fail(BSA_ERR_INVALID_ARG, "n_seqs %d < 1", n_seqs);
  if (shape->batch != 1) return fail(BSA_ERR_INVALID_ARG, "varlen: shape.batch must be 1 (packed layout)");
  if (shape->block != 64 && shape->block != 128)
    return fail(BSA_ERR_UNSUPPORTED, "block %d not in {64, 128}", shape->block);
  if (cu[0] != 0 || cu[n_seqs] != shape->seqlen)
    return fail(BSA_ERR_INVALID_ARG, "cu_seqlens must run from 0 to shape.seqlen (%d)", shape->seqlen);
  for (int i = 0; i < n_seqs; ++i) {
    const int len = cu[i + 1] - cu[i];
    if (len < 0 || len % shape->block != 0)
      return fail(BSA_ERR_INVALID_ARG, "sequence %d: length %d is negative or not a multiple of block %d", i,
                  len, shape->block);
  }
  return BSA_OK;
}

static bsa_shape sub_shape(const bsa_shape* shape, int len) {
  bsa_shape s = *shape;
  s.seqlen = len;
  return s;
}

static size_t meta_bytes_padded(const bsa_shape* s, int kinds) {
  return align_up(bsa_block_meta_bytes(s, kinds), 256);
}

size_t bsa_block_meta_bytes_varlen(const bsa_shape* shape, const int32_t* cu_seqlens, int32_t n_seqs,
                                   int kinds) {
  if (varlen_check(shape, cu_seqlens, n_seqs) != BSA_OK) return 0;
  size_t total = 0;
  for (int i = 0; i < n_seqs; ++i) {
    const int len = cu_seqlens[i + 1] - cu_seqlens[i];
    if (len == 0) continue;
    const bsa_shape s = sub_shape(shape, len);
    const size_t b = meta_bytes_padded(&s, kinds);
    if (b == 0) return 0;
    total += b;
  }
  return total;
}

bsa_status bsa_build_block_meta_varlen(const bsa_shape* shape, const int32_t* cu_seqlens, int32_t n_seqs,
                                       const void* K, int kinds, void* meta, void* stream) {
  bsa_status st = varlen_check(shape, cu_seqlens, n_seqs);
  if (st != BSA_OK) return st;
  if (!K || !meta) return fail(BSA_ERR_INVALID_ARG, "K or meta is NULL");
  size_t off = 0;
  for (int i = 0; i < n_seqs; ++i) {
    const int start = cu_seqlens[i], len = cu_seqlens[i + 1] - start;
    if (len == 0) continue;
    const bsa_shape s = sub_shape(shape, len);
    const char* Ki = static_cast<const char*>(K) + static_cast<int64_t>(start) * shape->kv_stride_n * 2;
    st = bsa_build_block_meta(&s, Ki, kinds, static_cast<char*>(meta) + off, stream);
    if (st != BSA_OK) return st;
    off += meta_bytes_padded(&s, kinds);
  }
  return BSA_OK;
}

bsa_status bsa_select_varlen(const bsa_shape* shape, const int32_t* cu_seqlens, int32_t n_seqs, const void* Q,
                             const void* meta, bsa_policy policy, int32_t k_budget, double q_frac,
                             int32_t* kv_idx, int32_t* kv_count, float* sigma, float* sigma_bar,
                             uint8_t* trigger, float* tau, void* stream) {
  bsa_status st = varlen_check(shape, cu_seqlens, n_seqs);
  if (st != BSA_OK) return st;
  if (!Q || !meta || !kv_idx || !kv_count || !sigma || !sigma_bar || !trigger || !tau)
    return fail(BSA_ERR_INVALID_ARG, "varlen select: every output pointer must be given");
  const int W = bsa_kv_width(policy, k_budget);
  if (W < 1) return fail(BSA_ERR_INVALID_ARG, "unknown policy or k_budget < 1");
  const int64_t H = shape->n_q_heads;
  size_t moff = 0;
  for (int i = 0; i < n_seqs; ++i) {
    const int start = cu_seqlens[i], len = cu_seqlens[i + 1] - start;
    if (len == 0) continue;
    const int64_t t0 = start / shape->block;
    const bsa_shape s = sub_shape(shape, len);
    const char* Qi = static_cast<const char*>(Q) + static_cast<int64_t>(start) * shape->q_stride_n * 2;
    st = bsa_select(&s, Qi, static_cast<const char*>(meta) + moff, policy, k_budget, q_frac,
                    kv_idx + H * W * t0, kv_count + H * t0, sigma + H * t0, sigma_bar + t0, trigger + t0,
                    tau + i, nullptr, 0, stream);
    if (st != BSA_OK) return st;
    moff += meta_bytes_padded(&s, BSA_META_MEAN | BSA_META_MINMAX);
  }
  return BSA_OK;
}

static bsa_status attn_varlen(const bsa_shape* shape, const int32_t* cu, int32_t n_seqs, const void* Q,
                              const void* K, const void* V, const int32_t* kv_idx, const int32_t* kv_count,
                              int32_t W, bool sparse, float scale, void* O, float* lse, void* stream) {
  bsa_status st = varlen_check(shape, cu, n_seqs);
  if (st != BSA_OK) return st;
  if (!Q || !K || !V || !O) return fail(BSA_ERR_INVALID_ARG, "Q, K, V and O must not be NULL");
  const int64_t H = shape->n_q_heads;
  for (int i = 0; i < n_seqs; ++i) {
    const int start = cu[i], len = cu[i + 1] - start;
    if (len == 0) continue;
    const int64_t t0 = start / shape->block;
    const bsa_shape s = sub_shape(shape, len);
    const int64_t qo = static_cast<int64_t>(start) * shape->q_stride_n * 2;
    const int64_t ko = static_cast<int64_t>(start) * shape->kv_stride_n * 2;
    st = attn_common(&s, static_cast<const char*>(Q) + qo, static_cast<const char*>(K) + ko,
                     static_cast<const char*>(V) + ko, sparse ? kv_idx + H * W * t0 : nullptr,
                     (sparse && kv_count) ? kv_count + H * t0 : nullptr, W, sparse, scale,
                     static_cast<char*>(O) + qo, lse ? lse + H * start : nullptr, stream);
    if (st != BSA_OK) return st;
  }
  return BSA_OK;
}

bsa_status bsa_sparse_attn_fwd_varlen(const bsa_shape* shape, const int32_t* cu_seqlens, int32_t n_seqs,
                                      const void* Q, const void* K, const void* V, const int32_t* kv_idx,
                                      const int32_t* kv_count, int32_t kv_width, float softmax_scale, void* O,
                                      float* lse, void* stream) {
  if (!kv_idx || kv_width < 1) return fail(BSA_ERR_INVALID_ARG, "kv_idx is NULL or kv_width < 1");
  return attn_varlen(shape, cu_seqlens, n_seqs, Q, K, V, kv_idx, kv_count, kv_width, true, softmax_scale, O,
                     lse, stream);
}

bsa_status bsa_dense_attn_fwd_varlen(const bsa_shape* shape, const int32_t* cu_seqlens, int32_t n_seqs,
                                     const void* Q, const void* K, const void* V, float softmax_scale, void* O,
                                     float* lse, void* stream) {
  return attn_varlen(shape, cu_seqlens, n_seqs, Q, K, V, nullptr, nullptr, 0, false, softmax_scale, O, lse,
                     stream);
}

/* ---- per-row selection scattered into a per-tile bitmap ---------------- */
size_t bsa_bitmap_words(const bsa_shape* shape) {
  Dims D;
  if (make_dims(shape, &D) != BSA_OK) return 0;
  return static_cast<size_t>((D.NB + 31) / 32);
}

bsa_status bsa_select_rows_bitmap(const bsa_shape* shape, const void* Q, const void* meta, bsa_policy policy,
                                  int32_t k_row, uint32_t* bitmap, int32_t* kv_count, void* stream) {
  Dims D;
  bsa_status st = make_dims(shape, &D);
  if (st != BSA_OK) return st;
  if (!Q || !meta || !bitmap || !kv_count)
    return fail(BSA_ERR_INVALID_ARG, "Q, meta, bitmap and kv_count must not be NULL");
  if (policy != BSA_POLICY_TOPK && policy != BSA_POLICY_QUEST)
    return fail(BSA_ERR_INVALID_ARG, "rows_bitmap: policy must be BSA_POLICY_TOPK (K-mean) or BSA_POLICY_QUEST");
  if (k_row < 3) return fail(BSA_ERR_INVALID_ARG, "k_row %d < 3", k_row);
  if (k_row > 64) return fail(BSA_ERR_UNSUPPORTED, "k_row %d > 64", k_row);
  if (!aligned16(Q) || (reinterpret_cast<uintptr_t>(meta) & 255u))
    return fail(BSA_ERR_INVALID_ARG, "Q must be 16-byte and meta 256-byte aligned");
  st = check_device();
  if (st != BSA_OK) return st;
  return launch_rowsel(D, Q, meta, policy == BSA_POLICY_QUEST, k_row, bitmap, kv_count,
                       static_cast<cudaStream_t>(stream));
}

bsa_status bsa_sparse_attn_fwd_bitmap(const bsa_shape* shape, const void* Q, const void* K, const void* V,
                                      const uint32_t* bitmap, float softmax_scale, void* O, float* lse,
                                      void* stream) {
  Dims D;
  bsa_status st = make_dims(shape, &D);
  if (st != BSA_OK) return st;
  if (!Q || !K || !V || !O || !bitmap) return fail(BSA_ERR_INVALID_ARG, "Q, K, V, O and bitmap must not be NULL");
  if (!aligned16(Q) || !aligned16(K) || !aligned16(V) || !aligned16(O))
    return fail(BSA_ERR_INVALID_ARG, "Q, K, V and O must be 16-byte aligned");
  st = check_device();
  if (st != BSA_OK) return st;
  const float scale = softmax_scale > 0.f ? softmax_scale
                                          : static_cast<float>(1.0 / sqrt(static_cast<double>(D.d)));
  return launch_attn(D, Q, K, V, nullptr, nullptr, 0, true, scale, O, lse, static_cast<cudaStream_t>(stream),
                     bitmap);
}

}  // extern "C"

/* ---- bsa_select_static: selection for callers that cannot allocate (include/bsa.h) -------------------------
 * sigma_bar [B, Q_t] fp32 and trigger [B, Q_t] u8 -- the scratch bsa_select otherwise takes from the caller's
 * workspace -- live in this file-scope array, in the layout of the workspace route (bsa_select_workspace_bytes).
 * Every GPU that loads libbsa holds the array until the process exits.  In host code `g_static_scratch` is a
 * host-side stand-in, not a device address: the kernels get the pointer cudaGetSymbolAddress returns, looked
 * up once per device with that device current. */
static constexpr size_t kStaticScratchBytes =
    (static_cast<size_t>(BSA_STATIC_MAX_TILES) * 4 + 255) / 256 * 256 +   // sigma_bar
    (static_cast<size_t>(BSA_STATIC_MAX_TILES) + 255) / 256 * 256 + 256;  // trigger + the workspace slack
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

static constexpr int kMaxDevices = 64;
static std::mutex g_static_mu;
static void* g_static_addr[kMaxDevices] = {nullptr};

// Device address of g_static_scratch on the current device (cached per device ordinal).
static bsa_status static_scratch_addr(void** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(BSA_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kMaxDevices)
    return fail(BSA_ERR_UNSUPPORTED, "bsa_select_static: device ordinal %d outside [0, %d)", dev, kMaxDevices);
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || !p)
      return fail(BSA_ERR_CUDA, "cudaGetSymbolAddress(static scratch): %s", cudaGetErrorString(e));
    g_static_addr[dev] = p;
  }
  *out = g_static_addr[dev];
  return BSA_OK;
}

extern "C" bsa_status bsa_select_static(const bsa_shape* shape, const void* Q, const void* meta,
                                        bsa_policy policy, int32_t k_budget, double q_frac, int32_t* kv_idx,
                                        int32_t* kv_count, float* sigma, float* tau, void* stream) {
  Dims D;
  bsa_status st = make_dims(shape, &D);
  if (st != BSA_OK) return st;
  const size_t tiles = static_cast<size_t>(D.B) * D.NB;
  if (tiles > static_cast<size_t>(BSA_STATIC_MAX_TILES))
    return fail(BSA_ERR_UNSUPPORTED,
                "bsa_select_static: batch * Q_t = %zu tiles, the static scratch holds at most %d "
                "(use bsa_select with a caller workspace)", tiles, BSA_STATIC_MAX_TILES);
  if (!Q || !meta || !kv_idx || !kv_count || !sigma)
    return fail(BSA_ERR_INVALID_ARG, "Q, meta, kv_idx, kv_count and sigma must not be NULL");
  st = check_device();
  if (st != BSA_OK) return st;
  void* scratch = nullptr;
  st = static_scratch_addr(&scratch);
  if (st != BSA_OK) return st;
  // the workspace route of bsa_select with the static array as the workspace: the remaining argument checks
  // run there before anything is enqueued.  Nothing in the scratch has to start at zero -- route_kernel
  // writes every sigma_bar / trigger element of this call before finalize_kernel reads trigger.
  return select_common(shape, Q, meta, policy, k_budget, q_frac, kv_idx, kv_count, sigma, nullptr, nullptr,
                       tau, nullptr, false, scratch, kStaticScratchBytes, stream);
}

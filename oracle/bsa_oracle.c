/*
 * bsa_oracle.c -- plain, slow CPU oracle for the selection + sparse-attention prefill path of
 * arxiv/paper_2607_07724 ("Uncertainty-gated selection for block-sparse attention").
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call it.  It shares no code with the CUDA library
 * (paper_2607_07724_b200/csrc) and neither includes the other.
 *
 * Every function follows the paper step by step (citations are PAPER.md line numbers + equation)
 * with the readings G1..G17 of SURVEY.md 8(c) / DESIGN.md "Readings".  Inputs are bf16 bit patterns
 * (uint16), widened exactly to fp32.  Dot products, the pooling sum and the softmax sums accumulate
 * in double and are rounded once to fp32 ("correctly rounded fp32", reading G11).
 * No blocking, no SIMD intrinsics, no BLAS; OpenMP only over independent (tile, head) pairs.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): brute force in numpy on tiny inputs, hand-worked
 * margin examples E1..E5 (tests/golden/margin_examples.txt), sigma in [0,1] and affine invariance,
 * Quest upper bound (L54, L82), routed count = ceil(qT) (L426), Eq.15 closed form (L346),
 * k_budget >= N_B  =>  sparse == dense, dense == torch CPU SDPA (library routine).
 * D.4 diagnostics (orc_diag_cells / orc_roughness / orc_diag_summary): hand-worked examples D1-D3
 * (tests/golden/diag_examples.txt), closed forms (identical / alternating rows), numpy brute force.
 * Per-row bitmap selection (orc_select_rows_bitmap, L269): numpy brute force, identical rows reduce to
 * the per-tile selection, k_row >= N_B selects every visible block, count bounds.
 * Parity unpinned (conventions fixed by fiat): G5 (sigma := 1 when nothing is dropped),
 * G6 (tie-break: lower block index first), G7 (GQA mapping h -> h / (H/H_kv)), G9 (per-sequence
 * quantile; batch is looped by the caller).
 *
 * Layouts (single sequence; the Python wrapper loops over batch):
 *   Q [H, N, d], K/V [Hkv, N, d] bf16 bits, contiguous.
 *   kmean [Hkv, N_B, d] fp32; kmin, kmax [Hkv, N_B, d] bf16 bits.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

static inline float bf16f(uint16_t h) {
  union { float f; uint32_t u; } v; v.u = ((uint32_t)h) << 16; return v.f;
}

enum { POLICY_TOPK = 0, POLICY_ROUTER = 1, POLICY_QUEST = 2, POLICY_ROUTER_QUEST = 3 };
#define RHO 2 /* L129 */

/* ---------------------------------------------------------------------------------------------
 * O1 / O2  block pooling.
 *   Eq.1 / Eq.6 (L74, L293): kbar_b = (1/BLOCK_N) sum_{j in block b} k_j
 *   Eq.2 (L78-80): element-wise K_b^min, K_b^max
 * ------------------------------------------------------------------------------------------- */
void orc_pool(const uint16_t* K, int64_t Hkv, int64_t N, int64_t d, int64_t Bn,
              float* kmean, uint16_t* kmin, uint16_t* kmax) {
  int64_t NB = N / Bn;
#pragma omp parallel for collapse(2) schedule(static)
  for (int64_t g = 0; g < Hkv; ++g)
    for (int64_t b = 0; b < NB; ++b)
      for (int64_t c = 0; c < d; ++c) {
        double sum = 0.0;
        uint16_t mn = 0, mx = 0;
        for (int64_t j = 0; j < Bn; ++j) {
          uint16_t bits = K[(g * N + b * Bn + j) * d + c];
          float v = bf16f(bits);
          sum += (double)v;
          if (j == 0) { mn = bits; mx = bits; }
          else {
            if (v < bf16f(mn)) mn = bits;
            if (v > bf16f(mx)) mx = bits;
          }
        }
        int64_t o = (g * NB + b) * d + c;
        if (kmean) kmean[o] = (float)(sum / (double)Bn);
        if (kmin) kmin[o] = mn;
        if (kmax) kmax[o] = mx;
      }
}

/* ---------------------------------------------------------------------------------------------
 * O3 / O3q  per-row block score.
 *   mean  (Eq.1 / Eq.7): s = (q . kbar_b) / sqrt(d)   -> fp32(dot) * fp32(1/sqrt(d))
 *   Quest (Eq.2): s = sum_c max(q_c Kmax_c, q_c Kmin_c)     (no 1/sqrt(d), reading G8)
 * ------------------------------------------------------------------------------------------- */
static float row_score_mean(const uint16_t* q, const float* km, int64_t d) {
  double acc = 0.0;
  for (int64_t c = 0; c < d; ++c) acc += (double)bf16f(q[c]) * (double)km[c];
  float inv_sqrt_d = (float)(1.0 / sqrt((double)d));
  return (float)acc * inv_sqrt_d;
}

static float row_score_quest(const uint16_t* q, const uint16_t* kmn, const uint16_t* kmx, int64_t d) {
  double acc = 0.0;
  for (int64_t c = 0; c < d; ++c) {
    double qc = (double)bf16f(q[c]);
    double a = qc * (double)bf16f(kmx[c]);
    double b = qc * (double)bf16f(kmn[c]);
    acc += (a > b) ? a : b;
  }
  return (float)acc;
}

/* O4 (Eq.3 / Eq.8): tile_score[t,h,b] = max_{r in tile t} s[r,h,b], visible b <= t (G4) */
static void tile_scores(const uint16_t* Q, const float* kmean, const uint16_t* kmin,
                        const uint16_t* kmax, int64_t H, int64_t Hkv, int64_t N, int64_t d,
                        int64_t Bn, int quest, int64_t t, int64_t h, float* ts /* [t+1] */) {
  int64_t NB = N / Bn, G = H / Hkv, g = h / G; /* G7 */
  (void)NB;
  for (int64_t b = 0; b <= t; ++b) {
    float best = -INFINITY;
    for (int64_t r = 0; r < Bn; ++r) {
      const uint16_t* q = Q + (h * N + t * Bn + r) * d;
      int64_t o = (g * (N / Bn) + b) * d;
      float s = quest ? row_score_quest(q, kmin + o, kmax + o, d) : row_score_mean(q, kmean + o, d);
      if (s > best) best = s;
    }
    ts[b] = best;
  }
}

/* O6 comparator: score descending, ties -> lower block index first (G6). */
typedef struct { float s; int32_t b; } cand_t;
static int cand_cmp(const void* pa, const void* pb) {
  const cand_t* a = (const cand_t*)pa; const cand_t* b = (const cand_t*)pb;
  if (a->s > b->s) return -1;
  if (a->s < b->s) return 1;
  return (a->b > b->b) - (a->b < b->b);
}

/*
 * O5-O7 for one (t, h) given its tile scores ts[0..t]:
 *   O5 (Eq.9): forced F = {0, t} rank on top, sink before self.
 *   O6 (Eq.10): sorted prefix; idx_sorted = [0, t, free blocks by score desc].
 *   O7 (Eq.4 / Eq.11; reading G1, G5):
 *        n = t+1 <= k          -> sigma = 1
 *        else num = s~[k-1]-s~[k], den = s~[f]-s~[k] (fp32), sigma = den==0 ? 0 : num/den
 * Outputs: idx_sorted[W2] (padded with NB), score_sorted[W2+1] (forced = +inf, padded with -inf).
 * W2 = RHO*k.
 */
static float select_one(const float* ts, int64_t t, int64_t NB, int64_t k,
                        int32_t* idx_sorted, float* score_sorted, cand_t* scratch) {
  int64_t W2 = RHO * k;
  int64_t n = t + 1;
  int64_t f = (t == 0) ? 1 : 2;
  int64_t nf = n - f;
  for (int64_t i = 0; i < nf; ++i) { scratch[i].s = ts[i + 1]; scratch[i].b = (int32_t)(i + 1); }
  qsort(scratch, (size_t)nf, sizeof(cand_t), cand_cmp);
  for (int64_t i = 0; i <= W2; ++i) {
    int32_t idx; float sc;
    if (i == 0) { idx = 0; sc = INFINITY; }
    else if (i == 1 && t > 0) { idx = (int32_t)t; sc = INFINITY; }
    else if (i - f < nf) { idx = scratch[i - f].b; sc = scratch[i - f].s; }
    else { idx = (int32_t)NB; sc = -INFINITY; }
    if (i < W2) idx_sorted[i] = idx;
    score_sorted[i] = sc;
  }
  if (n <= k) return 1.0f;                                     /* G5 */
  float sk1 = scratch[k - 1 - f].s, sk = scratch[k - f].s, s0 = scratch[0].s;
  float num = sk1 - sk, den = s0 - sk;
  return (den == 0.0f) ? 0.0f : num / den;                     /* L324 */
}

/*
 * Selection front half for a list of tiles (all heads): tile scores, sorted prefix, sigma.
 *   tiles[n_tiles]        tile ids t
 *   idx_sorted  [n_tiles, H, 2k]     int32, padded with N_B
 *   score_sorted[n_tiles, H, 2k+1]   fp32 (forced = +inf, missing = -inf)
 *   sigma       [n_tiles, H]
 *   tile_score  [n_tiles, H, N_B] or NULL; invisible blocks = -inf
 */
void orc_select_tiles(const uint16_t* Q, const float* kmean, const uint16_t* kmin,
                      const uint16_t* kmax, int64_t H, int64_t Hkv, int64_t N, int64_t d, int64_t Bn,
                      int policy, int64_t k, const int64_t* tiles, int64_t n_tiles,
                      int32_t* idx_sorted, float* score_sorted, float* sigma, float* tile_score) {
  int64_t NB = N / Bn, W2 = RHO * k;
  int quest = (policy == POLICY_QUEST || policy == POLICY_ROUTER_QUEST);
#pragma omp parallel
  {
    float* ts = (float*)malloc(sizeof(float) * (size_t)NB);
    cand_t* scratch = (cand_t*)malloc(sizeof(cand_t) * (size_t)NB);
#pragma omp for collapse(2) schedule(dynamic, 1)
    for (int64_t it = 0; it < n_tiles; ++it)
      for (int64_t h = 0; h < H; ++h) {
        int64_t t = tiles[it];
        tile_scores(Q, kmean, kmin, kmax, H, Hkv, N, d, Bn, quest, t, h, ts);
        int64_t o = it * H + h;
        sigma[o] = select_one(ts, t, NB, k, idx_sorted + o * W2, score_sorted + o * (W2 + 1), scratch);
        if (tile_score) {
          for (int64_t b = 0; b < NB; ++b) tile_score[o * NB + b] = (b <= t) ? ts[b] : -INFINITY;
        }
      }
    free(ts); free(scratch);
  }
}

/* Same as select_one but from caller-provided tile scores (used by the hand-worked examples). */
float orc_select_from_scores(const float* ts, int64_t t, int64_t NB, int64_t k,
                             int32_t* idx_sorted, float* score_sorted) {
  cand_t* scratch = (cand_t*)malloc(sizeof(cand_t) * (size_t)(NB + 1));
  float s = select_one(ts, t, NB, k, idx_sorted, score_sorted, scratch);
  free(scratch);
  return s;
}

/* ---------------------------------------------------------------------------------------------
 * O8-O9  head aggregation, per-layer quantile, trigger.
 *   O8 (Eq.12): sigma_bar[t] = (sum_h sigma[t,h], fp32, ascending h) / (float)H
 *   O9 (Eq.5 / Eq.13; readings G2, G3, G15; L426, L460):
 *       m = ceil(q*T - 1e-9) clamped to [0,T]; m == 0 -> no trigger, tau = -1;
 *       tau = m-th smallest sigma_bar (1-indexed order statistic); trigger = sigma_bar <= tau.
 *       Non-router policies: no trigger, tau = -1.
 * sigma layout here is [T, H].
 * ------------------------------------------------------------------------------------------- */
static int float_cmp(const void* a, const void* b) {
  float x = *(const float*)a, y = *(const float*)b;
  return (x > y) - (x < y);
}

void orc_route(const float* sigma, int64_t T, int64_t H, int policy, double q_frac,
               float* sigma_bar, float* tau_out, uint8_t* trigger) {
  for (int64_t t = 0; t < T; ++t) {
    float acc = 0.0f;
    for (int64_t h = 0; h < H; ++h) acc = acc + sigma[t * H + h];
    sigma_bar[t] = acc / (float)H;
    trigger[t] = 0;
  }
  *tau_out = -1.0f;
  if (!(policy == POLICY_ROUTER || policy == POLICY_ROUTER_QUEST)) return;
  int64_t m = (int64_t)ceil(q_frac * (double)T - 1e-9);
  if (m < 0) m = 0;
  if (m > T) m = T;
  if (m == 0) return;
  float* tmp = (float*)malloc(sizeof(float) * (size_t)T);
  memcpy(tmp, sigma_bar, sizeof(float) * (size_t)T);
  qsort(tmp, (size_t)T, sizeof(float), float_cmp);
  float tau = tmp[m - 1];
  free(tmp);
  *tau_out = tau;
  for (int64_t t = 0; t < T; ++t) trigger[t] = (sigma_bar[t] <= tau) ? 1 : 0;
}

/* ---------------------------------------------------------------------------------------------
 * O10 (Eq.14): padded expansion.
 *   cnt = min(trigger ? RHO*k : k, t+1); kv_idx[t,h,0..cnt) = idx_sorted[t,h,0..cnt); rest = N_B.
 *   idx_sorted [T, H, 2k] ; kv_idx [H, T, W] ; kv_count [H, T]   (W = k or 2k)
 * ------------------------------------------------------------------------------------------- */
void orc_fill(const int32_t* idx_sorted, const uint8_t* trigger, int64_t T, int64_t H, int64_t NB,
              int64_t k, int64_t W, int32_t* kv_idx, int32_t* kv_count) {
  int64_t W2 = RHO * k;
  for (int64_t t = 0; t < T; ++t)
    for (int64_t h = 0; h < H; ++h) {
      int64_t budget = trigger[t] ? W2 : k;
      if (budget > W) budget = W;
      int64_t cnt = (budget < t + 1) ? budget : t + 1;
      for (int64_t i = 0; i < W; ++i)
        kv_idx[(h * T + t) * W + i] = (i < cnt) ? idx_sorted[(t * H + h) * W2 + i] : (int32_t)NB;
      kv_count[h * T + t] = (int32_t)cnt;
    }
}

/* ---------------------------------------------------------------------------------------------
 * O11 / O12  attention (L43-47 softmax definition; L131, L342 iteration over kv_idx, sentinel
 * skip).  For each listed (t, h) pair and each row i of tile t:
 *     J = { j in selected blocks : j <= i },  l_j = (q_i . k_j) * scale,
 *     o_i = sum_J exp(l_j - max) v_j / sum_J exp(l_j - max),   lse_i = max + ln(sum)
 * dense != 0 ignores kv_idx and uses every block b <= t (O12).
 * Entries >= N_B or > t are skipped (sentinel, L342); duplicates are attended once.
 *   pairs [n_pairs, 2] = (t, h);  O [n_pairs, Bn, d] fp32;  lse [n_pairs, Bn] fp32
 * ------------------------------------------------------------------------------------------- */
void orc_attn_pairs(const uint16_t* Q, const uint16_t* K, const uint16_t* V, int64_t H, int64_t Hkv,
                    int64_t N, int64_t d, int64_t Bn, const int32_t* kv_idx, const int32_t* kv_count,
                    int64_t W, int dense, double scale, const int64_t* pairs, int64_t n_pairs,
                    float* O, float* lse) {
  int64_t NB = N / Bn, T = NB, G = H / Hkv;
#pragma omp parallel
  {
    uint8_t* sel = (uint8_t*)malloc((size_t)NB);
    double* logit = (double*)malloc(sizeof(double) * (size_t)N);
    double* acc = (double*)malloc(sizeof(double) * (size_t)d);
#pragma omp for schedule(dynamic, 1)
    for (int64_t ip = 0; ip < n_pairs; ++ip) {
      int64_t t = pairs[2 * ip], h = pairs[2 * ip + 1], g = h / G;
      memset(sel, 0, (size_t)NB);
      if (dense) { for (int64_t b = 0; b <= t; ++b) sel[b] = 1; }
      else {
        int64_t cnt = kv_count ? kv_count[h * T + t] : W;
        for (int64_t i = 0; i < cnt && i < W; ++i) {
          int32_t b = kv_idx[(h * T + t) * W + i];
          if (b >= 0 && b < NB && b <= t) sel[b] = 1;
        }
      }
      for (int64_t r = 0; r < Bn; ++r) {
        int64_t i = t * Bn + r;
        const uint16_t* q = Q + (h * N + i) * d;
        double mx = -INFINITY;
        for (int64_t b = 0; b <= t; ++b) {
          if (!sel[b]) continue;
          for (int64_t j = b * Bn; j < (b + 1) * Bn && j <= i; ++j) {
            const uint16_t* kk = K + (g * N + j) * d;
            double dot = 0.0;
            for (int64_t c = 0; c < d; ++c) dot += (double)bf16f(q[c]) * (double)bf16f(kk[c]);
            logit[j] = dot * scale;
            if (logit[j] > mx) mx = logit[j];
          }
        }
        double den = 0.0;
        for (int64_t c = 0; c < d; ++c) acc[c] = 0.0;
        for (int64_t b = 0; b <= t; ++b) {
          if (!sel[b]) continue;
          for (int64_t j = b * Bn; j < (b + 1) * Bn && j <= i; ++j) {
            double p = exp(logit[j] - mx);
            den += p;
            const uint16_t* vv = V + (g * N + j) * d;
            for (int64_t c = 0; c < d; ++c) acc[c] += p * (double)bf16f(vv[c]);
          }
        }
        float* o = O + (ip * Bn + r) * d;
        if (den > 0.0) {
          for (int64_t c = 0; c < d; ++c) o[c] = (float)(acc[c] / den);
          if (lse) lse[ip * Bn + r] = (float)(mx + log(den));
        } else {                        /* nothing attended (cannot happen with forced self block) */
          for (int64_t c = 0; c < d; ++c) o[c] = 0.0f;
          if (lse) lse[ip * Bn + r] = -INFINITY;
        }
      }
    }
    free(sel); free(logit); free(acc);
  }
}

/* ---------------------------------------------------------------------------------------------
 * D.4 diagnostics (App. D.4; definitions Eq.18; (A1)/(A2) L431-432;
 * Remark 1 L480; Proposition 1; measured-quantities paragraph L493-501).  SURVEY 8(f).3.
 *
 * Per cell (tile t, head h), from the sorted list s~ of Eq.10 (score_sorted[0..2k], forced blocks on
 * top as +inf, f of them; reading G1 puts the best NON-forced score in the place of s_(0)):
 *     g = s~[k-1] - s~[k]      G = s~[k-1] - s~[rho k]      r = s~[f] - s~[k]      (fp32 subtractions)
 *     d2 = min_{j = f .. rho k - 1, j != k-1} (s~[j] - s~[j+1])     secondary spacing (A1), on the
 *          ranks the selection keeps on chip
 * defined for cells with at least rho*k + 1 visible blocks (L493); NaN elsewhere.
 *   score_sorted [n_tiles, H, 2k+1];  g, G, r, d2 [n_tiles, H]
 * ------------------------------------------------------------------------------------------- */
void orc_diag_cells(const float* score_sorted, const int64_t* tiles, int64_t n_tiles, int64_t H,
                    int64_t k, float* g, float* G, float* r, float* d2) {
  int64_t W2 = RHO * k;
  for (int64_t it = 0; it < n_tiles; ++it)
    for (int64_t h = 0; h < H; ++h) {
      int64_t t = tiles[it], o = it * H + h;
      const float* ss = score_sorted + o * (W2 + 1);
      if (t + 1 < W2 + 1) { g[o] = G[o] = r[o] = d2[o] = NAN; continue; }
      int64_t f = (t == 0) ? 1 : 2;
      g[o] = ss[k - 1] - ss[k];
      G[o] = ss[k - 1] - ss[W2];
      r[o] = ss[f] - ss[k];
      float mn = INFINITY;
      for (int64_t j = f; j < W2; ++j) {
        if (j == k - 1) continue;
        float sp = ss[j] - ss[j + 1];
        if (sp < mn) mn = sp;
      }
      d2[o] = mn;
    }
}

/* Step 3 of the recipe (L489): row-to-row roughness of the per-row block scores,
 *     rough[t,h] = sum_{b <= t} sum_{i = 0}^{Bn-2} (s[tBn+i+1, h, b] - s[tBn+i, h, b])^2
 * with s the fp32 row scores of O3 / O3q; pairs of adjacent rows inside one tile only (reading G19).
 * Accumulated in double, rounded once.   rough [n_tiles, H] */
void orc_roughness(const uint16_t* Q, const float* kmean, const uint16_t* kmin, const uint16_t* kmax,
                   int64_t H, int64_t Hkv, int64_t N, int64_t d, int64_t Bn, int policy,
                   const int64_t* tiles, int64_t n_tiles, float* rough) {
  int64_t NB = N / Bn, G = H / Hkv;
  int quest = (policy == POLICY_QUEST || policy == POLICY_ROUTER_QUEST);
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
  for (int64_t it = 0; it < n_tiles; ++it)
    for (int64_t h = 0; h < H; ++h) {
      int64_t t = tiles[it], g = h / G;
      double acc = 0.0;
      for (int64_t b = 0; b <= t; ++b) {
        int64_t o = (g * NB + b) * d;
        float prev = 0.0f;
        for (int64_t i = 0; i < Bn; ++i) {
          const uint16_t* q = Q + (h * N + t * Bn + i) * d;
          float s = quest ? row_score_quest(q, kmin + o, kmax + o, d) : row_score_mean(q, kmean + o, d);
          if (i > 0) { double df = (double)s - (double)prev; acc += df * df; }
          prev = s;
        }
      }
      rough[it * H + h] = (float)acc;
    }
}

/* Per-layer aggregates over the valid cells (t >= rho k), see include/bsa.h for the index list:
 *  0 n | 1 r_bar | 2 CV(r) (population variance, A2) | 3 sigma_(q) = tau | 4 gamma_q = sigma_(q) r_bar |
 *  5 band mass m_q(beta), beta = CV(r) (Remark 1) | 6, 7 10 % / 50 % order statistics of d2 |
 *  8 tau_hat = sqrt(sum rough / (2 #pairs)) over ALL cells, #pairs = H T(T+1)/2 (Bn-1) |
 *  9 fraction g == 0 | 10 g_q^+ = 40th percentile of g on {g > 0} (L501) | 11 g_q^+ / tau_hat
 * Order statistic: the ceil(p n - 1e-9)-th smallest (as reading G3).
 * Inputs laid out [T, H] (all tiles of one sequence). */
void orc_diag_summary(const float* g, const float* r, const float* d2, const float* rough, int64_t T,
                      int64_t H, int64_t k, int64_t Bn, int router, float tau, float* out /* [16] */) {
  int64_t t_min = RHO * k;
  int64_t n = (T > t_min) ? H * (T - t_min) : 0;
  for (int i = 0; i < 16; ++i) out[i] = (i < 12) ? NAN : 0.0f;
  double rs = 0.0;
  for (int64_t i = 0; i < T * H; ++i) rs += (double)rough[i];
  double pairs = (double)H * ((double)T * (double)(T + 1) / 2.0) * (double)(Bn - 1);
  double tau_hat = sqrt(rs / (2.0 * pairs));
  out[0] = (float)n;
  out[8] = (float)tau_hat;
  if (n == 0) return;
  double sum = 0.0;
  for (int64_t t = t_min; t < T; ++t) for (int64_t h = 0; h < H; ++h) sum += (double)r[t * H + h];
  double r_bar = sum / (double)n, var = 0.0;
  for (int64_t t = t_min; t < T; ++t) for (int64_t h = 0; h < H; ++h) {
    double dv = (double)r[t * H + h] - r_bar; var += dv * dv;
  }
  var /= (double)n;
  double cv = sqrt(var) / r_bar;
  out[1] = (float)r_bar; out[2] = (float)cv;
  float* gv = (float*)malloc(sizeof(float) * (size_t)n);
  float* dv2 = (float*)malloc(sizeof(float) * (size_t)n);
  int64_t c = 0, npos = 0, nzero = 0, band = 0;
  double gamma = (double)tau * r_bar, lo = gamma * (1.0 - cv), hi = gamma * (1.0 + cv);
  for (int64_t t = t_min; t < T; ++t) for (int64_t h = 0; h < H; ++h) {
    float x = g[t * H + h];
    dv2[c++] = d2[t * H + h];
    if (x == 0.0f) ++nzero;
    if (x > 0.0f) gv[npos++] = x;
    if (router && (double)x >= lo && (double)x <= hi) ++band;
  }
  if (router) { out[3] = tau; out[4] = (float)gamma; out[5] = (float)((double)band / (double)n); }
  qsort(dv2, (size_t)n, sizeof(float), float_cmp);
  int64_t m10 = (int64_t)ceil(0.10 * (double)n - 1e-9), m50 = (int64_t)ceil(0.50 * (double)n - 1e-9);
  if (m10 < 1) m10 = 1;
  if (m50 < 1) m50 = 1;
  out[6] = dv2[m10 - 1]; out[7] = dv2[m50 - 1];
  out[9] = (float)((double)nzero / (double)n);
  if (npos > 0) {
    qsort(gv, (size_t)npos, sizeof(float), float_cmp);
    int64_t m40 = (int64_t)ceil(0.40 * (double)npos - 1e-9);
    if (m40 < 1) m40 = 1;
    out[10] = gv[m40 - 1];
    out[11] = (float)((double)gv[m40 - 1] / tau_hat);
  }
  free(gv); free(dv2);
}

/* ---------------------------------------------------------------------------------------------
 * Per-row selection scattered into a per-tile block bitmap (section 4.5 item 1: "A
 * per-row scatter-into-bitmap kernel would close the rest of the gap without re-materialising the
 * [B, H, M, N_B] keep tensor; not yet built").  SURVEY 8(f).4; reading G18:
 *   every query row i of tile t ranks the visible blocks by ITS OWN row score s[i,h,b] (O3 / O3q; no
 *   tile max), blocks 0 and t forced on top (Eq.9), ties -> lower block index (G6), and keeps its first
 *   min(k_row, t+1) blocks; the tile's bitmap is the union over its Bn rows and the whole tile attends
 *   the union (one bit per (tile, head, block) instead of one per (row, head, block)).
 *   bitmap [n_tiles, H, NBW] uint32, NBW = ceil(N_B / 32), bit b%32 of word b/32;  count [n_tiles, H]
 * ------------------------------------------------------------------------------------------- */
void orc_select_rows_bitmap(const uint16_t* Q, const float* kmean, const uint16_t* kmin,
                            const uint16_t* kmax, int64_t H, int64_t Hkv, int64_t N, int64_t d,
                            int64_t Bn, int policy, int64_t k_row, const int64_t* tiles, int64_t n_tiles,
                            uint32_t* bitmap, int32_t* count) {
  int64_t NB = N / Bn, NBW = (NB + 31) / 32, G = H / Hkv;
  int quest = (policy == POLICY_QUEST || policy == POLICY_ROUTER_QUEST);
#pragma omp parallel
  {
    cand_t* scratch = (cand_t*)malloc(sizeof(cand_t) * (size_t)NB);
#pragma omp for collapse(2) schedule(dynamic, 1)
    for (int64_t it = 0; it < n_tiles; ++it)
      for (int64_t h = 0; h < H; ++h) {
        int64_t t = tiles[it], g = h / G;
        uint32_t* bm = bitmap + (it * H + h) * NBW;
        for (int64_t w = 0; w < NBW; ++w) bm[w] = 0;
        int64_t f = (t == 0) ? 1 : 2, nf = t + 1 - f;
        bm[0] |= 1u;                                       /* sink */
        bm[t >> 5] |= 1u << (t & 31);                      /* self */
        int64_t keep = k_row - f;
        if (keep > nf) keep = nf;
        for (int64_t r = 0; r < Bn && keep > 0; ++r) {
          const uint16_t* q = Q + (h * N + t * Bn + r) * d;
          for (int64_t i = 0; i < nf; ++i) {
            int64_t b = i + 1, o = (g * NB + b) * d;
            scratch[i].s = quest ? row_score_quest(q, kmin + o, kmax + o, d) : row_score_mean(q, kmean + o, d);
            scratch[i].b = (int32_t)b;
          }
          qsort(scratch, (size_t)nf, sizeof(cand_t), cand_cmp);
          for (int64_t i = 0; i < keep; ++i) bm[scratch[i].b >> 5] |= 1u << (scratch[i].b & 31);
        }
        int32_t c = 0;
        for (int64_t w = 0; w < NBW; ++w) c += __builtin_popcount(bm[w]);
        count[it * H + h] = c;
      }
    free(scratch);
  }
}

int orc_max_threads(void) {
#ifdef _OPENMP
  extern int omp_get_max_threads(void);
  return omp_get_max_threads();
#else
  return 1;
#endif
}

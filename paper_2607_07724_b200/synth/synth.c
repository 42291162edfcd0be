/*
 * synth.c -- seeded synthetic input generator.
 *
 * This file holds NO arithmetic of the method (no pooling, scoring, selection,
 * softmax).  It only draws counter-based Gaussian tensors and applies the
 * pre-processing the recipe lists (block mean offsets, per-row RMSNorm for the
 * QK-Norm config).  Both the CPU oracle's tests and the CUDA path's tests read
 * their inputs from here, so the two sides see the same bf16 bit patterns.
 *
 * RNG (counter based, order independent):
 *   key = splitmix64(seed ^ (tensor_id * 0x9E3779B97F4A7C15))
 *   r   = splitmix64(key + flat_index)
 *   u1  = ((r >> 32) + 1) / 2^32,  u2 = (r & 0xffffffff) / 2^32
 *   z   = sqrt(-2 ln u1) * cos(2 pi u2)          (double)
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

static inline uint64_t splitmix64(uint64_t x) {
  x += 0x9E3779B97F4A7C15ULL;
  x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ULL;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBULL;
  return x ^ (x >> 31);
}

static inline uint64_t tensor_key(uint64_t seed, uint64_t tensor_id) {
  return splitmix64(seed ^ (tensor_id * 0x9E3779B97F4A7C15ULL));
}

static inline double gauss_at(uint64_t key, uint64_t idx) {
  uint64_t r = splitmix64(key + idx);
  double u1 = ((double)(r >> 32) + 1.0) / 4294967296.0;
  double u2 = (double)(r & 0xffffffffULL) / 4294967296.0;
  return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
}

static inline uint16_t f32_to_bf16_rne(float f) {
  union { float f; uint32_t u; } v; v.f = f;
  uint32_t u = v.u;
  if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x40); /* NaN */
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

static inline float bf16_to_f32(uint16_t h) {
  union { float f; uint32_t u; } v; v.u = ((uint32_t)h) << 16; return v.f;
}

/* Raw 64-bit draws (for needle positions etc.). */
void synth_u64(uint64_t seed, uint64_t tensor_id, uint64_t start, uint64_t n, uint64_t* out) {
  uint64_t key = tensor_key(seed, tensor_id);
  for (uint64_t i = 0; i < n; ++i) out[i] = splitmix64(key + start + i);
}

/* Gaussian draws as double (small tensors: offsets, needle directions). */
void synth_gauss_f64(uint64_t seed, uint64_t tensor_id, uint64_t start, uint64_t n, double* out) {
  uint64_t key = tensor_key(seed, tensor_id);
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < (int64_t)n; ++i) out[i] = gauss_at(key, start + (uint64_t)i);
}

/*
 * out[h, n, c] (bf16 bits, contiguous [heads, rows, d]) =
 *     bf16( (float)( z[h,n,c] + off_scale * zoff[h, n / block, c] ) )
 * off_tensor_id == 0 means "no offsets".
 */
void synth_gauss_bf16(uint64_t seed, uint64_t tensor_id, uint64_t off_tensor_id, double off_scale,
                      int64_t heads, int64_t rows, int64_t d, int64_t block, uint16_t* out) {
  uint64_t key = tensor_key(seed, tensor_id);
  uint64_t okey = tensor_key(seed, off_tensor_id);
  int64_t nblk = rows / block;
#pragma omp parallel for schedule(static) collapse(2)
  for (int64_t h = 0; h < heads; ++h) {
    for (int64_t n = 0; n < rows; ++n) {
      uint64_t base = (uint64_t)((h * rows + n) * d);
      uint64_t obase = (uint64_t)((h * nblk + n / block) * d);
      for (int64_t c = 0; c < d; ++c) {
        double z = gauss_at(key, base + (uint64_t)c);
        if (off_tensor_id) z += off_scale * gauss_at(okey, obase + (uint64_t)c);
        out[base + (uint64_t)c] = f32_to_bf16_rne((float)z);
      }
    }
  }
}

/* In-place per-row RMSNorm (unit gain) on bf16 rows of length d: fp32 arithmetic, bf16 result. */
void synth_rmsnorm_rows_bf16(uint16_t* x, int64_t n_rows, int64_t d, float eps) {
#pragma omp parallel for schedule(static)
  for (int64_t r = 0; r < n_rows; ++r) {
    uint16_t* row = x + r * d;
    float ss = 0.f;
    for (int64_t c = 0; c < d; ++c) { float v = bf16_to_f32(row[c]); ss += v * v; }
    float inv = 1.0f / sqrtf(ss / (float)d + eps);
    for (int64_t c = 0; c < d; ++c) row[c] = f32_to_bf16_rne(bf16_to_f32(row[c]) * inv);
  }
}

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
// One CTA per (tile, head), two CTAs per SM, 7 warps: 0-3 softmax (thread = key), 4 TMA producer,
// 5 QK issue (runs one iteration ahead, S^T double buffered), 6 PV issue.  K and V have separate rings
// of 16 KB units, each with a single in-order consumer (see attn.cu on why): a K unit is one 64-column
// slab of BOTH blocks (rows 0-63 = block a, 64-127 = block b, the M = 128 A operand needs them adjacent),
// a V unit is one block.
#include <cuda_bf16.h>

#include "bsa_internal.h"
#include "sm100_ptx.cuh"
#include "tmap.h"

namespace bsa {

namespace {

constexpr int TD = 128;                 // head_dim
constexpr int TB = 64;                  // block = Q tile rows
constexpr int kTThreads = 224;
constexpr int kTMaxW = 256;
constexpr int UNIT = 16384;             // ring unit
constexpr int NKU = 3, NVU = 2;         // K / V ring units
constexpr int T_Q_BYTES = TB * TD * 2;  // 16 KB
constexpr int T_P_BYTES = 128 * TB * 2; // P^T [128 keys][64 queries] bf16 = 16 KB
constexpr int T_SMEM = T_Q_BYTES + T_P_BYTES + (NKU + NVU) * UNIT + 1024;
static_assert(T_SMEM <= 115712, "two CTAs per SM");
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
  uint64_t q_full, p_full, o_done;
  uint64_t s_full[2], s_free[2];
  uint64_t k_full[NKU], k_empty[NKU], v_full[NVU], v_empty[NVU];
  uint32_t tmem_base;
  int32_t n_valid;
  uint16_t list[kTMaxW];
};
static_assert(sizeof(TCtl) <= 1024, "TCtl must fit the 1 KB bookkeeping area");
// Scratch of the slow path inside the P^T buffer (free between PV(j-1) and the P^T(j) store):
//   float wmax[4][64] at byte 0 (per-warp column maxima), float alpha[64] at byte 1024

__device__ __forceinline__ void bar_sm() { asm volatile("bar.sync 1, 128;" ::: "memory"); }
__device__ __forceinline__ bool bar_or(bool pred) {   // barrier 2 over the 128 softmax threads + OR
  uint32_t r;
  asm volatile(
      "{\n\t.reg .pred p, q;\n\tsetp.ne.b32 p, %1, 0;\n\t"
      "barrier.cta.red.or.pred q, 2, 128, p;\n\tselp.u32 %0, 1, 0, q;\n\t}"
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

}  // namespace

}  // namespace bsa

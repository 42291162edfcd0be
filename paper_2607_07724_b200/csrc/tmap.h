// tmap.h -- host helper: TMA tensor maps through cuTensorMapEncodeTiled, fetched with
// cudaGetDriverEntryPoint so libbsa does not link libcuda directly.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace bsa {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn tmap_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

// bf16 tensor of `rank` dims (dims[0] contiguous, strides_bytes[i] = stride of dim i+1), 128-byte
// swizzle (box[0] must be 64 elements), out-of-bounds elements read as zero.
inline bool make_tmap_bf16(CUtensorMap* m, const void* base, int rank, const cuuint64_t* dims,
                           const cuuint64_t* strides_bytes, const cuuint32_t* box) {
  EncodeTiledFn fn = tmap_encode_fn();
  if (!fn) return false;
  cuuint32_t es[5] = {1, 1, 1, 1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, static_cast<cuuint32_t>(rank),
                  const_cast<void*>(base), dims, strides_bytes, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

// bf16 tensor [B, heads, N, d] (strides in elements) viewed as 5-D (64, N, d/64, heads, B) so one
// TMA instruction lands a [rows x d] tile as d/64 consecutive 128B-swizzled [rows x 64] chunks
// (box_chunks = d/64, box_heads = 1), or one [heads x rows x 64] slab of a single 64-column chunk
// (box_chunks = 1, box_heads > 1).
inline bool make_tmap_bhnd(CUtensorMap* m, const void* base, int B, int heads, int N, int d, int64_t sb,
                           int64_t sh, int64_t sn, int box_rows, int box_chunks, int box_heads) {
  cuuint64_t dims[5] = {64, static_cast<cuuint64_t>(N), static_cast<cuuint64_t>(d / 64),
                        static_cast<cuuint64_t>(heads), static_cast<cuuint64_t>(B)};
  cuuint64_t strides[4] = {static_cast<cuuint64_t>(sn) * 2, 128, static_cast<cuuint64_t>(sh) * 2,
                           static_cast<cuuint64_t>(sb) * 2};
  if (heads == 1) strides[2] = strides[0] * static_cast<cuuint64_t>(N);
  if (B == 1) strides[3] = strides[2] * static_cast<cuuint64_t>(heads);
  cuuint32_t box[5] = {64, static_cast<cuuint32_t>(box_rows), static_cast<cuuint32_t>(box_chunks),
                       static_cast<cuuint32_t>(box_heads), 1};
  return make_tmap_bf16(m, base, 5, dims, strides, box);
}

}  // namespace bsa

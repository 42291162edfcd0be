// bsa_internal.h -- host-side declarations shared by the translation units of libbsa.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/bsa.h"

namespace bsa {

// Validated problem dimensions (derived from bsa_shape).
struct Dims {
  int B, N, H, Hkv, d, Bn, NB, G;
  int64_t qsb, qsh, qsn;  // Q / O strides in elements
  int64_t ksb, ksh, ksn;  // K / V strides in elements
};

bsa_status fail(bsa_status code, const char* fmt, ...);
bsa_status check_launch(const char* what);
int sm_count();  // SMs of the current device (cached per device; 148 on B200)

// meta plane offsets in bytes (see include/bsa.h); the three bf16 split planes of kmean
// (hi, mid, lo; hi+mid+lo == kmean exactly) follow kmax and feed the tensor-core scoring.
struct MetaLayout {
  size_t elems;      // B*Hkv*NB*d
  size_t off_mean;   // fp32
  size_t off_min;    // bf16
  size_t off_max;    // bf16
  size_t off_split;  // bf16 x 3 planes
  size_t bytes;
};
MetaLayout meta_layout(const Dims& D);

// kernels (each only enqueues on `stream`)
bsa_status launch_pool(const Dims& D, const void* K, int kinds, void* meta, cudaStream_t stream);
// D.4 diagnostics outputs of the selection (device pointers, each [B,H,T]; all nullptr = off) and the
// per-sequence summary [B, BSA_DIAG_SUMMARY_LEN] (may be nullptr).
struct SelectDiag {
  float *g, *G, *r, *d2, *rough, *summary;
};
bsa_status launch_select(const Dims& D, const void* Q, const void* meta, int policy, int k, int W,
                         long long m_route, int32_t* kv_idx, int32_t* kv_count, float* sigma,
                         float* sigma_bar, uint8_t* trigger, float* tau, const SelectDiag& dg,
                         cudaStream_t stream);
// tensor-core scoring + tile max + top-(2k) + sigma (score_tc.cuh); writes kv_idx (all 2k/k slots),
// sigma and, for the non-router policies, kv_count.  One translation unit per backbone.
bsa_status launch_score_tc_quest(const Dims& D, const void* Q, const void* meta, int k, int W, int router,
                                 int32_t* kv_idx, int32_t* kv_count, float* sigma, const SelectDiag& dg,
                                 cudaStream_t stream);
bsa_status launch_score_tc_mean(const Dims& D, const void* Q, const void* meta, int k, int W, int router,
                                int32_t* kv_idx, int32_t* kv_count, float* sigma, const SelectDiag& dg,
                                cudaStream_t stream);
// per-sequence reduction of the D.4 per-cell quantities (diag.cu)
bsa_status launch_diag_summary(const Dims& D, int k, int router, const float* tau, const SelectDiag& dg,
                               cudaStream_t stream);
// per-row selection scattered into a per-tile bitmap (rowsel.cu)
bsa_status launch_rowsel(const Dims& D, const void* Q, const void* meta, bool quest, int k_row,
                         uint32_t* bitmap, int32_t* count, cudaStream_t stream);
bsa_status launch_attn(const Dims& D, const void* Q, const void* K, const void* V,
                       const int32_t* kv_idx, const int32_t* kv_count, int W, bool sparse,
                       float scale, void* O, float* lse, cudaStream_t stream,
                       const uint32_t* bitmap = nullptr, bool pdl = false);

// transposed sparse attention for block 64 / head_dim 128 (attn_t.cu)
bool attn_t_supported(const Dims& D, int W);
bsa_status launch_attn_t(const Dims& D, const void* Q, const void* K, const void* V, const int32_t* kv_idx,
                         const int32_t* kv_count, int W, float scale, void* O, float* lse,
                         cudaStream_t stream);

}  // namespace bsa

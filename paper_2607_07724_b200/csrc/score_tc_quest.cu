// score_tc_quest.cu -- the Quest (K-min / K-max, Eq.2) instantiations of score_tc.cuh.
#include "score_tc.cuh"

namespace bsa {

bsa_status launch_score_tc_quest(const Dims& S, const void* Q, const void* meta, int k, int W, int router,
                                 int32_t* kv_idx, int32_t* kv_count, float* sigma, const SelectDiag& dg,
                                 cudaStream_t stream) {
  const DiagPtrs d = {dg.g, dg.G, dg.r, dg.d2, dg.rough};
  return launch_score_tc_backbone<true>(S, Q, meta, k, W, router, kv_idx, kv_count, sigma, d, stream);
}

}  // namespace bsa

// gemm_tc.cuh - tcgen05 (3xTF32) batched GEMM for the large-block rebuild and Dalecki-Krein products.
// Placeholder until the tensor-core kernel lands: reports "unsupported" so the FMA GEMM is used.
#pragma once
#include <string>
#include "cdu.h"
namespace cdu {
inline bool gemm_tc_supported(int) { return false; }
inline cdu_status gemm_tc_batched(int, const int*, const int*, const long long*, const int*, const float*, int, const float*,
                                  int, float*, const float*, int, float*, cudaStream_t, long long*, std::string& err) {
  err = "tcgen05 GEMM not built";
  return CDU_EINVAL;
}
}  // namespace cdu

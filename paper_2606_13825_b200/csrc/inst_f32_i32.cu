// inst_f32_i32.cu - kernels and host driver for value type float, index type int (see handle.cuh).
#include "handle.cuh"

namespace cdu {
cdu_status create_f32_i32(const cdu_problem* pr, const cdu_options* op, cudaStream_t st, cdu_handle* out) {
  return impl::create_t<float, int>(pr, op, st, out);
}
}  // namespace cdu

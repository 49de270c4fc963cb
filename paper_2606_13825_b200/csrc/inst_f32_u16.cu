// inst_f32_u16.cu - kernels and host driver for value type float, index type uint16_t (see handle.cuh).
#include "handle.cuh"

namespace cdu {
cdu_status create_f32_u16(const cdu_problem* pr, const cdu_options* op, cudaStream_t st, cdu_handle* out) {
  return impl::create_t<float, uint16_t>(pr, op, st, out);
}
cdu_status psd_op_f32(bool vjp, int count, int p, const void* in1, const void* in2, const void* in3, void* out1, void* out2,
                      void* out3, int path, int use_tc, cudaStream_t st) {
  return impl::psd_op_t<float>(vjp, count, p, in1, in2, in3, out1, out2, out3, path, use_tc, st);
}
}  // namespace cdu

// cdu_api.cu - the C ABI of include/cdu.h. Argument checks, the device guard and dispatch to the per-dtype translation
// units (inst_*.cu, which hold every kernel of the hot path); the peak micro-benchmarks of peaks.cuh live here too.
// No CPU fallback exists: without a CUDA device every entry point that computes returns CDU_ECUDA.
#include <cuda_runtime.h>

#include <string>

#include "cdu.h"
#include "handle_base.h"
#include "peaks.cuh"

namespace cdu {
std::string& create_error() {
  static thread_local std::string e;
  return e;
}
}  // namespace cdu

namespace {
// Makes the handle's device current for the duration of an entry point (the caller may have switched devices).
struct DeviceGuard {
  int prev = -1; bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};
}  // namespace

extern "C" {

cdu_status cdu_create(const cdu_problem* prob, const cdu_options* opts, void* cuda_stream, cdu_handle* out) {
  std::string& cerr = cdu::create_error();
  if (!prob || !out) { cerr = "cdu_create: NULL argument"; return CDU_EINVAL; }
  *out = nullptr;
  int ndev = 0, dev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1 || cudaGetDevice(&dev) != cudaSuccess) {
    (void)cudaGetLastError();
    cerr = "cdu_create: no CUDA device (there is no CPU fallback)"; return CDU_ECUDA;
  }
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  bool narrow = prob->batch >= 1 && prob->var_off && prob->row_off;      // 16-bit local indices suffice
  for (int b = 0; narrow && b < prob->batch; ++b)
    if (prob->var_off[b + 1] - prob->var_off[b] > 65535 || prob->row_off[b + 1] - prob->row_off[b] > 65535) narrow = false;
  cdu_status s;
  if (prob->dtype == CDU_F32) s = narrow ? cdu::create_f32_u16(prob, opts, st, out) : cdu::create_f32_i32(prob, opts, st, out);
  else if (prob->dtype == CDU_F64) s = narrow ? cdu::create_f64_u16(prob, opts, st, out) : cdu::create_f64_i32(prob, opts, st, out);
  else { cerr = "cdu_create: bad dtype"; return CDU_EINVAL; }
  if (s == CDU_OK) (*out)->device = dev;
  return s;
}

cdu_status cdu_forward(cdu_handle h, int32_t K, const void* rho, int32_t rho_mode, double sigma, const void* alpha,
                       const void* x0, const void* s0, const void* y0, void* xK, void* sK, void* yK, int32_t io_on_host,
                       void* cuda_stream) {
  if (!h) return CDU_EINVAL;
  DeviceGuard g(h->device);
  return h->forward(K, rho, rho_mode, sigma, alpha, x0, s0, y0, xK, sK, yK, io_on_host, reinterpret_cast<cudaStream_t>(cuda_stream));
}

cdu_status cdu_backward(cdu_handle h, const void* g_xK, const void* g_sK, const void* g_yK, void* g_rho, void* g_sigma,
                        void* g_alpha, void* g_x0, void* g_s0, void* g_y0, int32_t io_on_host, void* cuda_stream) {
  if (!h) return CDU_EINVAL;
  DeviceGuard g(h->device);
  return h->backward(g_xK, g_sK, g_yK, g_rho, g_sigma, g_alpha, g_x0, g_s0, g_y0, io_on_host, reinterpret_cast<cudaStream_t>(cuda_stream));
}

cdu_status cdu_backward_inject(cdu_handle h, const void* g_xK, const void* g_sK, const void* g_yK, const void* inj_x,
                               const void* inj_s, const void* inj_y, void* g_rho, void* g_sigma, void* g_alpha, void* g_x0,
                               void* g_s0, void* g_y0, int32_t io_on_host, void* cuda_stream) {
  if (!h) return CDU_EINVAL;
  DeviceGuard g(h->device);
  cdu_handle_s::Extra ex; ex.ix = inj_x; ex.is = inj_s; ex.iy = inj_y;
  return h->backward(g_xK, g_sK, g_yK, g_rho, g_sigma, g_alpha, g_x0, g_s0, g_y0, io_on_host, reinterpret_cast<cudaStream_t>(cuda_stream), &ex);
}

cdu_status cdu_backward_eq12(cdu_handle h, void* loss, void* g_rho, void* g_sigma, void* g_alpha, void* g_x0, void* g_s0,
                             void* g_y0, int32_t io_on_host, void* cuda_stream) {
  if (!h) return CDU_EINVAL;
  DeviceGuard g(h->device);
  cdu_handle_s::Extra ex; ex.eq12 = 1; ex.loss = loss;
  return h->backward(nullptr, nullptr, nullptr, g_rho, g_sigma, g_alpha, g_x0, g_s0, g_y0, io_on_host, reinterpret_cast<cudaStream_t>(cuda_stream), &ex);
}

cdu_status cdu_get_features(cdu_handle h, int32_t k, void* rp_bar, void* rd_bar, void* delta_p, void* delta_d, void* scal,
                            int32_t io_on_host, void* cuda_stream) {
  if (!h) return CDU_EINVAL;
  DeviceGuard g(h->device);
  return h->features(k, rp_bar, rd_bar, delta_p, delta_d, scal, io_on_host, reinterpret_cast<cudaStream_t>(cuda_stream));
}

cdu_status cdu_solve(cdu_handle h, int32_t max_iter, int32_t check_every, double eps, double rho0, double alpha, double sigma,
                     int32_t adapt_rho, double eq_scale, const void* x0, const void* s0, const void* y0, void* x, void* s, void* y, int32_t* iters_out,
                     double* res_out, int32_t io_on_host, void* cuda_stream) {
  if (!h) return CDU_EINVAL;
  DeviceGuard g(h->device);
  return h->solve(max_iter, check_every, eps, rho0, alpha, sigma, adapt_rho, eq_scale, x0, s0, y0, x, s, y, iters_out, res_out, io_on_host,
                  reinterpret_cast<cudaStream_t>(cuda_stream));
}

cdu_status cdu_rectify_rho(cdu_handle h, int32_t K, void* rho, int32_t io_on_host, void* cuda_stream) {
  if (!h) return CDU_EINVAL;
  DeviceGuard g(h->device);
  return h->rectify(K, rho, io_on_host, reinterpret_cast<cudaStream_t>(cuda_stream));
}

cdu_status cdu_get_stats(cdu_handle h, cdu_stats* out) {
  if (!h) return CDU_EINVAL;
  DeviceGuard g(h->device);
  return h->stats(out);
}

cdu_status cdu_get_iterate(cdu_handle h, int32_t k, void* x, void* s, void* y, int32_t io_on_host, void* cuda_stream) {
  if (!h) return CDU_EINVAL;
  DeviceGuard g(h->device);
  return h->iterate(k, x, s, y, io_on_host, reinterpret_cast<cudaStream_t>(cuda_stream));
}

const char* cdu_last_error(cdu_handle h) { return h ? h->err.c_str() : cdu::create_error().c_str(); }

cdu_status cdu_destroy(cdu_handle h) {
  if (!h) return CDU_EINVAL;
  DeviceGuard g(h->device);
  cudaStreamSynchronize(h->stream_of_last_call());   // only the stream this handle's work was ordered on
  delete h;
  return CDU_OK;
}

const char* cdu_version(void) { return "cdu 0.2 (sm_100a)"; }

cdu_status cdu_profile(cdu_handle h, int32_t enable) {
  if (!h) return CDU_EINVAL;
  h->profile_enable(enable);
  return CDU_OK;
}

cdu_status cdu_get_profile(cdu_handle h, int32_t nclass, double* ms, int64_t* count) {
  if (!h || !ms || !count || nclass < 1) return CDU_EINVAL;
  DeviceGuard g(h->device);
  double m[cdu::PROFILE_CLASSES]; long long c[cdu::PROFILE_CLASSES];
  h->profile_collect(m, c);
  for (int i = 0; i < nclass; ++i) { ms[i] = i < cdu::PROFILE_CLASSES ? m[i] : 0.0; count[i] = i < cdu::PROFILE_CLASSES ? c[i] : 0; }
  return CDU_OK;
}

cdu_status cdu_psd_project(int32_t dtype, int32_t count, int32_t p, const void* S, void* PiS, void* U, void* lam,
                           int32_t path, int32_t use_tensor_cores, void* cuda_stream) {
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  if (dtype == CDU_F32) return cdu::psd_op_f32(false, count, p, S, nullptr, nullptr, PiS, U, lam, path, use_tensor_cores, st);
  if (dtype == CDU_F64) return cdu::psd_op_f64(false, count, p, S, nullptr, nullptr, PiS, U, lam, path, use_tensor_cores, st);
  return CDU_EINVAL;
}

cdu_status cdu_psd_vjp(int32_t dtype, int32_t count, int32_t p, const void* U, const void* lam, const void* Gbar,
                       void* Sbar, int32_t path, int32_t use_tensor_cores, void* cuda_stream) {
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  if (dtype == CDU_F32) return cdu::psd_op_f32(true, count, p, U, lam, Gbar, Sbar, nullptr, nullptr, path, use_tensor_cores, st);
  if (dtype == CDU_F64) return cdu::psd_op_f64(true, count, p, U, lam, Gbar, Sbar, nullptr, nullptr, path, use_tensor_cores, st);
  return CDU_EINVAL;
}

cdu_status cdu_measure_peak(int32_t kind, double* value, void* cuda_stream) {
  if (!value) return CDU_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { (void)cudaGetLastError(); return CDU_ECUDA; }
  return cdu::peaks::measure(kind, value, reinterpret_cast<cudaStream_t>(cuda_stream));
}

}  // extern "C"

// handle_base.h - the abstract handle behind cdu_handle and the per-dtype factory functions (one translation unit per
// (value type, index type) pair so that the kernels compile in parallel).
#pragma once
#include <cuda_runtime.h>
#include <string>
#include "cdu.h"

struct cdu_handle_s {
  std::string err;
  int device = 0;              // CUDA device the handle was created on; every entry point switches to it
  virtual ~cdu_handle_s() {}
  virtual cdu_status forward(int K, const void* rho, int mode, double sigma, const void* alpha, const void* x0,
                             const void* s0, const void* y0, void* xK, void* sK, void* yK, int host, cudaStream_t st) = 0;
  struct Extra {             // cotangents on the intermediate iterates (cdu_backward_inject / cdu_backward_eq12)
    const void *ix = nullptr, *is = nullptr, *iy = nullptr;   // [K-1][.]: row k-1 is added to the cotangent of z^k
    int eq12 = 0;            // add dL/dz^k of PAPER.md Eq. 12 for k = 1..K
    void* loss = nullptr;    // eq12: [B] loss values out
  };
  virtual cdu_status backward(const void* gx, const void* gs, const void* gy, void* g_rho, void* g_sigma, void* g_alpha,
                              void* g_x0, void* g_s0, void* g_y0, int host, cudaStream_t st, const Extra* ex = nullptr) = 0;
  virtual cdu_status solve(int max_iter, int check_every, double eps, double rho0, double alpha, double sigma, int adapt_rho,
                           double eq_scale, const void* x0, const void* s0, const void* y0, void* x, void* s, void* y, int* iters_out, double* res_out,
                           int host, cudaStream_t st) = 0;
  virtual cdu_status rectify(int K, void* rho, int host, cudaStream_t st) = 0;
  virtual cdu_status features(int k, void* rp_bar, void* rd_bar, void* delta_p, void* delta_d, void* scal, int host, cudaStream_t st) = 0;
  virtual cdu_status stats(cdu_stats* out) = 0;
  virtual cdu_status iterate(int k, void* x, void* s, void* y, int host, cudaStream_t st) = 0;
  virtual void profile_enable(int on) = 0;
  virtual void profile_collect(double* ms, long long* cnt) = 0;
  virtual cudaStream_t stream_of_last_call() const = 0;
};

namespace cdu {
std::string& create_error();   // text of the last cdu_create / stand-alone operator failure on this thread
// factories, defined in inst_*.cu
cdu_status create_f32_u16(const cdu_problem*, const cdu_options*, cudaStream_t, cdu_handle*);
cdu_status create_f32_i32(const cdu_problem*, const cdu_options*, cudaStream_t, cdu_handle*);
cdu_status create_f64_u16(const cdu_problem*, const cdu_options*, cudaStream_t, cdu_handle*);
cdu_status create_f64_i32(const cdu_problem*, const cdu_options*, cudaStream_t, cdu_handle*);
cdu_status psd_op_f32(bool vjp, int count, int p, const void* in1, const void* in2, const void* in3, void* out1, void* out2,
                      void* out3, int path, int use_tc, cudaStream_t st);
cdu_status psd_op_f64(bool vjp, int count, int p, const void* in1, const void* in2, const void* in3, void* out1, void* out2,
                      void* out3, int path, int use_tc, cudaStream_t st);
constexpr int PROFILE_CLASSES = 8;
}  // namespace cdu

// common.cuh - device helpers shared by the cdu kernels (sm_100a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cdu {

enum : int { FLAG_CG_CAP = 1, FLAG_CG_CURV = 2, FLAG_EIG_CAP = 4, FLAG_NONFINITE = 8, FLAG_BAD_HYPER = 16 };
enum : int { KIND_ZERO = 0, KIND_NONNEG = 1, KIND_SOC = 2, KIND_PSD = 3 };

template <typename T> struct Eps;
template <> struct Eps<float>  { static __host__ __device__ constexpr float  v() { return 5.9604645e-8f; } };
template <> struct Eps<double> { static __host__ __device__ constexpr double v() { return 1.1102230246251565e-16; } };

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Deterministic block-wide sum of NV doubles; every thread returns with the totals in v[].
// sh must hold NV*32 doubles. Ends with a barrier, so sh (and anything written before) is safe to reuse.
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* sh) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int i = 0; i < NV; ++i) v[i] = warp_sum(v[i]);
  if (lane == 0) {
#pragma unroll
    for (int i = 0; i < NV; ++i) sh[i * 32 + wid] = v[i];
  }
  __syncthreads();
  if (wid == 0) {   // one warp folds the per-warp partials (fixed shuffle tree: deterministic) and publishes the totals
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      double t = lane < nw ? sh[i * 32 + lane] : 0.0;
      t = warp_sum(t);
      if (lane == 0) sh[i * 32] = t;
    }
  }
  __syncthreads();
#pragma unroll
  for (int i = 0; i < NV; ++i) v[i] = sh[i * 32];
  __syncthreads();
}

__device__ __forceinline__ int svec_idx(int i, int j) {  // i <= j
  return j * (j + 1) / 2 + i;
}

}  // namespace cdu

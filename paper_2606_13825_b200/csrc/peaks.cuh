// peaks.cuh - in-tree micro-benchmarks for the roofline denominators that MEASURED_PEAKS.json does not carry
// ("measure with the builder's own micro-benchmark"): plain-ALU FMA throughput in fp32 and fp64, and the
// dense TF32 rate of the tcgen05 tensor pipe (kind::tf32, M128 N256 K8, operands resident in shared memory, accumulators
// in TMEM - no loads in the loop, so this is the pipe's own ceiling for the 3xTF32 products of gemm_tc.cuh).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "gemm_tc.cuh"

namespace cdu {
namespace peaks {

template <typename T, int CH>
static __global__ void __launch_bounds__(1024) k_fma_peak(int iters, T* sink) {
  T a[CH];
  const T m = (T)0.999 + (T)1e-6 * (T)(threadIdx.x & 7), c = (T)1e-3;
#pragma unroll
  for (int i = 0; i < CH; ++i) a[i] = (T)(threadIdx.x + i) * (T)1e-4;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 8; ++u)
#pragma unroll
      for (int i = 0; i < CH; ++i) a[i] = a[i] * m + c;
  }
  T s = (T)0;
#pragma unroll
  for (int i = 0; i < CH; ++i) s += a[i];
  if (s == (T)-1.2345) sink[0] = s;   // never true: keeps the chains alive
}

// warp-level mma.sync m16n8k8 tf32 (the path of the blocked Jacobi's Gram / apply products): 8 independent accumulators
static __global__ void __launch_bounds__(512) k_mma_sync_peak(int iters, float* sink) {
  float acc[8][4] = {};
  const uint32_t a = 0x3f800000u + threadIdx.x, b = 0x3f000000u + threadIdx.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < 8; ++j)
      asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                   : "+f"(acc[j][0]), "+f"(acc[j][1]), "+f"(acc[j][2]), "+f"(acc[j][3]) : "r"(a), "r"(b), "r"(a), "r"(b), "r"(b), "r"(a));
  }
  float s = 0.f;
#pragma unroll
  for (int j = 0; j < 8; ++j) s += acc[j][0] + acc[j][1] + acc[j][2] + acc[j][3];
  if (s == -1.2345f) sink[0] = s;
}

constexpr int TF32_N = 256;
static __global__ void __launch_bounds__(128, 1) k_tf32_peak(int iters, float* sink) {
  extern __shared__ unsigned char smem_dyn[];
  const uint32_t raw = tc::smem_u32(smem_dyn);
  const uint32_t base = (raw + 1023u) & ~1023u;
  float* tiles = reinterpret_cast<float*>(smem_dyn + (base - raw));
  constexpr int A_BYTES = 128 * 32 * 4, B_BYTES = TF32_N * 32 * 4;
  __shared__ uint64_t bar;
  __shared__ uint32_t tmem_slot;
  for (int t = threadIdx.x; t < (A_BYTES + B_BYTES) / 4; t += blockDim.x) tiles[t] = 0.01f * (float)((t * 7 + 3) % 13) - 0.05f;
  if (threadIdx.x == 0) {
    tc::mbar_init(tc::smem_u32(&bar), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  if (threadIdx.x < 32) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tc::smem_u32(&tmem_slot)), "n"(512) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = tmem_slot;
  if (threadIdx.x == 0) {
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(TF32_N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    for (int it = 0; it < iters; ++it) {
      const uint32_t d = tmem + (uint32_t)(it & 1) * TF32_N;
#pragma unroll
      for (int k = 0; k < 4; ++k)
        tc::umma_tf32(d, tc::umma_desc_sw128(base + k * 32), tc::umma_desc_sw128(base + A_BYTES + k * 32), idesc, k ? 1u : 0u);
    }
    tc::umma_commit(tc::smem_u32(&bar));
    tc::mbar_wait(tc::smem_u32(&bar), 0);
  }
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  if (threadIdx.x < 32) {
    uint32_t r[32];
    tc::tmem_ld32(tmem, r);
    if (__uint_as_float(r[0]) == -1.2345f) sink[0] = __uint_as_float(r[1]);
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (threadIdx.x < 32) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(512) : "memory");
}

static __global__ void __launch_bounds__(1024) k_copy_peak(const float4* __restrict__ src, float4* __restrict__ dst, size_t n) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}

// Best of `reps` timed launches after one warm-up; returns seconds (< 0 on a CUDA error).
template <typename F>
inline double time_best(F launch, int reps, cudaStream_t st) {
  cudaEvent_t a, b;
  if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return -1.0;
  launch();
  double best = -1.0;
  for (int r = 0; r < reps; ++r) {
    cudaEventRecord(a, st);
    launch();
    cudaEventRecord(b, st);
    if (cudaEventSynchronize(b) != cudaSuccess) { best = -1.0; break; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    if (best < 0 || ms * 1e-3 < best) best = ms * 1e-3;
  }
  cudaEventDestroy(a); cudaEventDestroy(b);
  if (cudaGetLastError() != cudaSuccess) return -1.0;
  return best;
}

inline cdu_status measure(int kind, double* value, cudaStream_t st) {
  int dev = 0, nsm = 148;
  if (cudaGetDevice(&dev) != cudaSuccess) return CDU_ECUDA;
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  float* sink = nullptr;
  if (cudaMalloc(&sink, 256) != cudaSuccess) return CDU_ENOMEM;
  double t = -1.0, work = 0.0;
  if (kind == CDU_PEAK_FP32_FMA) {
    constexpr int CH = 16; const int iters = 4096, grid = nsm * 2;
    t = time_best([&] { k_fma_peak<float, CH><<<grid, 1024, 0, st>>>(iters, sink); }, 5, st);
    work = 2.0 * grid * 1024.0 * CH * 8.0 * iters / 1e12;
  } else if (kind == CDU_PEAK_FP64_FMA) {
    constexpr int CH = 8; const int iters = 1024, grid = nsm * 2;
    t = time_best([&] { k_fma_peak<double, CH><<<grid, 1024, 0, st>>>(iters, reinterpret_cast<double*>(sink)); }, 5, st);
    work = 2.0 * grid * 1024.0 * CH * 8.0 * iters / 1e12;
  } else if (kind == CDU_PEAK_TF32_TENSOR) {
    const int iters = 8192, smem = 128 * 32 * 4 + TF32_N * 32 * 4 + 1024;
    if (cudaFuncSetAttribute(k_tf32_peak, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) { cudaFree(sink); return CDU_ECUDA; }
    t = time_best([&] { k_tf32_peak<<<nsm, 128, smem, st>>>(iters, sink); }, 5, st);
    work = 2.0 * 128.0 * TF32_N * 32.0 * iters * nsm / 1e12;
  } else if (kind == CDU_PEAK_TF32_MMA_SYNC) {
    const int iters = 4096, grid = nsm;
    t = time_best([&] { k_mma_sync_peak<<<grid, 512, 0, st>>>(iters, sink); }, 5, st);
    work = 2.0 * 16.0 * 8.0 * 8.0 * 8.0 * iters * 16.0 * grid / 1e12;      // 8 mma of 16x8x8 per warp and iteration, 16 warps
  } else if (kind == CDU_PEAK_HBM_COPY) {
    const size_t n = (size_t)1 << 26;   // 2 x 1 GiB
    float4 *a = nullptr, *b = nullptr;
    if (cudaMalloc(&a, n * 16) != cudaSuccess || cudaMalloc(&b, n * 16) != cudaSuccess) { cudaFree(a); cudaFree(sink); return CDU_ENOMEM; }
    cudaMemsetAsync(a, 0, n * 16, st);
    t = time_best([&] { k_copy_peak<<<nsm * 8, 1024, 0, st>>>(a, b, n); }, 5, st);
    work = 2.0 * n * 16 / 1e9;
    cudaFree(a); cudaFree(b);
  } else {
    cudaFree(sink);
    return CDU_EINVAL;
  }
  cudaFree(sink);
  if (!(t > 0.0)) return CDU_ECUDA;
  *value = work / t;
  return CDU_OK;
}

}  // namespace peaks
}  // namespace cdu

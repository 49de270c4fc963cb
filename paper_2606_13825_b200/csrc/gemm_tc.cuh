// gemm_tc.cuh - tcgen05 (3xTF32) batched GEMM for the large-block rebuild U max(L,0) U' (Eq. 7)
// and the four Dalecki-Krein products (Eq. 9).
//
//   C[b] = A[b] * Bt[b]'      A[b], Bt[b]: p x p row-major (both operands "K-major"), p a multiple of 128,
//                              all blocks of the batch the same order; optional fused Hadamard C o Gamma(lam).
// tcgen05.mma has no fp32 kind (tf32 / f16 / i8 / f8f6f4 only), and TF32's 10 mantissa bits would break the 1e-4
// iterate tolerance, so every product is the 3xTF32 split
//   a = a_hi + a_lo (a_hi = a rounded to TF32, a_lo = a - a_hi rounded to TF32)
//   a b ~= a_lo b_hi + a_hi b_lo + a_hi b_hi,  fp32 accumulation in TMEM        (error ~2^-21 relative per term, unbiased)
// One CTA computes one 128 x 128 tile of one block: grid = (p/128)^2 x nblk (cfg5: 16 x 8 = 128 CTAs on 148 SMs).
//   warp 0      TMA producer: cp.async.bulk.tensor of the raw fp32 A / Bt tiles (128 rows x 32 floats, 128-byte
//               swizzle) into a STAGES-deep ring
//   warp 1      TMEM allocation; one elected lane issues 12 tcgen05.mma (M128 N128 K8, kind::tf32) per stage: the
//               leading term a_hi b_hi into a per-stage accumulator (H0 / H1 alternate), the small terms into L
//   warps 2-5   "split" warps: round the hi tiles in place and derive the lo tiles in shared memory (same swizzled offsets, so purely element-wise),
//   warps 6-9   "drain" warps: tcgen05.ld of every per-stage accumulator, summed in registers round-to-nearest (the
//               tensor core's own accumulation truncates; see the kernel), then L, the Gamma Hadamard and the stores
// Synchronisation: full[s] (TMA bytes landed) -> split[s] (hi/lo tiles written, fence.proxy.async) -> tcgen05.commit
// -> empty[s] and tfull[slot] -> drain -> tempty[slot]; a last commit -> lfull.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <map>
#include <string>
#include "cdu.h"

namespace cdu {
namespace tc {

constexpr int TILE = 128;          // M = N = 128
constexpr int BK = 32;             // floats per stage row = 128 bytes = one swizzle atom
constexpr int STAGES = 3;
constexpr int TILE_BYTES = TILE * BK * 4;                    // 16 KB
constexpr int STAGE_BYTES = 4 * TILE_BYTES;                  // A, A_lo, B, B_lo
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*alignment slack*/ + 256 /*barriers*/;
constexpr int SPLIT_WARPS = 4;
constexpr int DRAIN_WARPS = 8;          // (TMEM lane quarter, column half) each
constexpr int THREADS = 32 * (2 + SPLIT_WARPS + DRAIN_WARPS);
constexpr int TMEM_COLS = 512;        // H0, H1 (leading term, double buffered), L (small terms); power of two

#ifdef CDU_GEMM_TIMING
__device__ long long g_gemm_tim[128 * 16];
#define GT_DECL() long long gt_a_ = 0, gt_b_ = 0, gt_c_ = 0, gt_t_ = clock64(), gt_0_ = gt_t_
#define GT_MARK(x) do { const long long n_ = clock64(); x += n_ - gt_t_; gt_t_ = n_; } while (0)
#define GT_OUT(base) do { const long long n_ = clock64(); g_gemm_tim[(blockIdx.x + gridDim.x * blockIdx.y) * 16 + (base)] = gt_a_; g_gemm_tim[(blockIdx.x + gridDim.x * blockIdx.y) * 16 + (base) + 1] = gt_b_; g_gemm_tim[(blockIdx.x + gridDim.x * blockIdx.y) * 16 + (base) + 2] = gt_c_; g_gemm_tim[(blockIdx.x + gridDim.x * blockIdx.y) * 16 + (base) + 3] = n_ - gt_0_; } while (0)
#else
#define GT_DECL() do {} while (0)
#define GT_MARK(x) do {} while (0)
#define GT_OUT(base) do {} while (0)
#endif
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok = 0;
  while (!ok) {
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  }
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
// K-major, 128-byte swizzle: rows of 128 bytes, 8-row groups 1024 bytes apart (SBO); LBO unused; version 1 (sm_100).
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
  d |= (uint64_t)1 << 16;                 // leading byte offset (ignored for swizzled K-major)
  d |= (uint64_t)(1024 >> 4) << 32;       // stride byte offset
  d |= (uint64_t)1 << 46;                 // descriptor version
  d |= (uint64_t)2 << 61;                 // SWIZZLE_128B
  return d;
}
// kind::tf32, fp32 accumulate, A and B K-major, M = 128, N = 128
__host__ __device__ constexpr uint32_t umma_idesc_tf32() {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(TILE >> 3) << 17) | ((uint32_t)(TILE >> 4) << 24);
}
__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, "
      "%24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
        "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]),
        "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]),
        "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
// a = hi + lo with hi = a rounded to nearest TF32 and lo = (a - hi) rounded to nearest TF32: the tensor core
// truncates its fp32 inputs to 19 bits, which would bias every sum; pre-rounded values pass through unchanged.
__device__ __forceinline__ void split_tf32(float a, float& hi, float& lo) {
  uint32_t h, l;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(h) : "f"(a));
  hi = __uint_as_float(h);
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(l) : "f"(a - hi));
  lo = __uint_as_float(l);
}
// lo part of the 3xTF32 split against the tensor core's own truncation of the hi operand
__device__ __forceinline__ float lo_tf32(float a) {
  const float r = a - __uint_as_float(__float_as_uint(a) & 0xffffe000u);
  return __uint_as_float((__float_as_uint(r) + 0x1000u) & 0xffffe000u);
}
__device__ __forceinline__ float gamma_relu_f(float li, float lj) {   // same rule as psd_small.cuh (reading A11)
  const bool pi = li > 0.f, pj = lj > 0.f;
  if (pi && pj) return 1.f;
  if (!pi && !pj) return 0.f;
  return (li > lj ? li : lj) / (fabsf(li) + fabsf(lj));
}

// C[lb] (p x p, row-major) = A[lb] Bt[lb]'  (+ Hadamard with Gamma(lam) when lam != NULL). mapA / mapB: 3-D tensor maps
// {p, p, nblk} of the fp32 operands, box {BK, TILE, 1}, 128-byte swizzle.
static __global__ void __launch_bounds__(THREADS, 1)
k_gemm_tc(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB, float* __restrict__ C, int p,
          const float* __restrict__ lam, const int* __restrict__ need) {
  extern __shared__ unsigned char smem_dyn[];
  if (need && !need[blockIdx.y]) return;
  const uint32_t raw = smem_u32(smem_dyn);
  const uint32_t base = (raw + 1023u) & ~1023u;
  unsigned char* gbase = smem_dyn + (base - raw);
  const uint32_t bars = base + STAGES * STAGE_BYTES;      // 8 bytes each
  auto full = [&](int s) { return bars + 8u * s; };
  auto split = [&](int s) { return bars + 8u * (STAGES + s); };
  auto empty = [&](int s) { return bars + 8u * (2 * STAGES + s); };
  auto tfull = [&](int i) { return bars + 8u * (3 * STAGES + i); };
  auto tempty = [&](int i) { return bars + 8u * (3 * STAGES + 2 + i); };
  const uint32_t lfull = bars + 8u * (3 * STAGES + 4);
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(gbase + STAGES * STAGE_BYTES + 8 * (3 * STAGES + 5));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nt = p / TILE, tm = blockIdx.x / nt, tn = blockIdx.x - tm * nt, lb = blockIdx.y;
  const int nk = p / BK;

  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(full(s), 1); mbar_init(split(s), 32 * SPLIT_WARPS); mbar_init(empty(s), 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(tfull(i), 1); mbar_init(tempty(i), 32 * DRAIN_WARPS); }
    mbar_init(lfull, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    // the first ring of operand tiles is requested before the TMEM allocation and the block-wide barrier below
    for (int kb = 0; kb < STAGES && kb < p / BK; ++kb) {
      mbar_expect_tx(full(kb), 2 * TILE_BYTES);
      const uint32_t st = base + kb * STAGE_BYTES;
      tma_load_3d(st, &mapA, full(kb), kb * BK, (int)(blockIdx.x / (p / TILE)) * TILE, blockIdx.y);
      tma_load_3d(st + 2 * TILE_BYTES, &mapB, full(kb), kb * BK, (int)(blockIdx.x % (p / TILE)) * TILE, blockIdx.y);
    }
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32((const void*)tmem_slot)), "n"(TMEM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = *tmem_slot;           // columns [0,128) H0, [128,256) H1, [256,384) L

  if (warp == 0) {
    if (lane == 0) {
      GT_DECL();
      for (int kb = STAGES; kb < nk; ++kb) {
        const int s = kb % STAGES; const uint32_t ph = (uint32_t)(kb / STAGES) & 1u;
        GT_MARK(gt_b_);
        mbar_wait(empty(s), ph ^ 1u);
        GT_MARK(gt_a_);
        mbar_expect_tx(full(s), 2 * TILE_BYTES);
        const uint32_t st = base + s * STAGE_BYTES;
        tma_load_3d(st, &mapA, full(s), kb * BK, tm * TILE, lb);
        tma_load_3d(st + 2 * TILE_BYTES, &mapB, full(s), kb * BK, tn * TILE, lb);
      }
      GT_OUT(0);
    }
  } else if (warp == 1) {
    if (lane == 0) {
      constexpr uint32_t idesc = umma_idesc_tf32();
      GT_DECL();
      for (int kb = 0; kb < nk; ++kb) {
        const int s = kb % STAGES; const uint32_t ph = (uint32_t)(kb / STAGES) & 1u;
        const int slot = kb & 1;
        GT_MARK(gt_c_);
        mbar_wait(tempty(slot), ((uint32_t)(kb >> 1) & 1u) ^ 1u);     // the drain warps have emptied H[slot]
        GT_MARK(gt_a_);
        mbar_wait(split(s), ph);
        GT_MARK(gt_b_);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const uint32_t st = base + s * STAGE_BYTES;
        const uint32_t dH = tmem + (uint32_t)slot * TILE, dL = tmem + 2u * TILE;
#pragma unroll
        for (int k = 0; k < BK / 8; ++k) {
          const uint64_t ah = umma_desc_sw128(st + k * 32), al = umma_desc_sw128(st + TILE_BYTES + k * 32);
          const uint64_t bh = umma_desc_sw128(st + 2 * TILE_BYTES + k * 32), bl = umma_desc_sw128(st + 3 * TILE_BYTES + k * 32);
          umma_tf32(dL, al, bh, idesc, (kb | k) ? 1u : 0u);   // small terms: one accumulator over the whole K
          umma_tf32(dL, ah, bl, idesc, 1u);
          umma_tf32(dH, ah, bh, idesc, k ? 1u : 0u);          // leading term: a fresh accumulator per 32-wide K chunk
        }
        umma_commit(empty(s));
        umma_commit(tfull(slot));
      }
      umma_commit(lfull);
      GT_OUT(4);
    }
  } else if (warp < 2 + SPLIT_WARPS) {
    // split warps: the hi operand is the raw fp32 tile - the tensor core drops the low 13 mantissa bits of a kind::tf32
    // input, i.e. it multiplies trunc(a) - and lo = a - trunc(a), rounded to nearest TF32, makes up for exactly that
    // truncation (|error| <= 2^-21 |a|, unbiased). Only the lo tiles are written: 1 shared-memory write per element read.
    const int t = threadIdx.x - 64;   // 0 .. 32 SPLIT_WARPS - 1
    constexpr int NT = 32 * SPLIT_WARPS;
    GT_DECL();
    for (int kb = 0; kb < nk; ++kb) {
      const int s = kb % STAGES; const uint32_t ph = (uint32_t)(kb / STAGES) & 1u;
      GT_MARK(gt_b_);
      mbar_wait(full(s), ph);
      GT_MARK(gt_a_);
      float4* st = reinterpret_cast<float4*>(gbase + s * STAGE_BYTES);
#pragma unroll
      for (int half = 0; half < 2; ++half) {
        const float4* hi = st + half * (2 * TILE_BYTES / 16);
        float4* lo = st + half * (2 * TILE_BYTES / 16) + TILE_BYTES / 16;
#pragma unroll
        for (int i = 0; i < TILE_BYTES / 16 / NT; ++i) {
          const float4 v = hi[t + NT * i];
          float4 l;
          l.x = lo_tf32(v.x); l.y = lo_tf32(v.y); l.z = lo_tf32(v.z); l.w = lo_tf32(v.w);
          lo[t + NT * i] = l;
        }
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_arrive(split(s));
    }
    if (t == 0) GT_OUT(8);
  } else {
    // drain warps: the tensor core adds into its accumulator with truncation, which over K/8 additions biases the
    // result by ~1e-5 relative - too much for BPTT through hundreds of steps. So the leading term is accumulated in
    // TMEM over one 32-wide K chunk only (4 additions) and the chunks are summed here, in registers, round-to-nearest.
    // TMEM lane = tile row; a warp may only touch lanes 32 (warp % 4) .. +31.
    const int q = warp & 3, row = q * 32 + lane, half = (warp - (2 + SPLIT_WARPS)) >> 2;
    constexpr int HC = TILE / 2;       // columns per drain warp
    const uint32_t lane_off = (uint32_t)(q * 32) << 16;
    float acc[HC];
#pragma unroll
    for (int j = 0; j < HC; ++j) acc[j] = 0.f;
    GT_DECL();
    for (int kb = 0; kb < nk; ++kb) {
      const int slot = kb & 1;
      GT_MARK(gt_b_);
      mbar_wait(tfull(slot), (uint32_t)(kb >> 1) & 1u);
      GT_MARK(gt_a_);
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
      for (int c = 0; c < HC / 32; ++c) {
        uint32_t r[32];
        tmem_ld32(tmem + lane_off + (uint32_t)(slot * TILE + half * HC + c * 32), r);
#pragma unroll
        for (int j = 0; j < 32; ++j) acc[c * 32 + j] += __uint_as_float(r[j]);
      }
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      mbar_arrive(tempty(slot));
    }
    GT_MARK(gt_b_);
    mbar_wait(lfull, 0);
    GT_MARK(gt_a_);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const int gi = tm * TILE + row;
    const float* l = lam ? lam + (size_t)lb * p : nullptr;
    const float li = l ? l[gi] : 0.f;
    // every MMA has completed (lfull): the operand ring is free and stages the tile, so that the global stores are whole
    // 256-byte row segments per half warp instead of one 16-byte piece per lane and row
    constexpr int LDS_ = TILE + 4;
    float* stg = reinterpret_cast<float*>(gbase);
#pragma unroll
    for (int c = 0; c < HC / 32; ++c) {
      uint32_t r[32];
      tmem_ld32(tmem + lane_off + (uint32_t)(2 * TILE + half * HC + c * 32), r);
#pragma unroll
      for (int j = 0; j < 32; j += 4) {
        float4 o = make_float4(acc[c * 32 + j] + __uint_as_float(r[j]), acc[c * 32 + j + 1] + __uint_as_float(r[j + 1]),
                               acc[c * 32 + j + 2] + __uint_as_float(r[j + 2]), acc[c * 32 + j + 3] + __uint_as_float(r[j + 3]));
        if (l) {
          const float4 lj = *reinterpret_cast<const float4*>(l + tn * TILE + half * HC + c * 32 + j);
          o.x *= gamma_relu_f(li, lj.x); o.y *= gamma_relu_f(li, lj.y); o.z *= gamma_relu_f(li, lj.z); o.w *= gamma_relu_f(li, lj.w);
        }
        *reinterpret_cast<float4*>(stg + row * LDS_ + half * HC + c * 32 + j) = o;
      }
    }
    __syncwarp();      // a warp stages and stores the same 32 rows x 64 columns
    float* cbase = C + (size_t)lb * p * p + (size_t)(tm * TILE + q * 32) * p + tn * TILE + half * HC;
    const int r2 = lane >> 4, c4 = 4 * (lane & 15);
#pragma unroll 4
    for (int rr = 0; rr < 32; rr += 2)
      *reinterpret_cast<float4*>(cbase + (size_t)(rr + r2) * p + c4) = *reinterpret_cast<const float4*>(stg + (q * 32 + rr + r2) * LDS_ + half * HC + c4);
    GT_MARK(gt_c_);
    if (row == 0 && half == 0) GT_OUT(12);
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(TMEM_COLS) : "memory");
}

// Vt (rows = eigenvectors) -> V = Vt' and Vs = V diag(lam) (lam = the rebuild's scale vector): the K-major operands
// of the rebuild Vs V' and of the products that contract over the eigenvector index. 32 x 32 tiles through shared memory.
static __global__ void __launch_bounds__(256) k_tc_transpose(int p, const float* __restrict__ Vt, const float* __restrict__ lam,
                                                      float* __restrict__ V, float* __restrict__ Vs) {
  __shared__ float tl[32][33];
  const size_t off = (size_t)blockIdx.z * p * p;
  const int i0 = blockIdx.y * 32, a0 = blockIdx.x * 32;   // Vt[i][a], i = eigenvector
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  for (int r = ty; r < 32; r += 8) tl[r][tx] = Vt[off + (size_t)(i0 + r) * p + a0 + tx];
  __syncthreads();
  const float sc = lam ? lam[(size_t)blockIdx.z * p + i0 + tx] : 0.f;
  for (int r = ty; r < 32; r += 8) {
    const float v = tl[tx][r];   // Vt[i0 + tx][a0 + r]
    const size_t o = off + (size_t)(a0 + r) * p + i0 + tx;
    if (V) V[o] = v;
    if (Vs) Vs[o] = v * sc;
  }
}

// ---- host side -------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
inline EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(f);
  }
  return fn;
}

// Tensor maps of the [nblk][p][p] fp32 operand buffers, made once per buffer (the scratch pointers of a handle never change).
struct Maps {
  int nblk = 0, p = 0;
  bool attr_set = false;
  std::map<const void*, CUtensorMap> cache;
  const CUtensorMap* get(const float* buf, std::string& err) {
    auto it = cache.find(buf);
    if (it != cache.end()) return &it->second;
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) { err = "cuTensorMapEncodeTiled not available"; return nullptr; }
    CUtensorMap m;
    const cuuint64_t dims[3] = {(cuuint64_t)p, (cuuint64_t)p, (cuuint64_t)nblk};
    const cuuint64_t strides[2] = {(cuuint64_t)p * 4, (cuuint64_t)p * p * 4};
    const cuuint32_t box[3] = {BK, TILE, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = enc(&m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(buf), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { err = "cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")"; return nullptr; }
    return &(cache[buf] = m);
  }
};

// C = A Bt' per block (A, Bt, C: [nblk][p][p] fp32, row-major), optional Hadamard with Gamma(lam).
inline cdu_status gemm_nt(Maps& M, const float* A, const float* Bt, float* C, const float* lam, const int* need, cudaStream_t st, std::string& err) {
  const CUtensorMap* ma = M.get(A, err);
  const CUtensorMap* mb = M.get(Bt, err);
  if (!ma || !mb) return CDU_ECUDA;
  if (!M.attr_set) {
    if (cudaFuncSetAttribute(k_gemm_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES) != cudaSuccess) {
      err = "cudaFuncSetAttribute(k_gemm_tc)"; return CDU_ECUDA;
    }
    M.attr_set = true;
  }
  const int nt = M.p / TILE;
  k_gemm_tc<<<dim3(nt * nt, M.nblk), THREADS, SMEM_BYTES, st>>>(*ma, *mb, C, M.p, lam, need);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { err = std::string("k_gemm_tc: ") + cudaGetErrorString(e); return CDU_ECUDA; }
  return CDU_OK;
}

}  // namespace tc

inline bool gemm_tc_supported(int p) { return p >= tc::TILE && p % tc::TILE == 0; }

}  // namespace cdu

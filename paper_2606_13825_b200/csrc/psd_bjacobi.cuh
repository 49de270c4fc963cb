// psd_bjacobi.cuh - eigendecomposition of the large PSD blocks: blocked one-sided Jacobi in shared memory.
//
// Same fixed point as k_hestenes (psd_large.cuh): the rows g_i = (S + mu I) v_i of G are made mutually orthogonal by
// plane rotations applied to (G, Vt) alike; then v_i are eigenvectors of S and lambda_i = ||g_i|| / ||v_i|| - mu
// (Eq. 7: only U max(L,0) U' is compared with the oracle, never U - reading A15). What changes is
// the schedule, which is built for the SM instead of for L2 latency:
//   * rows are grouped in blocks of BR; one round of a round-robin tournament over the NB blocks pairs every block
//     with one other, and one CTA of the matrix's thread-block cluster takes one pair: it brings the 2 BR rows of G
//     and of Vt (2 BR x p each) into shared memory, forms their Gram matrix W = X X' (2 BR x 2 BR, register-tiled,
//     k split over 8 thread groups), runs ONE cyclic sweep of two-sided Jacobi on W in shared memory (rotation
//     threshold relative to sqrt(w_ii w_jj), de Rijk), accumulating the rotations in Q, and applies Q to both row
//     sets (X <- Q X, Y <- Q Y; one thread per column, Q broadcast from shared memory). Rows go back to L2 and the
//     cluster meets at one barrier per ROUND OF BLOCKS (NB - 1 per sweep) instead of one per round of rows (p - 1);
//   * a pair whose Gram matrix is already diagonal to the tolerance costs a load and the Gram product only;
//   * the sweep count falls further with a warm start: the caller may pass Vt = the previous iterate's eigenvectors
//     and G = Vt (S + mu I) (one GEMM), since consecutive ADMM iterates have nearby eigenbases.
// On exit Vt holds the normalised rows of G (orthonormal to the convergence tolerance whatever rounding did to the
// accumulated rotations), lam the eigenvalues.
#pragma once
#include <cooperative_groups.h>
#include "common.cuh"
#include "psd_small.cuh"

namespace cdu {
namespace bj {
namespace cg = cooperative_groups;

constexpr int THREADS = 512;
constexpr int KSL = 8;            // k slices of the Gram product
constexpr int MAXSW = 64;

template <typename T> struct V4 { using type = float4; static constexpr int W = 4; };
template <> struct V4<double> { using type = double2; static constexpr int W = 2; };

// shared-memory plan for RP = 2 BR rows of length p
template <typename T, int RP> struct Plan {
  int ldx;           // row stride of X / Y (elements); columns [p, ldx) stay zero
  size_t off_y, off_part, off_w, off_q, off_rot, off_red, bytes;
  __host__ __device__ explicit Plan(int p) {
    constexpr int VW = V4<T>::W;
    ldx = ((p + 3) / 4) * 4 + 4;     // multiple of 4 (16-byte rows for float), +4: rows 0..7 start in distinct bank groups
    size_t o = (size_t)RP * ldx * sizeof(T);
    off_y = o; o += (size_t)RP * ldx * sizeof(T);
    off_part = o; o += (size_t)KSL * RP * (RP + 1) * sizeof(T);
    off_w = o; o += (size_t)RP * (RP + 1) * sizeof(T);
    off_q = o; o += (size_t)RP * (RP + 4) * sizeof(T);
    off_rot = o; o += (size_t)(RP / 2) * 4 * sizeof(T);
    off_red = (o + 15) & ~(size_t)15; o = off_red + 64 * sizeof(double);
    bytes = o;
  }
};

__device__ __forceinline__ float ld_cg(const float* p) { return __ldcg(p); }
__device__ __forceinline__ double ld_cg(const double* p) { return __ldcg(p); }

// rows [r0, r0 + BR) of a p x p row-major matrix -> shared rows [s0, s0 + BR); rows >= p are zero.
template <typename T, int BR>
__device__ __forceinline__ void load_rows(const T* __restrict__ g, int p, int r0, T* X, int ldx, int s0) {
  using VT = typename V4<T>::type;
  constexpr int VW = V4<T>::W;
  if ((p % VW) == 0) {
    const int nv = p / VW;
    for (int t = threadIdx.x; t < BR * nv; t += blockDim.x) {
      const int r = t / nv, c = t - r * nv;
      VT v;
      if (r0 + r < p) v = __ldcg(reinterpret_cast<const VT*>(g + (size_t)(r0 + r) * p) + c);
      else memset(&v, 0, sizeof(v));
      reinterpret_cast<VT*>(X + (size_t)(s0 + r) * ldx)[c] = v;
    }
  } else {
    for (int t = threadIdx.x; t < BR * p; t += blockDim.x) {
      const int r = t / p, c = t - r * p;
      X[(size_t)(s0 + r) * ldx + c] = (r0 + r < p) ? ld_cg(g + (size_t)(r0 + r) * p + c) : (T)0;
    }
  }
}
template <typename T, int BR>
__device__ __forceinline__ void store_rows(T* __restrict__ g, int p, int r0, const T* X, int ldx, int s0) {
  using VT = typename V4<T>::type;
  constexpr int VW = V4<T>::W;
  if ((p % VW) == 0) {
    const int nv = p / VW;
    for (int t = threadIdx.x; t < BR * nv; t += blockDim.x) {
      const int r = t / nv, c = t - r * nv;
      if (r0 + r < p) __stcg(reinterpret_cast<VT*>(g + (size_t)(r0 + r) * p) + c, reinterpret_cast<const VT*>(X + (size_t)(s0 + r) * ldx)[c]);
    }
  } else {
    for (int t = threadIdx.x; t < BR * p; t += blockDim.x) {
      const int r = t / p, c = t - r * p;
      if (r0 + r < p) __stcg(g + (size_t)(r0 + r) * p + c, X[(size_t)(s0 + r) * ldx + c]);
    }
  }
}

__device__ __forceinline__ void load4(const float* p, float (&o)[4]) {
  const float4 v = *reinterpret_cast<const float4*>(p); o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w;
}
__device__ __forceinline__ void load4(const double* p, double (&o)[4]) {
  const double2 a = *reinterpret_cast<const double2*>(p), b = *reinterpret_cast<const double2*>(p + 2);
  o[0] = a.x; o[1] = a.y; o[2] = b.x; o[3] = b.y;
}

// part[s] = X[:, slice s] X[:, slice s]'  for the 8 k slices; thread (s, it, jt) owns rows it + 8 r and jt + 8 r'.
template <typename T, int RP>
__device__ __forceinline__ void gram_partials(const T* X, int ldx, int p, T* part) {
  constexpr int TR = RP / 8;
  const int s = threadIdx.x >> 6, it = threadIdx.x & 7, jt = (threadIdx.x >> 3) & 7;
  const int ks = ((p + KSL - 1) / KSL + 3) & ~3;
  const int k0 = s * ks, k1 = min(p, k0 + ks);
  T acc[TR][TR];
#pragma unroll
  for (int a = 0; a < TR; ++a)
#pragma unroll
    for (int b = 0; b < TR; ++b) acc[a][b] = (T)0;
  for (int k = k0; k < k1; k += 4) {      // rows are zero padded to ldx >= k1 rounded up to 4
    T xi[TR][4], xj[TR][4];
#pragma unroll
    for (int a = 0; a < TR; ++a) {
      load4(X + (size_t)(it + 8 * a) * ldx + k, xi[a]);
      load4(X + (size_t)(jt + 8 * a) * ldx + k, xj[a]);
    }
#pragma unroll
    for (int a = 0; a < TR; ++a)
#pragma unroll
      for (int b = 0; b < TR; ++b)
#pragma unroll
        for (int e = 0; e < 4; ++e) acc[a][b] += xi[a][e] * xj[b][e];
  }
#pragma unroll
  for (int a = 0; a < TR; ++a)
#pragma unroll
    for (int b = 0; b < TR; ++b) part[((size_t)s * RP + it + 8 * a) * (RP + 1) + jt + 8 * b] = acc[a][b];
}

// W = sum_s part[s]; returns (to every thread) max_{i<j} |w_ij| / sqrt(w_ii w_jj).
template <typename T, int RP>
__device__ __forceinline__ double gram_reduce(const T* part, T* W, double* red) {
  for (int t = threadIdx.x; t < RP * RP; t += blockDim.x) {
    const int i = t / RP, j = t - i * RP;
    double a = 0.0;
#pragma unroll
    for (int s = 0; s < KSL; ++s) a += (double)part[((size_t)s * RP + i) * (RP + 1) + j];
    W[i * (RP + 1) + j] = (T)a;
  }
  __syncthreads();
  double mx = 0.0;
  for (int t = threadIdx.x; t < RP * RP; t += blockDim.x) {
    const int i = t / RP, j = t - i * RP;
    if (i < j) {
      const double d = (double)W[i * (RP + 1) + i] * (double)W[j * (RP + 1) + j];
      if (d > 0.0) mx = fmax(mx, fabs((double)W[i * (RP + 1) + j]) * rsqrt(d));
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = mx;
  __syncthreads();
  mx = 0.0;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) mx = fmax(mx, red[w]);
  __syncthreads();
  return mx;
}

// One cyclic sweep (RP - 1 rounds of RP / 2 disjoint rotations) of two-sided Jacobi on W; Q (RP x RP, row stride
// RP + 4) accumulates the rotations: on exit row i of Q holds the combination of the old rows that makes new row i.
template <typename T, int RP>
__device__ __forceinline__ void inner_sweep(T* W, T* Q, T* rot, T thresh) {
  constexpr int H = RP / 2, LW = RP + 1, LQ = RP + 4;
  const int tid = threadIdx.x;
  for (int t = tid; t < RP * RP; t += blockDim.x) { const int i = t / RP, j = t - i * RP; Q[i * LQ + j] = (i == j) ? (T)1 : (T)0; }
  __syncthreads();
  for (int r = 0; r < RP - 1; ++r) {
    if (tid < H) {
      int i, j; rr_pair(r, tid, RP, i, j);
      const T a = W[i * LW + i], b = W[j * LW + j], c = W[i * LW + j];
      T sn = (T)0, tau = (T)0;
      if (fabs(c) > thresh * sqrt(a * b)) {
        const T th = (b - a) / ((T)2 * c);
        const T t = ((th >= (T)0) ? (T)1 : (T)-1) / (fabs(th) + sqrt((T)1 + th * th));
        const T cs = (T)1 / sqrt((T)1 + t * t);
        sn = t * cs; tau = sn / ((T)1 + cs);
      }
      rot[2 * tid] = sn; rot[2 * tid + 1] = tau;
    }
    __syncthreads();
    // W <- J' W J on 2 x 2 blocks (rows pair q1, columns pair q2); Q <- J' Q on row pairs
    for (int t = tid; t < H * H; t += blockDim.x) {
      const int q1 = t / H, q2 = t - q1 * H;
      int i1, j1, i2, j2; rr_pair(r, q1, RP, i1, j1); rr_pair(r, q2, RP, i2, j2);
      const T s1 = rot[2 * q1], t1 = rot[2 * q1 + 1], s2 = rot[2 * q2], t2 = rot[2 * q2 + 1];
      T a = W[i1 * LW + i2], b = W[i1 * LW + j2], c = W[j1 * LW + i2], d = W[j1 * LW + j2];
      rot2(s1, t1, a, c); rot2(s1, t1, b, d);      // rows i1, j1
      rot2(s2, t2, a, b); rot2(s2, t2, c, d);      // columns i2, j2
      W[i1 * LW + i2] = a; W[i1 * LW + j2] = b; W[j1 * LW + i2] = c; W[j1 * LW + j2] = d;
    }
    for (int t = tid; t < H * RP; t += blockDim.x) {
      const int q = t / RP, col = t - q * RP;
      int i, j; rr_pair(r, q, RP, i, j);
      T x = Q[i * LQ + col], y = Q[j * LQ + col];
      rot2(rot[2 * q], rot[2 * q + 1], x, y);
      Q[i * LQ + col] = x; Q[j * LQ + col] = y;
    }
    __syncthreads();
  }
}

// X <- Q X for the columns [0, p): one thread per column, Q read as broadcast vectors.
template <typename T, int RP>
__device__ __forceinline__ void apply_q(const T* Q, T* X, int ldx, int p) {
  constexpr int LQ = RP + 4;
  for (int k = threadIdx.x; k < p; k += blockDim.x) {
    T x[RP];
#pragma unroll
    for (int j = 0; j < RP; ++j) x[j] = X[(size_t)j * ldx + k];
#pragma unroll 4
    for (int i = 0; i < RP; ++i) {
      T o = (T)0;
#pragma unroll
      for (int j = 0; j < RP; j += 4) {
        T q[4];
        load4(Q + i * LQ + j, q);
        o += q[0] * x[j] + q[1] * x[j + 1] + q[2] * x[j + 2] + q[3] * x[j + 3];
      }
      X[(size_t)i * ldx + k] = o;       // rows < i are already overwritten: x[] holds the old column
    }
  }
}

// One cluster per matrix; CTA `rank` takes block pairs rank, rank + C, ... of every round. G, Vt: p x p row-major,
// row i = (S + mu I) v_i resp. v_i. rotflags[lb][sweep] is raised by any CTA that met a pair above the tolerance.
template <typename T, int RP>
__global__ void __launch_bounds__(THREADS, 1)
k_bjacobi(int nblk, const int* pvec, const long long* moff, const int* voff, T* G, T* Vt, const T* mu, T* lam, int* rotflags,
          int* sweeps_out, unsigned long long* sweeps_sum, int max_sweeps, double tol) {
  constexpr int BR = RP / 2;
  extern __shared__ __align__(16) unsigned char smem_bj[];
  cg::cluster_group cluster = cg::this_cluster();
  const int C = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
  const int lb = blockIdx.x / C;
  const int p = pvec[lb];
  const Plan<T, RP> pl(p);
  T* X = reinterpret_cast<T*>(smem_bj);
  T* Y = reinterpret_cast<T*>(smem_bj + pl.off_y);
  T* part = reinterpret_cast<T*>(smem_bj + pl.off_part);
  T* W = reinterpret_cast<T*>(smem_bj + pl.off_w);
  T* Q = reinterpret_cast<T*>(smem_bj + pl.off_q);
  T* rot = reinterpret_cast<T*>(smem_bj + pl.off_rot);
  double* red = reinterpret_cast<double*>(smem_bj + pl.off_red);
  T* g = G + moff[lb];
  T* vt = Vt + moff[lb];
  int* rf = rotflags + lb * MAXSW;
  const int ldx = pl.ldx;
  const int NB = (p + BR - 1) / BR, NBe = (NB + 1) & ~1, NP = NBe >> 1;
  for (int t = threadIdx.x; t < 2 * RP * ldx; t += blockDim.x) X[t] = (T)0;    // X and Y are contiguous; pads stay zero
  __syncthreads();
  const T thresh = (T)(0.25 * tol);
  int sweep = 0;
  for (; sweep < max_sweeps; ++sweep) {
    for (int r = 0; r < NBe - 1 || (NBe == 2 && r == 0); ++r) {
      for (int q = rank; q < NP; q += C) {
        int bi, bj2; rr_pair(r, q, NBe, bi, bj2);
        load_rows<T, BR>(g, p, bi * BR, X, ldx, 0);
        load_rows<T, BR>(g, p, bj2 * BR, X, ldx, BR);
        __syncthreads();
        gram_partials<T, RP>(X, ldx, p, part);
        __syncthreads();
        const double mx = gram_reduce<T, RP>(part, W, red);
        if (mx > tol) {
          load_rows<T, BR>(vt, p, bi * BR, Y, ldx, 0);          // in flight while the sweep runs
          load_rows<T, BR>(vt, p, bj2 * BR, Y, ldx, BR);
          inner_sweep<T, RP>(W, Q, rot, thresh);
          apply_q<T, RP>(Q, X, ldx, p);
          apply_q<T, RP>(Q, Y, ldx, p);
          __syncthreads();
          store_rows<T, BR>(g, p, bi * BR, X, ldx, 0);
          store_rows<T, BR>(g, p, bj2 * BR, X, ldx, BR);
          store_rows<T, BR>(vt, p, bi * BR, Y, ldx, 0);
          store_rows<T, BR>(vt, p, bj2 * BR, Y, ldx, BR);
          if (threadIdx.x == 0) __stcg(rf + sweep, 1);
        }
        __syncthreads();
      }
      cluster.sync();
      if (NBe == 2) break;
    }
    if (!__ldcg(rf + sweep)) break;
  }
  // eigenvalues; Vt <- normalised rows of G
  const int lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  const double m = (double)mu[lb];
  for (int i = rank * nw + (threadIdx.x >> 5); i < p; i += C * nw) {
    double a = 0.0, b = 0.0;
    for (int c = lane; c < p; c += 32) {
      const double x = (double)ld_cg(g + (size_t)i * p + c), y = (double)ld_cg(vt + (size_t)i * p + c);
      a += x * x; b += y * y;
    }
    a = warp_sum(a); b = warp_sum(b);
    const double na = sqrt(a);
    if (lane == 0) lam[voff[lb] + i] = (T)((b > 0.0 ? na / sqrt(b) : 0.0) - m);
    if (na > 0.0) {
      const double inv = 1.0 / na;
      for (int c = lane; c < p; c += 32) vt[(size_t)i * p + c] = (T)((double)ld_cg(g + (size_t)i * p + c) * inv);
    }
  }
  if (rank == 0 && threadIdx.x == 0) { atomicMax(sweeps_out, sweep); if (sweeps_sum) atomicAdd(sweeps_sum, (unsigned long long)sweep); }
}

template <typename T, int RP> inline size_t smem_bytes(int p) { return Plan<T, RP>(p).bytes; }

}  // namespace bj
}  // namespace cdu

// psd_bjacobi.cuh - eigendecomposition of the large PSD blocks: blocked one-sided Jacobi in shared memory.
//
// Same fixed point as k_hestenes (psd_large.cuh): the rows g_i = v_i' (S + mu I) of G, for an orthonormal set {v_i},
// are made mutually orthogonal by plane rotations; then v_i = g_i / ||g_i|| are eigenvectors of S (Eq. 7,
// L102: only U max(L,0) U' is compared with the oracle, never U - reading A15). The v_i are never formed: rotating
// the rows of G rotates them implicitly, so only G is carried. What changes against k_hestenes is the schedule,
// built for the SM instead of for L2 latency:
//   * rows are grouped in blocks of BR; one round of a round-robin tournament over the NB blocks pairs every block
//     with one other, and one CTA of the matrix's thread-block cluster takes one pair: it brings the 2 BR rows of G
//     (2 BR x p) into shared memory, forms their Gram matrix W = X X' (2 BR x 2 BR, register-tiled, k split over 8
//     thread groups), runs ONE cyclic sweep of two-sided Jacobi on W in shared memory (rotation threshold relative to
//     sqrt(w_ii w_jj), de Rijk), accumulating the rotations in Q, and writes Q X straight back to L2 (4 x 4 register
//     tiles). The cluster meets at one barrier per ROUND OF BLOCKS (NB - 1 per sweep) instead of one per round of
//     rows (p - 1);
//   * a pair whose Gram matrix is already diagonal to the tolerance costs a load and the Gram product only;
//   * the sweep count falls further with a warm start: the caller passes G = V_prev' (S + mu I) (one GEMM) for the
//     previous iterate's eigenvectors, since consecutive ADMM iterates have nearby eigenbases, and a mu from Weyl's
//     inequality (k_large_smat) instead of ||S||_F.
// On exit Vt holds the normalised rows of G (orthonormal to the convergence tolerance by construction) and lam =
// ||g_i|| - mu, which the caller replaces by Rayleigh quotients against the unshifted S (k_large_rayleigh): the
// approximate reciprocals in the rotation set-up scale row pairs by 1 + O(eps), which the quotient does not see.
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
  int ldx;           // row stride of X (elements); columns [p, ldx) stay zero
  size_t off_part, off_w, off_q, off_red, off_pairs, bytes;
  __host__ __device__ explicit Plan(int p) {
    ldx = ((p + 3) / 4) * 4 + 4;     // multiple of 4 (16-byte rows for float), +4: rows 0..7 start in distinct bank groups
    size_t o = (size_t)RP * ldx * sizeof(T);
    off_part = o; o += (size_t)KSL * RP * (RP + 1) * sizeof(T);   // Gram partials; later the second W buffer and Q'
    off_w = o; o += (size_t)RP * (RP + 1) * sizeof(T);
    off_q = o; o += (size_t)RP * (RP + 4) * sizeof(T);
    off_red = (o + 15) & ~(size_t)15; o = off_red + 64 * sizeof(double);
    off_pairs = o; o += (size_t)(RP - 1) * (RP / 2) * sizeof(int);
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

// Rotation (sin, tau = sin / (1 + cos)) that annihilates w_ij, or the identity when |w_ij| <= thresh sqrt(w_ii w_jj).
__device__ __forceinline__ float rcp_approx(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rsqrt_approx(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ void sweep_angle(float a, float b, float c, float thresh, float& sn, float& tau) {
  // approximate reciprocals / square roots: they only perturb the angle and scale the row pair by 1 + O(eps s^2);
  // eigenvalues are Rayleigh quotients taken afterwards and eigenvectors are the normalised rows, so neither matters.
  sn = 0.f; tau = 0.f;
  if (c * c > thresh * thresh * a * b) {
    const float th = (b - a) * rcp_approx(2.f * c);
    const float h2 = 1.f + th * th;
    const float t = copysignf(rcp_approx(fabsf(th) + h2 * rsqrt_approx(h2)), th);
    const float cs = rsqrt_approx(1.f + t * t);
    sn = t * cs; tau = sn * rcp_approx(1.f + cs);
  }
}
__device__ __forceinline__ void sweep_angle(double a, double b, double c, double thresh, double& sn, double& tau) {
  sn = 0.0; tau = 0.0;
  if (fabs(c) > thresh * sqrt(a * b)) {
    const double th = (b - a) / (2.0 * c);
    const double t = (th >= 0.0 ? 1.0 : -1.0) / (fabs(th) + sqrt(1.0 + th * th));
    const double cs = 1.0 / sqrt(1.0 + t * t);
    sn = t * cs; tau = sn / (1.0 + cs);
  }
}

// One cyclic sweep (RP - 1 rounds of RP / 2 disjoint rotations) of two-sided Jacobi on W (double buffered: W0 holds
// the matrix on entry, the result is in the buffer returned). Q (RP x RP, row stride RP + 4) accumulates the
// rotations: row i of Q = the combination of the old rows that makes new row i. One barrier per round: warp q owns
// row pair q; every lane derives the rotation of pair (lane mod RP/2) from the current buffer itself, the warp's own
// rotation comes by shuffle; lanes < RP/2 update the 2 x 2 block (pair q rows, pair lane columns), all lanes the Q rows.
template <typename T, int RP>
__device__ __forceinline__ T* inner_sweep(T* W0, T* W1, T* Q, T thresh, const int* pairs, unsigned* mask) {
  constexpr int H = RP / 2, LW = RP + 1, LQ = RP + 4;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  for (int t = tid; t < RP * RP; t += blockDim.x) { const int i = t / RP, j = t - i * RP; Q[i * LQ + j] = (i == j) ? (T)1 : (T)0; }
  if (tid == 0) *mask = 0u;
  __syncthreads();
  // rounds that hold at least one pair above the convergence tolerance: the others are skipped (late sweeps of a warm-started
  // matrix leave a handful of pairs to rotate; what a rotation adds to other entries is second order and is met by the
  // next sweep of the blocks)
  for (int t = tid; t < (RP - 1) * H; t += blockDim.x) {
    const int pr = pairs[t], i = pr & 0xffff, j = pr >> 16;
    const T c = W0[i * LW + j];
    if (c * c > (T)16 * thresh * thresh * W0[i * LW + i] * W0[j * LW + j]) atomicOr(mask, 1u << (t / H));   // 4 thresh = tol
  }
  __syncthreads();
  const unsigned active = *mask;
  T* Wc = W0; T* Wn = W1;
  for (int r = 0; r < RP - 1; ++r) {
    if (!((active >> r) & 1u)) continue;
    if (warp < H) {
      const int q2 = lane % H;
      const int pr = pairs[r * H + q2], i2 = pr & 0xffff, j2 = pr >> 16;
      T s2, t2;
      sweep_angle(Wc[i2 * LW + i2], Wc[j2 * LW + j2], Wc[i2 * LW + j2], thresh, s2, t2);
      const T s1 = __shfl_sync(0xffffffffu, s2, warp), t1 = __shfl_sync(0xffffffffu, t2, warp);
      const int i1 = __shfl_sync(0xffffffffu, i2, warp), j1 = __shfl_sync(0xffffffffu, j2, warp);
      if (lane < H) {
        T a = Wc[i1 * LW + i2], b = Wc[i1 * LW + j2], c = Wc[j1 * LW + i2], d = Wc[j1 * LW + j2];
        rot2(s1, t1, a, c); rot2(s1, t1, b, d);      // rows i1, j1
        rot2(s2, t2, a, b); rot2(s2, t2, c, d);      // columns i2, j2
        Wn[i1 * LW + i2] = a; Wn[i1 * LW + j2] = b; Wn[j1 * LW + i2] = c; Wn[j1 * LW + j2] = d;
      }
      for (int col = lane; col < RP; col += 32) {
        T x = Q[i1 * LQ + col], y = Q[j1 * LQ + col];
        rot2(s1, t1, x, y);
        Q[i1 * LQ + col] = x; Q[j1 * LQ + col] = y;
      }
    }
    __syncthreads();
    T* tmp = Wc; Wc = Wn; Wn = tmp;
  }
  return Wc;
}

// rows of the pair -> global: new row i = sum_k Q[i][k] X[k][:], written straight to the matrix (rows [0, BR) of the
// pair live at rowA.., rows [BR, RP) at rowB..). Qt = Q' (row stride RP + 4). 4 x 4 register tiles.
template <typename T, int RP>
__device__ __forceinline__ void apply_store(const T* Qt, const T* X, int ldx, int p, T* g, int rowA, int rowB) {
  constexpr int LQ = RP + 4, NRG = RP / 4, TPT = (NRG + 3) / 4, BR = RP / 2;
  const int cl = threadIdx.x & 127, rl = threadIdx.x >> 7;
  const int ncg = (p + 3) >> 2;
  for (int cgi = cl; cgi < ncg; cgi += 128) {
    T acc[TPT][4][4];
#pragma unroll
    for (int u = 0; u < TPT; ++u)
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) acc[u][a][b] = (T)0;
#pragma unroll 4
    for (int k = 0; k < RP; ++k) {
      T x[4];
      load4(X + (size_t)k * ldx + 4 * cgi, x);
#pragma unroll
      for (int u = 0; u < TPT; ++u) {
        const int rg = rl + 4 * u;
        if (rg < NRG) {
          T q[4];
          load4(Qt + k * LQ + 4 * rg, q);
#pragma unroll
          for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) acc[u][a][b] += q[a] * x[b];
        }
      }
    }
#pragma unroll
    for (int u = 0; u < TPT; ++u) {
      const int rg = rl + 4 * u;
      if (rg < NRG) {
#pragma unroll
        for (int a = 0; a < 4; ++a) {
          const int i = 4 * rg + a;
          const int grow = i < BR ? rowA + i : rowB + (i - BR);
          if (grow < p) {
            T* dst = g + (size_t)grow * p + 4 * cgi;
            if ((p & 3) == 0) {
              if (sizeof(T) == 4) __stcg(reinterpret_cast<float4*>(dst), make_float4((float)acc[u][a][0], (float)acc[u][a][1], (float)acc[u][a][2], (float)acc[u][a][3]));
              else { __stcg(reinterpret_cast<double2*>(dst), make_double2((double)acc[u][a][0], (double)acc[u][a][1])); __stcg(reinterpret_cast<double2*>(dst) + 1, make_double2((double)acc[u][a][2], (double)acc[u][a][3])); }
            } else {
#pragma unroll
              for (int b = 0; b < 4; ++b) if (4 * cgi + b < p) __stcg(dst + b, acc[u][a][b]);
            }
          }
        }
      }
    }
  }
}

// One cluster per matrix; CTA `rank` takes block pairs rank, rank + C, ... of every round. G: p x p row-major, row i
// = v_i' (S + mu I) for an orthonormal set {v_i} that is never formed: a rotation of the rows of G rotates the v_i
// with it, and once the rows are mutually orthogonal v_i = g_i / ||g_i|| and lambda_i = ||g_i|| - mu.
// rotflags[lb][sweep] is raised by any CTA that met a pair above the tolerance.
template <typename T, int RP>
__global__ void __launch_bounds__(THREADS, 1)
k_bjacobi(int nblk, const int* pvec, const long long* moff, const int* voff, T* G, T* Vt, const T* mu, T* lam, int* rotflags,
          int* sweeps_out, unsigned long long* sweeps_sum, int max_sweeps, double tol, const int* prob_of, int* flags) {
  constexpr int BR = RP / 2, LQ = RP + 4;
  extern __shared__ __align__(16) unsigned char smem_bj[];
  cg::cluster_group cluster = cg::this_cluster();
  const int C = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
  const int lb = blockIdx.x / C;
  const int p = pvec[lb];
  const Plan<T, RP> pl(p);
  T* X = reinterpret_cast<T*>(smem_bj);
  T* part = reinterpret_cast<T*>(smem_bj + pl.off_part);
  T* W = reinterpret_cast<T*>(smem_bj + pl.off_w);
  T* Q = reinterpret_cast<T*>(smem_bj + pl.off_q);
  T* W1 = part;                                  // free once gram_reduce has consumed the partials
  T* Qt = part + RP * (RP + 1) + 3;              // 16-byte aligned below
  Qt = reinterpret_cast<T*>((reinterpret_cast<uintptr_t>(Qt)) & ~(uintptr_t)15);
  double* red = reinterpret_cast<double*>(smem_bj + pl.off_red);
  T* g = G + moff[lb];
  int* rf = rotflags + lb * MAXSW;
  const int ldx = pl.ldx;
  const int NB = (p + BR - 1) / BR, NBe = (NB + 1) & ~1, NP = NBe >> 1;
  int* pairs = reinterpret_cast<int*>(smem_bj + pl.off_pairs);              // pair (i | j << 16) of round r, table q
  for (int t = threadIdx.x; t < (RP - 1) * BR; t += blockDim.x) { int i, j; rr_pair(t / BR, t % BR, RP, i, j); pairs[t] = i | (j << 16); }
  for (int t = threadIdx.x; t < RP * ldx; t += blockDim.x) X[t] = (T)0;    // the pads stay zero
  __syncthreads();
  const T thresh = (T)(0.25 * tol);
  const float quad_exit = (float)sqrt(tol / (16.0 * sqrt((double)p)));   // 2.9e-5 for fp32 at p = 512
  int sweep = 0;
  bool capped = true;
  for (; sweep < max_sweeps; ++sweep) {
    for (int r = 0; r < NBe - 1; ++r) {
      for (int q = rank; q < NP; q += C) {
        int bi, bj2; rr_pair(r, q, NBe, bi, bj2);
        load_rows<T, BR>(g, p, bi * BR, X, ldx, 0);
        load_rows<T, BR>(g, p, bj2 * BR, X, ldx, BR);
        __syncthreads();
        gram_partials<T, RP>(X, ldx, p, part);
        __syncthreads();
        const double mx = gram_reduce<T, RP>(part, W, red);
        if (mx > tol) {
          const T* Wf = inner_sweep<T, RP>(W, W1, Q, thresh, pairs, reinterpret_cast<unsigned*>(red + 40));
          (void)Wf;
          for (int t = threadIdx.x; t < RP * RP; t += blockDim.x) { const int i = t / RP, k = t - i * RP; Qt[k * LQ + i] = Q[i * LQ + k]; }
          __syncthreads();
          apply_store<T, RP>(Qt, X, ldx, p, g, bi * BR, bj2 * BR);
          if (threadIdx.x == 0) atomicMax(reinterpret_cast<unsigned*>(rf) + sweep, __float_as_uint((float)mx));   // mx > 0: ordered as unsigned
        }
        __syncthreads();
      }
      cluster.sync();
    }
    const unsigned worst = (unsigned)__ldcg(rf + sweep);     // largest |w_ij| / sqrt(w_ii w_jj) any pair showed in this sweep
    if (!worst) { capped = false; break; }                    // nothing above the tolerance: converged
    if (__uint_as_float(worst) <= quad_exit) { ++sweep; capped = false; break; }   // quadratic convergence: every pair above tol was rotated while
  }                                                           // all ratios were <= quad_exit; what is left is ~quad_exit^2 sqrt(p) <= tol / 16
  // eigenvalues and eigenvectors
  const int lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  const double m = (double)mu[lb];
  T* vt = Vt + moff[lb];
  for (int i = rank * nw + (threadIdx.x >> 5); i < p; i += C * nw) {
    double a = 0.0;
    for (int c = lane; c < p; c += 32) { const double x = (double)ld_cg(g + (size_t)i * p + c); a += x * x; }
    a = warp_sum(a);
    const double na = sqrt(a);
    if (lane == 0) lam[voff[lb] + i] = (T)(na - m);
    const double inv = na > 0.0 ? 1.0 / na : 0.0;
    for (int c = lane; c < p; c += 32) vt[(size_t)i * p + c] = (T)((double)ld_cg(g + (size_t)i * p + c) * inv);
  }
  if (rank == 0 && threadIdx.x == 0) {
    atomicMax(sweeps_out, sweep);
    if (sweeps_sum) atomicAdd(sweeps_sum, (unsigned long long)sweep);
    if (capped && flags) atomicOr(flags + prob_of[lb], FLAG_EIG_CAP);   // the sweep cap ended the iteration
  }
}

template <typename T, int RP> inline size_t smem_bytes(int p) { return Plan<T, RP>(p).bytes; }

// ---------------------------------------------------------------------------------------------------------
// fp32 variant on the tensor cores (mma.sync m16n8k8, 3xTF32). Same algorithm and the same fixed point as k_bjacobi;
// what changes is where the time of a block round goes (profiles/r01_bjacobi_cfg5.md: 20 % Gram + 12 % apply on FMA
// units with the tensor pipe idle, half of it in the 31 dependent rounds of the inner sweep):
//   * rows come in with cp.async (16-byte chunks, all in flight at once) instead of dependent L2 loads;
//   * Gram W = X X' (32 x 32 x p): warp w contracts its own k slice of p/16 columns with 3xTF32 mma.sync into fresh
//     accumulators (leading term a_hi b_hi apart from the two small terms, so the tensor core's truncating adder sees at
//     most 4 additions per accumulator); the 16 partial matrices are summed in fp64 in a fixed order. Only the six
//     16 x 8 tiles of the upper block triangle are formed. Shared-memory row stride = 4 mod 32 words: conflict free;
//   * apply X' = Q X (32 x 32 x p): warp w owns p/16 columns, Q's fragments stay in registers, 3xTF32, results go
//     from the accumulators straight to L2. The k slots of a fragment map to rows (2t, 2t+1) instead of (t, t+4) so that
//     the transposed reads of X are conflict free with the same stride;
//   * the pair table of the inner sweep meets the 256 CROSS pairs (one row of each block) in its first 16 rounds and
//     the pairs inside a block in the last 15: rows of one block leave every block round mutually orthogonal, so once a
//     matrix is past its first sweep the within-block rounds hold nothing above the tolerance and the round mask skips
//     them - the dependent chain of a block round is 16 rotations long instead of 31.
// Raises FLAG_EIG_CAP on the owning problem when the sweep cap ends the iteration (cdu.h, cdu_stats.flags_or).
// ---------------------------------------------------------------------------------------------------------
namespace tcv {
constexpr int RP = 32, BR = 16, NWARP = 16, LW = RP + 1, LQ = RP + 4, LP = 40;   // LP: row stride of a Gram partial

struct Plan {
  int pk, ldx;
  size_t off_part, off_w, off_w1, off_q, off_red, off_pairs, bytes;
  __host__ __device__ explicit Plan(int p) {
    pk = ((p + 127) / 128) * 128;            // every warp's k slice / column slice is a multiple of 8
    ldx = pk + 4;
    size_t o = (size_t)RP * ldx * sizeof(float);
    off_part = o; o += (size_t)NWARP * RP * LP * sizeof(float);
    off_w = o; o += (size_t)RP * LW * sizeof(float);
    off_w1 = o; o += (size_t)RP * LW * sizeof(float);
    off_q = (o + 15) & ~(size_t)15; o = off_q + (size_t)RP * LQ * sizeof(float);
    off_red = (o + 15) & ~(size_t)15; o = off_red + 64 * sizeof(double);
    off_pairs = o; o += (size_t)(RP - 1) * (RP / 2) * sizeof(int);
    bytes = o;
  }
};

__device__ __forceinline__ void split3(float a, uint32_t& hi, uint32_t& lo) {
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(hi) : "f"(a));
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(lo) : "f"(a - __uint_as_float(hi)));
}
__device__ __forceinline__ void mma_tf32(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3]) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}

// rows of blocks bi, bj -> X[0..15], X[16..31]; pad columns [p, pk) keep their zeros, rows >= p are zero filled.
__device__ __forceinline__ void load_pair(const float* __restrict__ g, int p, int bi, int bj, float* X, int ldx) {
  if ((p & 3) == 0) {
    const int nv = p >> 2;
    for (int t = threadIdx.x; t < RP * nv; t += blockDim.x) {
      const int r = t / nv, c = t - r * nv;
      const int row = (r < BR ? bi * BR + r : bj * BR + r - BR);
      float* dst = X + (size_t)r * ldx + 4 * c;
      if (row < p) cp_async16(dst, g + (size_t)row * p + 4 * c);
      else *reinterpret_cast<float4*>(dst) = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    asm volatile("cp.async.wait_group 0;" ::: "memory");
  } else {
    for (int t = threadIdx.x; t < RP * p; t += blockDim.x) {
      const int r = t / p, c = t - r * p;
      const int row = (r < BR ? bi * BR + r : bj * BR + r - BR);
      X[(size_t)r * ldx + c] = row < p ? __ldcg(g + (size_t)row * p + c) : 0.f;
    }
  }
}

// part[warp] (32 x 32, stride LP; the block (rows 16-31, columns 0-15) is NOT written: read its mirror image).
__device__ __forceinline__ void gram_mma(const float* X, int ldx, int ks, float* part) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  float accM[6][4], accS[6][4];
#pragma unroll
  for (int i = 0; i < 6; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) { accM[i][j] = 0.f; accS[i][j] = 0.f; }
  const float* xb = X + (size_t)g * ldx + warp * ks + t;
  for (int kk = 0; kk < ks; kk += 8) {
    uint32_t h[4][2], l[4][2];     // rows g + 8 a, columns t and t + 4 of this k step: A and B fragments share them
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      split3(xb[(size_t)(8 * a) * ldx + kk], h[a][0], l[a][0]);
      split3(xb[(size_t)(8 * a) * ldx + kk + 4], h[a][1], l[a][1]);
    }
    // tiles (m tile, n tile): (0,0) (0,1) (0,2) (0,3) (1,2) (1,3)
#pragma unroll
    for (int tl = 0; tl < 6; ++tl) {
      const int mt = tl < 4 ? 0 : 1, nt = tl < 4 ? tl : tl - 2;
      mma_tf32(accS[tl], l[2 * mt][0], l[2 * mt + 1][0], l[2 * mt][1], l[2 * mt + 1][1], h[nt][0], h[nt][1]);
      mma_tf32(accS[tl], h[2 * mt][0], h[2 * mt + 1][0], h[2 * mt][1], h[2 * mt + 1][1], l[nt][0], l[nt][1]);
      mma_tf32(accM[tl], h[2 * mt][0], h[2 * mt + 1][0], h[2 * mt][1], h[2 * mt + 1][1], h[nt][0], h[nt][1]);
    }
  }
  float* pw = part + (size_t)warp * RP * LP;
#pragma unroll
  for (int tl = 0; tl < 6; ++tl) {
    const int mt = tl < 4 ? 0 : 1, nt = tl < 4 ? tl : tl - 2;
    const int r0 = 16 * mt + g, c0 = 8 * nt + 2 * t;
    *reinterpret_cast<float2*>(pw + r0 * LP + c0) = make_float2(accM[tl][0] + accS[tl][0], accM[tl][1] + accS[tl][1]);
    *reinterpret_cast<float2*>(pw + (r0 + 8) * LP + c0) = make_float2(accM[tl][2] + accS[tl][2], accM[tl][3] + accS[tl][3]);
  }
}

// W = sum of the 16 partials (fp64, fixed order); returns max_{i<j} |w_ij| / sqrt(w_ii w_jj) to every thread.
__device__ __forceinline__ double gram_reduce(const float* part, float* W, double* red) {
  for (int e = threadIdx.x; e < RP * RP; e += blockDim.x) {
    const int i = e >> 5, j = e & 31;
    const int ri = (i >= 16 && j < 16) ? j : i, rj = (i >= 16 && j < 16) ? i : j;
    double a = 0.0;
#pragma unroll
    for (int w = 0; w < NWARP; ++w) a += (double)part[(size_t)w * RP * LP + ri * LP + rj];
    W[i * LW + j] = (float)a;
  }
  __syncthreads();
  double mx = 0.0;
  for (int e = threadIdx.x; e < RP * RP; e += blockDim.x) {
    const int i = e >> 5, j = e & 31;
    if (i < j) {
      const double d = (double)W[i * LW + i] * (double)W[j * LW + j];
      if (d > 0.0) mx = fmax(mx, fabs((double)W[i * LW + j]) * rsqrt(d));
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = mx;
  __syncthreads();
  mx = 0.0;
#pragma unroll
  for (int w = 0; w < NWARP; ++w) mx = fmax(mx, red[w]);
  __syncthreads();
  return mx;
}

// X' = Q X for this warp's column slice, written straight to the matrix (rows 0-15 -> block bi, 16-31 -> block bj).
__device__ __forceinline__ void apply_mma(const float* Q, const float* X, int ldx, int ns, int p, float* __restrict__ gm, int rowA, int rowB) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  uint32_t qh[2][4][4], ql[2][4][4];      // [m tile][k step][fragment register]; k slot t <-> row 2t, slot t+4 <-> row 2t+1
#pragma unroll
  for (int mt = 0; mt < 2; ++mt)
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      const float2 u = *reinterpret_cast<const float2*>(Q + (16 * mt + g) * LQ + 8 * ks + 2 * t);
      const float2 v = *reinterpret_cast<const float2*>(Q + (16 * mt + g + 8) * LQ + 8 * ks + 2 * t);
      split3(u.x, qh[mt][ks][0], ql[mt][ks][0]); split3(v.x, qh[mt][ks][1], ql[mt][ks][1]);
      split3(u.y, qh[mt][ks][2], ql[mt][ks][2]); split3(v.y, qh[mt][ks][3], ql[mt][ks][3]);
    }
  for (int n0 = warp * ns; n0 < (warp + 1) * ns; n0 += 8) {
    if (n0 >= p) break;
    float accM[2][4], accS[2][4];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) { accM[i][j] = 0.f; accS[i][j] = 0.f; }
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      uint32_t bh0, bl0, bh1, bl1;
      split3(X[(size_t)(8 * ks + 2 * t) * ldx + n0 + g], bh0, bl0);
      split3(X[(size_t)(8 * ks + 2 * t + 1) * ldx + n0 + g], bh1, bl1);
#pragma unroll
      for (int mt = 0; mt < 2; ++mt) {
        mma_tf32(accS[mt], ql[mt][ks][0], ql[mt][ks][1], ql[mt][ks][2], ql[mt][ks][3], bh0, bh1);
        mma_tf32(accS[mt], qh[mt][ks][0], qh[mt][ks][1], qh[mt][ks][2], qh[mt][ks][3], bl0, bl1);
        mma_tf32(accM[mt], qh[mt][ks][0], qh[mt][ks][1], qh[mt][ks][2], qh[mt][ks][3], bh0, bh1);
      }
    }
    const int col = n0 + 2 * t;
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
      for (int hf = 0; hf < 2; ++hf) {
        const int i = 16 * mt + g + 8 * hf;
        const int grow = i < BR ? rowA + i : rowB + (i - BR);
        if (grow < p) {
          const float v0 = accM[mt][2 * hf] + accS[mt][2 * hf], v1 = accM[mt][2 * hf + 1] + accS[mt][2 * hf + 1];
          float* dst = gm + (size_t)grow * p + col;
          if (col + 1 < p && (p & 1) == 0) __stcg(reinterpret_cast<float2*>(dst), make_float2(v0, v1));
          else { if (col < p) __stcg(dst, v0); if (col + 1 < p) __stcg(dst + 1, v1); }
        }
      }
  }
}

static __global__ void __launch_bounds__(THREADS, 1)
k_bjacobi_tc(int nblk, const int* pvec, const long long* moff, const int* voff, float* G, float* Vt, const float* mu, float* lam,
             int* rotflags, int* sweeps_out, unsigned long long* sweeps_sum, int max_sweeps, double tol, const int* prob_of,
             int* flags) {
  extern __shared__ __align__(16) unsigned char smem_bj[];
  cg::cluster_group cluster = cg::this_cluster();
  const int C = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
  const int lb = blockIdx.x / C;
  const int p = pvec[lb];
  const Plan pl(p);
  float* X = reinterpret_cast<float*>(smem_bj);
  float* part = reinterpret_cast<float*>(smem_bj + pl.off_part);
  float* W = reinterpret_cast<float*>(smem_bj + pl.off_w);
  float* W1 = reinterpret_cast<float*>(smem_bj + pl.off_w1);
  float* Q = reinterpret_cast<float*>(smem_bj + pl.off_q);
  double* red = reinterpret_cast<double*>(smem_bj + pl.off_red);
  int* pairs = reinterpret_cast<int*>(smem_bj + pl.off_pairs);
  float* g = G + moff[lb];
  int* rf = rotflags + lb * MAXSW;
  const int ldx = pl.ldx, ks = pl.pk / NWARP;
  const int NB = (p + BR - 1) / BR, NBe = (NB + 1) & ~1, NP = NBe >> 1;
  // inner pair table: rounds 0-15 cross pairs (q, 16 + (q + r) mod 16), rounds 16-30 the pairs inside each block
  for (int t = threadIdx.x; t < (RP - 1) * BR; t += blockDim.x) {
    const int r = t / BR, q = t - r * BR;
    int i, j;
    if (r < BR) { i = q; j = BR + ((q + r) & (BR - 1)); }
    else { rr_pair(r - BR, q & 7, BR, i, j); if (q >= 8) { i += BR; j += BR; } }
    pairs[t] = i | (j << 16);
  }
  for (int t = threadIdx.x; t < RP * ldx; t += blockDim.x) X[t] = 0.f;    // the pads stay zero
  __syncthreads();
  const float thresh = (float)(0.25 * tol);
  const float quad_exit = (float)sqrt(tol / (16.0 * sqrt((double)p)));
  int sweep = 0;
  bool capped = true;
  for (; sweep < max_sweeps; ++sweep) {
    for (int r = 0; r < NBe - 1; ++r) {
      for (int q = rank; q < NP; q += C) {
        int bi, bj2; rr_pair(r, q, NBe, bi, bj2);
        load_pair(g, p, bi, bj2, X, ldx);
        __syncthreads();
        gram_mma(X, ldx, ks, part);
        __syncthreads();
        const double mx = gram_reduce(part, W, red);
        if (mx > tol) {
          inner_sweep<float, RP>(W, W1, Q, thresh, pairs, reinterpret_cast<unsigned*>(red + 40));
          apply_mma(Q, X, ldx, ks, p, g, bi * BR, bj2 * BR);
          if (threadIdx.x == 0) atomicMax(reinterpret_cast<unsigned*>(rf) + sweep, __float_as_uint((float)mx));
        }
        __syncthreads();
      }
      cluster.sync();
    }
    const unsigned worst = (unsigned)__ldcg(rf + sweep);
    if (!worst) { capped = false; break; }
    if (__uint_as_float(worst) <= quad_exit) { ++sweep; capped = false; break; }
  }
  const int lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  const double m = (double)mu[lb];
  float* vt = Vt + moff[lb];
  for (int i = rank * nw + (threadIdx.x >> 5); i < p; i += C * nw) {
    double a = 0.0;
    for (int c = lane; c < p; c += 32) { const double x = (double)__ldcg(g + (size_t)i * p + c); a += x * x; }
    a = warp_sum(a);
    const double na = sqrt(a);
    if (lane == 0) lam[voff[lb] + i] = (float)(na - m);
    const double inv = na > 0.0 ? 1.0 / na : 0.0;
    for (int c = lane; c < p; c += 32) vt[(size_t)i * p + c] = (float)((double)__ldcg(g + (size_t)i * p + c) * inv);
  }
  if (rank == 0 && threadIdx.x == 0) {
    atomicMax(sweeps_out, sweep);
    if (sweeps_sum) atomicAdd(sweeps_sum, (unsigned long long)sweep);
    if (capped && flags) atomicOr(flags + prob_of[lb], FLAG_EIG_CAP);
  }
}

inline size_t smem_bytes(int p) { return Plan(p).bytes; }
}  // namespace tcv


}  // namespace bj
}  // namespace cdu

// psd_bjacobi.cuh - eigendecomposition of the large PSD blocks: blocked one-sided Jacobi in shared memory.
//
// One-sided (Hestenes) Jacobi on the shifted matrix: the rows g_i = v_i' (S + mu I) of G, for an orthonormal set {v_i},
// are made mutually orthogonal by plane rotations; then v_i = g_i / ||g_i|| are eigenvectors of S (Eq. 7,
// L102: only U max(L,0) U' is compared with the oracle, never U - reading A15). The v_i are never formed: rotating
// the rows of G rotates them implicitly, so only G is carried. The schedule is built for the SM, not for L2 latency:
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
          int* sweeps_out, unsigned long long* sweeps_sum, int max_sweeps, double tol, const int* prob_of, int* flags,
          const int* need) {
  constexpr int BR = RP / 2, LQ = RP + 4;
  extern __shared__ __align__(16) unsigned char smem_bj[];
  cg::cluster_group cluster = cg::this_cluster();
  const int C = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
  const int lb = blockIdx.x / C;
  if (need && !need[lb]) return;                 // the whole cluster leaves
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
// fp32 kernel on the tensor cores (mma.sync m16n8k8, 3xTF32). Same algorithm and fixed point as k_bjacobi above:
//   * rows come in with cp.async (16-byte chunks, all in flight at once);
//   * Gram W = X X' (32 x 32 x p): warp w contracts its own k slice of p/16 columns with 3xTF32 mma.sync into fresh
//     accumulators; only the six 16 x 8 tiles of the upper block triangle are formed. Row stride = 4 mod 32 words:
//     conflict free;
//   * apply X' = X + (Q - I) X (32 x 32 x p): warp w owns p/16 columns, the fragments of Q - I stay in registers; the k
//     slots of a fragment map to rows (2t, 2t+1) so that the transposed reads of X are conflict free with the same stride;
//   * the pair table of the inner sweep meets the 256 CROSS pairs (one row of each block) in its first 16 rounds and the
//     pairs inside a block in the last 15: rows of one block leave every block round mutually orthogonal, so past the
//     first sweep the within-block rounds hold nothing above the tolerance and the round mask skips them.
// Phase by phase (cycle counts per block pair at p = 512 in profiles/r02_bjacobi_phases.md):
//   * no thread-block clusters. A 16-CTA cluster needs 16 free SMs inside one GPC and only 7 such clusters fit a B200,
//     so a batch of 8 matrices ran in two waves. The CTAs of a matrix now meet at a counter in global memory
//     (cooperative launch guarantees co-residency): any 16 SMs serve, all 8 matrices run at once;
//   * Gram reduction: float2 loads of the 16 partials, convergence ratio as w_ij^2 / (w_ii w_jj) in fp32 (no fp64
//     rsqrt), warp maxima by redux.sync; the same pass builds the mask of inner rounds that hold a pair above the
//     tolerance;
//   * inner sweep: 256 threads own the 256 2x2 blocks (row pair a, column pair b) of W, 256 threads the row pairs of Q.
//     Every thread derives the rotations it needs from the current W itself (two rsqrt in the dependent chain), cross
//     rounds index arithmetically (no table load), rotations are applied as (cos, sin) (depth 2 instead of 4), W is
//     double buffered: one barrier per round. (cos, sin) come from approximate rsqrt and are renormalised by
//     one Newton step: a pair of rows scaled differently from the others would not rotate into eigenvectors.
// ---------------------------------------------------------------------------------------------------------
namespace tcw {
#ifdef CDU_BJ_TIMING
__device__ long long g_bj_tim[256 * 16];
#define BW_T0() long long bw_t0_ = clock64()
#define BW_T(i) do { __syncthreads(); if (threadIdx.x == 0) { asm volatile("membar.cta;" ::: "memory"); const long long t_ = clock64(); g_bj_tim[blockIdx.x * 16 + (i)] += t_ - bw_t0_; bw_t0_ = t_; } else bw_t0_ = 0; } while (0)
#define BW_CNT(i, n) do { if (threadIdx.x == 0) g_bj_tim[blockIdx.x * 16 + (i)] += (n); } while (0)
#else
#define BW_T0() do {} while (0)
#define BW_T(i) do {} while (0)
#define BW_CNT(i, n) do {} while (0)
#endif
constexpr int RP = 32, BR = 16, NWARP = 16, LW = 48, LQ = 40, LP = 40;

struct Plan {
  int pk, ldx;
  size_t off_part, off_w, off_w1, off_q, off_red, off_rtab, off_ptab, bytes;
  __host__ __device__ explicit Plan(int p) {
    pk = ((p + 127) / 128) * 128;            // every warp's k slice / column slice is a multiple of 8
    ldx = pk + 4;
    size_t o = (size_t)RP * ldx * sizeof(float);
    off_part = o; o += (size_t)NWARP * RP * LP * sizeof(float);
    off_w = o; o += (size_t)RP * LW * sizeof(float);
    off_w1 = o; o += (size_t)RP * LW * sizeof(float);
    off_q = o; o += (size_t)RP * LQ * sizeof(float);
    off_red = o; o += 64 * sizeof(unsigned);
    off_rtab = o; o += (size_t)RP * RP;                       // inner round of every pair (i, j)
    off_ptab = o; o += (size_t)(BR - 1) * BR * 2;             // pairs of the within-block rounds 16..30
    bytes = (o + 15) & ~(size_t)15;
  }
};

// rows 0-15 against 16-31 in rounds 0-15, the pairs inside each block in rounds 16-30
__device__ __forceinline__ void inner_pair(int r, int q, const unsigned char* ptab, int& i, int& j) {
  if (r < BR) { i = q; j = BR + ((q + r) & (BR - 1)); }
  else { const int o = ((r - BR) * BR + q) * 2; i = ptab[o]; j = ptab[o + 1]; }
}

// W = sum of the 16 partials (fixed order). Returns max_{i<j} w_ij^2 / (w_ii w_jj) and the mask of inner rounds that
// hold a pair with that ratio above lim2.
__device__ __forceinline__ float gram_reduce(const float* part, float* W, unsigned* red, const unsigned char* rtab, float lim2,
                                             unsigned& active, bool cross_only = false) {
  const int tid = threadIdx.x;
  if (tid < 384) {     // (i, j pair): rows 0-15 all 16 column pairs, rows 16-31 column pairs 8-15 (the rest by symmetry)
    int i, jp;
    if (tid < 256) { i = tid >> 4; jp = tid & 15; } else { i = 16 + ((tid - 256) >> 3); jp = 8 + ((tid - 256) & 7); }
    const float* src = part + i * LP + 2 * jp;
    float2 a = make_float2(0.f, 0.f);
#pragma unroll
    for (int w = 0; w < NWARP; ++w) { const float2 v = *reinterpret_cast<const float2*>(src + (size_t)w * RP * LP); a.x += v.x; a.y += v.y; }
    const int j = 2 * jp;
    if (cross_only && ((i < 16) == (j < 16))) {      // inside a diagonal block only the diagonal entry was formed (gram_mma_cross)
      a.x = (j == i) ? a.x : 0.f; a.y = (j + 1 == i) ? a.y : 0.f;
    }
    W[i * LW + j] = a.x; W[i * LW + j + 1] = a.y;
    if (i < 16 && j >= 16) { W[j * LW + i] = a.x; W[(j + 1) * LW + i] = a.y; }
  }
  __syncthreads();
  float mx = 0.f; unsigned m = 0u;
#pragma unroll
  for (int e = tid; e < RP * RP; e += 512) {
    const int i = e >> 5, j = e & 31;
    if (i < j) {
      const float c = W[i * LW + j], d = W[i * LW + i] * W[j * LW + j];
      if (d > 0.f) {
        const float r2 = __fdividef(c * c, d);
        mx = fmaxf(mx, r2);
        if (r2 > lim2) m |= 1u << rtab[e];
      }
    }
  }
  const unsigned mb = __reduce_max_sync(0xffffffffu, __float_as_uint(mx));   // non-negative floats order as unsigned
  m = __reduce_or_sync(0xffffffffu, m);
  if ((tid & 31) == 0) { red[tid >> 5] = mb; red[16 + (tid >> 5)] = m; }
  __syncthreads();
  unsigned mm = 0u, am = 0u;
#pragma unroll
  for (int w = 0; w < NWARP; ++w) { mm = max(mm, red[w]); am |= red[16 + w]; }
  active = am;
  return __uint_as_float(mm);
}

// (cos, sin) of the rotation that annihilates w_ij, identity when w_ij^2 <= thr2 w_ii w_jj.
__device__ __forceinline__ void rot_cs(float a, float b, float c, float thr2, float& cs, float& sn) {
  // branch free, so that the two rotations a thread needs overlap; the select discards the NaN of c = d = 0
  const float d = b - a;
  const float rh = rsqrt_approx(fmaf(d, d, 4.f * c * c));      // tan 2phi = 2c / d, |phi| <= pi/4
  const float cq = fmaf(0.5f * fabsf(d), rh, 0.5f);            // cos^2 phi = (1 + cos 2phi) / 2
  const float rc = rsqrt_approx(cq);
  const bool rot = c * c > thr2 * a * b;
  const float c0 = cq * rc, s0 = copysignf(1.f, d) * c * rh * rc;   // sin phi = sin 2phi / (2 cos phi)
  const float f = fmaf(-0.5f, fmaf(c0, c0, s0 * s0), 1.5f);      // one Newton step to cos^2 + sin^2 = 1: the approximate rsqrt
  cs = rot ? c0 * f : 1.f;                                         // leaves 1 + O(1e-7), and rows of one pair that carry different
  sn = rot ? s0 * f : 0.f;                                         // scale factors would no longer rotate into eigenvectors
}

// a = hi + lo, both exactly representable in TF32 (round to nearest, ties away: add half an ulp, clear the low 13 bits).
__device__ __forceinline__ void split_fast(float a, uint32_t& hi, uint32_t& lo) {
  hi = (__float_as_uint(a) + 0x1000u) & 0xffffe000u;
  lo = (__float_as_uint(a - __uint_as_float(hi)) + 0x1000u) & 0xffffe000u;
}

// One cyclic sweep of two-sided Jacobi on W (rounds outside `active` skipped), Q = product of the rotations
// (row i of Q: the combination of old rows that makes new row i). Warps 0-7 work, one named barrier per round among
// them; thread (a, b) owns the 2x2 block (row pair a, column pair b) of W and columns 2b, 2b+1 of the row pair a of Q.
// It derives BOTH of its rotations (pair a for the rows, pair b for the columns) from the current W itself: 32-fold
// redundant arithmetic, but no shuffle and every load of a round issues at its top, and the round is a dependent chain
// (load, rotation, update, store, barrier: 440 cycles against 530 with one rotation per thread and shuffles, measured).
// The pair indices of the next active round are fetched while the rotations are computed. Ends with a CTA barrier.
__device__ __forceinline__ void inner_sweep(float* W0, float* W1, float* Q, float thr2, unsigned active, const unsigned char* ptab) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  for (int e = tid; e < RP * RP; e += 512) { const int i = e >> 5, j = e & 31; Q[i * LQ + j] = (i == j) ? 1.f : 0.f; }
  __syncthreads();
  if (warp < 8) {
    const int b = lane & 15, a = 2 * warp + (lane >> 4);
    float* Wc = W0; float* Wn = W1;
    int r = __ffs(active) - 1;           // active != 0 (caller)
    int ib, jb, ia, ja;
    inner_pair(r, b, ptab, ib, jb); inner_pair(r, a, ptab, ia, ja);
    while (r >= 0) {
      const unsigned rest = active & ~((2u << r) - 1u);
      const int rn = rest ? __ffs(rest) - 1 : -1;
      const float bii = Wc[ib * LW + ib], bjj = Wc[jb * LW + jb], bij = Wc[ib * LW + jb];
      const float aii = Wc[ia * LW + ia], ajj = Wc[ja * LW + ja], aij = Wc[ia * LW + ja];
      const float p0 = Wc[ia * LW + ib], q0 = Wc[ia * LW + jb], r0 = Wc[ja * LW + ib], s0 = Wc[ja * LW + jb];
      float2* xi = reinterpret_cast<float2*>(Q + ia * LQ + 2 * b); float2* xj = reinterpret_cast<float2*>(Q + ja * LQ + 2 * b);
      const float2 x = *xi, y = *xj;
      int ibn = 0, jbn = 0, ian = 0, jan = 0;
      if (rn >= 0) { inner_pair(rn, b, ptab, ibn, jbn); inner_pair(rn, a, ptab, ian, jan); }
      float csB, snB, csA, snA;
      rot_cs(bii, bjj, bij, thr2, csB, snB);
      rot_cs(aii, ajj, aij, thr2, csA, snA);
      const float p1 = csA * p0 - snA * r0, r1 = snA * p0 + csA * r0, q1 = csA * q0 - snA * s0, s1 = snA * q0 + csA * s0;
      Wn[ia * LW + ib] = csB * p1 - snB * q1; Wn[ia * LW + jb] = snB * p1 + csB * q1;
      Wn[ja * LW + ib] = csB * r1 - snB * s1; Wn[ja * LW + jb] = snB * r1 + csB * s1;
      *xi = make_float2(csA * x.x - snA * y.x, csA * x.y - snA * y.y);
      *xj = make_float2(snA * x.x + csA * y.x, snA * x.y + csA * y.y);
      asm volatile("bar.sync 1, 256;" ::: "memory");
      float* t2 = Wc; Wc = Wn; Wn = t2;
      r = rn; ib = ibn; jb = jbn; ia = ian; ja = jan;
    }
  }
  __syncthreads();
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
      split_fast(xb[(size_t)(8 * a) * ldx + kk], h[a][0], l[a][0]);
      split_fast(xb[(size_t)(8 * a) * ldx + kk + 4], h[a][1], l[a][1]);
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


// X' = X + E X, E = Q - I (hi / lo parts pre-split in shared memory, fragment order), for this warp's column slice, in place. The tensor core adds into its accumulators with truncation; on Q X that
// is a bias of ~1e-7 per block round on every row, which BPTT through 200 iterations amplified to wrong gradients (measured:
// cfg5 gradient error 0.48). On E X it is 1e-7 of the correction only, and the correction is small once the sweeps converge.
// The cross block only (rows 0-15 against rows 16-31: tiles (0,2), (0,3)) and the 32 diagonal entries, for the visits that
// rotate cross pairs only (block-cyclic ordering, see the kernel): a third of the mma of gram_mma. The diagonal entries are
// plain fp32 sums of squares of the fragments the thread holds anyway (lanes t = 0..3 of a row group add by shuffle); the
// entries inside the two diagonal blocks are NOT written (gram_reduce takes them as zero: they are of second order after the
// block's round-0 visit, and an error there only perturbs the angles of later inner rounds, not the orthogonality of Q).
__device__ __forceinline__ void gram_mma_cross(const float* X, int ldx, int ks, float* part) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  float accM[2][4], accS[2][4], sq[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) { accM[i][j] = 0.f; accS[i][j] = 0.f; }
  const float* xb = X + (size_t)g * ldx + warp * ks + t;
  for (int kk = 0; kk < ks; kk += 8) {
    uint32_t h[4][2], l[4][2];
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      const float x0 = xb[(size_t)(8 * a) * ldx + kk], x1 = xb[(size_t)(8 * a) * ldx + kk + 4];
      sq[a] = fmaf(x0, x0, fmaf(x1, x1, sq[a]));
      split_fast(x0, h[a][0], l[a][0]);
      split_fast(x1, h[a][1], l[a][1]);
    }
#pragma unroll
    for (int n = 0; n < 2; ++n) {      // m tile 0 (rows g, g + 8), n tiles 2, 3 (rows 16 + g, 24 + g)
      mma_tf32(accS[n], l[0][0], l[1][0], l[0][1], l[1][1], h[2 + n][0], h[2 + n][1]);
      mma_tf32(accS[n], h[0][0], h[1][0], h[0][1], h[1][1], l[2 + n][0], l[2 + n][1]);
      mma_tf32(accM[n], h[0][0], h[1][0], h[0][1], h[1][1], h[2 + n][0], h[2 + n][1]);
    }
  }
  float* pw = part + (size_t)warp * RP * LP;
#pragma unroll
  for (int n = 0; n < 2; ++n) {
    const int c0 = 8 * (2 + n) + 2 * t;
    *reinterpret_cast<float2*>(pw + g * LP + c0) = make_float2(accM[n][0] + accS[n][0], accM[n][1] + accS[n][1]);
    *reinterpret_cast<float2*>(pw + (g + 8) * LP + c0) = make_float2(accM[n][2] + accS[n][2], accM[n][3] + accS[n][3]);
  }
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    float v = sq[a];
    v += __shfl_xor_sync(0xffffffffu, v, 1);
    v += __shfl_xor_sync(0xffffffffu, v, 2);
    if (t == 0) pw[(g + 8 * a) * LP + g + 8 * a] = v;
  }
}

// Element (i, k) of E -> its place in the fragment-ordered copies [m tile][k step][lane][4] that apply_mma reads: a thread's
// four A registers of one mma are one 16-byte piece, a warp's load is 512 contiguous bytes (16 conflict-free LDS.128 per
// thread instead of 32 LDS.64 that cost 900 cycles more per visit, measured).
__device__ __forceinline__ int frag_pos(int i, int k) {
  const int mt = i >> 4, r = i & 15, g = r & 7, hf = r >> 3, ks = k >> 3, kk = k & 7, t = kk >> 1, wh = kk & 1;
  return ((mt * 4 + ks) * 32 + 4 * g + t) * 4 + hf + 2 * wh;
}
__device__ __forceinline__ void apply_mma(const uint32_t* Qh, const uint32_t* Ql, float* X, int ldx, int ns, int p) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  uint32_t qh[2][4][4], ql[2][4][4];      // [m tile][k step][fragment register]; k slot t <-> row 2t, slot t+4 <-> row 2t+1
#pragma unroll
  for (int mt = 0; mt < 2; ++mt)
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      const uint4 h = *reinterpret_cast<const uint4*>(Qh + ((mt * 4 + ks) * 32 + lane) * 4);
      const uint4 l = *reinterpret_cast<const uint4*>(Ql + ((mt * 4 + ks) * 32 + lane) * 4);
      qh[mt][ks][0] = h.x; qh[mt][ks][1] = h.y; qh[mt][ks][2] = h.z; qh[mt][ks][3] = h.w;
      ql[mt][ks][0] = l.x; ql[mt][ks][1] = l.y; ql[mt][ks][2] = l.z; ql[mt][ks][3] = l.w;
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
      split_fast(X[(size_t)(8 * ks + 2 * t) * ldx + n0 + g], bh0, bl0);
      split_fast(X[(size_t)(8 * ks + 2 * t + 1) * ldx + n0 + g], bh1, bl1);
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
        float2* xp = reinterpret_cast<float2*>(X + (size_t)i * ldx + col);       // X' = X + (Q - I) X, in place: this warp alone
        const float2 x0 = *xp;                                                   // reads and writes its columns
        *xp = make_float2(x0.x + (accM[mt][2 * hf] + accS[mt][2 * hf]), x0.y + (accM[mt][2 * hf + 1] + accS[mt][2 * hf + 1]));
      }
  }
}

// rows of X -> rows of blocks bi, bj of the matrix (coalesced 16-byte stores)
__device__ __forceinline__ void store_pair(float* __restrict__ g, int p, int bi, int bj, const float* X, int ldx) {
  if ((p & 3) == 0) {
    const int nv = p >> 2;
    for (int t = threadIdx.x; t < RP * nv; t += blockDim.x) {
      const int r = t / nv, c = t - r * nv;
      const int row = (r < BR ? bi * BR + r : bj * BR + r - BR);
      if (row < p) __stcg(reinterpret_cast<float4*>(g + (size_t)row * p) + c, *reinterpret_cast<const float4*>(X + (size_t)r * ldx + 4 * c));
    }
  } else {
    for (int t = threadIdx.x; t < RP * p; t += blockDim.x) {
      const int r = t / p, c = t - r * p;
      const int row = (r < BR ? bi * BR + r : bj * BR + r - BR);
      if (row < p) __stcg(g + (size_t)row * p + c, X[(size_t)r * ldx + c]);
    }
  }
}

// Per-warp forms (p % 4 == 0): warp w owns the columns [w ks, (w + 1) ks) of the 32 rows from the load to the store - its k
// slice of the Gram product and its column slice of the apply are the same columns - so no CTA barrier stands between the
// load and the Gram product or between the apply and the store (measured: load phase 2.3k -> 1.4k cycles per block pair,
// 1.75 -> 1.65 ms per batch of 8 at p = 512). A lane moves 16-byte pieces; at p = 512 eight lanes cover one 128-byte row segment.
template <int NPC>   // NPC = ks / 4 16-byte pieces per row of the slice (compile time: the 32 x NPC pieces unroll into NPC instructions per lane)
__device__ __forceinline__ void load_slice_t(const float* __restrict__ g, int p, int bi, int bj, float* X, int ldx) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
  for (int it = 0; it < NPC; ++it) {
    const int t = lane + 32 * it, r = t / NPC, c = warp * (4 * NPC) + 4 * (t - r * NPC);
    if (c < p) {                                                                  // pad columns keep their zeros
      const int row = (r < BR ? bi * BR + r : bj * BR + r - BR);
      float* dst = X + (size_t)r * ldx + c;
      if (row < p) cp_async16(dst, g + (size_t)row * p + c);
      else *reinterpret_cast<float4*>(dst) = make_float4(0.f, 0.f, 0.f, 0.f);
    }
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncwarp();
}
template <int NPC>
__device__ __forceinline__ void store_slice_t(float* __restrict__ g, int p, int bi, int bj, const float* X, int ldx) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncwarp();
#pragma unroll
  for (int it = 0; it < NPC; ++it) {
    const int t = lane + 32 * it, r = t / NPC, c = warp * (4 * NPC) + 4 * (t - r * NPC);
    const int row = (r < BR ? bi * BR + r : bj * BR + r - BR);
    if (c < p && row < p) __stcg(reinterpret_cast<float4*>(g + (size_t)row * p + c), *reinterpret_cast<const float4*>(X + (size_t)r * ldx + c));
  }
}
// The C CTAs of one matrix meet here once per round of blocks: everything they stored before is visible to all of
// them after. ctr counts arrivals since the launch (zeroed by the host), gen the barriers this CTA has passed.
__device__ __forceinline__ void matrix_barrier(unsigned* ctr, unsigned& gen, int C) {
  __syncthreads();
  if (threadIdx.x == 0) {
    ++gen;
    if (C > 1) {
      __threadfence();
      atomicAdd(ctr, 1u);
      const unsigned target = gen * (unsigned)C;
      unsigned v;
      do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory"); } while (v < target);
    }
  }
  __syncthreads();
}

// grid = nmat * C CTAs, launched cooperatively (all co-resident); CTA blockIdx.x works on matrix lb0 + blockIdx.x / C
// as member blockIdx.x % C: block pairs rank, rank + C, ... of every round. G, Vt, mu, lam, rotflags as k_bjacobi.
static __global__ void __launch_bounds__(THREADS, 1)
k_bjacobi_tc2(int lb0, int C, const int* pvec, const long long* moff, const int* voff, float* G, float* Vt, const float* mu, float* lam,
              int* rotflags, int* sweeps_out, unsigned long long* sweeps_sum, int max_sweeps, double tol, const int* prob_of,
              int* flags, unsigned* bar, const int* need) {
  extern __shared__ __align__(16) unsigned char smem_bj[];
  const int rank = blockIdx.x % C, lb = lb0 + blockIdx.x / C;
  if (need && !need[lb]) return;                 // all CTAs of the matrix leave
  const int p = pvec[lb];
  const Plan pl(p);
  float* X = reinterpret_cast<float*>(smem_bj);
  float* part = reinterpret_cast<float*>(smem_bj + pl.off_part);
  float* W = reinterpret_cast<float*>(smem_bj + pl.off_w);
  float* W1 = reinterpret_cast<float*>(smem_bj + pl.off_w1);
  float* Q = reinterpret_cast<float*>(smem_bj + pl.off_q);
  unsigned* red = reinterpret_cast<unsigned*>(smem_bj + pl.off_red);
  unsigned char* rtab = smem_bj + pl.off_rtab;
  unsigned char* ptab = smem_bj + pl.off_ptab;
  float* g = G + moff[lb];
  int* rf = rotflags + lb * MAXSW;
  unsigned* ctr = bar + lb;
  unsigned gen = 0;
  const int ldx = pl.ldx, ks = pl.pk / NWARP;
  const int NB = (p + BR - 1) / BR, NBe = (NB + 1) & ~1, NP = NBe >> 1;
  for (int t = threadIdx.x; t < (BR - 1) * BR; t += blockDim.x) {     // within-block rounds: 8 pairs in each of the two blocks
    const int r = t / BR, q = t - r * BR;
    int i, j;
    rr_pair(r, q & 7, BR, i, j);
    if (q >= 8) { i += BR; j += BR; }
    ptab[2 * t] = (unsigned char)i; ptab[2 * t + 1] = (unsigned char)j;
    rtab[i * RP + j] = (unsigned char)(BR + r);
  }
  for (int t = threadIdx.x; t < BR * BR; t += blockDim.x) {           // cross rounds
    const int i = t >> 4, j = BR + (t & 15);
    rtab[i * RP + j] = (unsigned char)((j - BR - i) & (BR - 1));
  }
  for (int t = threadIdx.x; t < RP * ldx; t += blockDim.x) X[t] = 0.f;    // the pads stay zero
  __syncthreads();
  const bool sliced = (p & 3) == 0 && ks == 32;     // 384 < p <= 512; other widths: a run-time piece count does not unroll and was slower than load_pair / store_pair, one instantiation per width made the kernel spill
  const float thr = (float)(0.25 * tol), thr2 = thr * thr, lim2 = (float)(tol * tol);
  const float quad_exit = (float)sqrt(tol / (16.0 * sqrt((double)p)));
  int sweep = 0;
  bool capped = true;
  bool small_rot = false;      // the previous sweep met no cosine above 0.1: what cross rotations leave inside a block is negligible
  for (; sweep < max_sweeps; ++sweep) {
    for (int r = 0; r < NBe - 1; ++r) {
      for (int q = rank; q < NP; q += C) {
        int bi, bj2; rr_pair(r, q, NBe, bi, bj2);
        BW_T0();
        if (sliced) load_slice_t<8>(g, p, bi, bj2, X, ldx);
        else { load_pair(g, p, bi, bj2, X, ldx); __syncthreads(); }
        BW_T(0);
        const bool cross_only = r > 0 && small_rot;
        if (cross_only) gram_mma_cross(X, ldx, ks, part); else gram_mma(X, ldx, ks, part);
        __syncthreads();
        BW_T(1);
        unsigned active;
        const float mx2 = gram_reduce(part, W, red, rtab, lim2, active, cross_only);
        // block-cyclic ordering: the pairs inside a block are rotated at the block's visit of round 0 (every block has one), the
        // other 30 visits of a sweep rotate the 256 cross pairs only; what those leave inside a block is of second order
        if (r > 0) active &= 0xffffu;
        BW_T(2);
        if (active) {
          inner_sweep(W, W1, Q, thr2, active, ptab);
          BW_T(3);
          uint32_t* Qh = reinterpret_cast<uint32_t*>(part); uint32_t* Ql = Qh + RP * LQ;    // the Gram partials are spent
          for (int e = threadIdx.x; e < RP * RP; e += 512) { const int i = e >> 5, k = e & 31, o = frag_pos(i, k); split_fast(Q[i * LQ + k] - (i == k ? 1.f : 0.f), Qh[o], Ql[o]); }
          __syncthreads();
          BW_T(9);
          apply_mma(Qh, Ql, X, ldx, ks, p);
          if (sliced) store_slice_t<8>(g, p, bi, bj2, X, ldx);
          else { __syncthreads(); store_pair(g, p, bi, bj2, X, ldx); }
          BW_T(10);
          if (threadIdx.x == 0) atomicMax(reinterpret_cast<unsigned*>(rf) + sweep, __float_as_uint(sqrtf(mx2)));
          BW_CNT(7, 1); BW_CNT(8, __popc(active));
        }
        __syncthreads();
        BW_T(4);
        BW_CNT(6, 1);
      }
      BW_T0();
      matrix_barrier(ctr, gen, C);
      BW_T(5);
      // first sweep: round 0 has shown every block once (a thirty-first of the pairs); if no cosine there exceeded 0.03 the
      // rotations of this sweep are small already (a good warm start) and the other rounds form the cross block only
      if (sweep == 0 && r == 0) small_rot = __uint_as_float((unsigned)__ldcg(rf)) <= 0.03f;
    }
    const unsigned worst = (unsigned)__ldcg(rf + sweep);     // largest |w_ij| / sqrt(w_ii w_jj) any pair showed in this sweep
    small_rot = __uint_as_float(worst) <= 0.1f;
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
}  // namespace tcw


}  // namespace bj
}  // namespace cdu

// psd_large.cuh - PSD projection / Dalecki-Krein VJP for blocks too large for one CTA's shared memory.
//
// Eigendecomposition: one-sided (Hestenes) Jacobi on the shifted matrix S + mu I >= 0, one thread-block
// cluster per matrix, one warp per column pair, columns contiguous in memory (coalesced, L2 resident),
// rounds separated by cluster barriers. On convergence the columns g_i = (S + mu I) v_i are orthogonal, so
// v_i are eigenvectors and lambda_i = ||g_i|| - mu. Only Pi(S) and the DK products are compared with the
// oracle, never U (any orthonormal basis inside an eigenvalue cluster is valid).
// Rebuild U max(L,0) U' (Eq. 7) and the four DK products (Eq. 9) are dense p x p x p GEMMs:
// fp32/fp64 FMA kernel here, tcgen05 3xTF32 kernel in gemm_tc.cuh.
// Eigenvectors are stored as ROWS (Vt[i][:] = v_i).
#pragma once
#include <cooperative_groups.h>
#include "common.cuh"
#include "psd_small.cuh"

namespace cdu {
namespace cg = cooperative_groups;

struct LargeTab {
  int nblk;              // number of large blocks
  const int* gblk;       // index into the global PSD table
  const long long* moff; // offset of the block's p x p scratch matrices (elements)
  const int* voff;       // offset of the block's length-p scratch vectors
  const int* pvec;       // order of each large block
  const long long* soff; // offset of the block's svec in the engine's own svec buffers
  int pmax;
};

// G = smat(v [+ scale v2]) + mu I; optionally Vt = I and an unshifted copy. The shift mu >= ||S||_2 makes G >= 0:
//   shift = 0: mu = 0;   shift = 1: mu = ||S||_F (svec is an isometry, so this is ||svec||_2);
//   shift = 2: warm call - Weyl's inequality against the previous matrix of this block, whose svec is kept in wprev
//              and whose largest |eigenvalue| is lmax: ||S||_2 <= lmax + ||S - S_prev||_F. mu = 1.5 x that bound
//              (capped by ||S||_F): between ADMM iterates the difference is small, so mu ~ 1.5 ||S||_2 instead of
//              ~ sqrt(p) ||S||_2, and the rounding error of the Jacobi sweeps (eps (mu + ||S||_2)) shrinks with it.
// shift >= 1 also refreshes wprev.
constexpr int LARGE_NCH = 144;  // CTAs per block in the chunked glue kernels (one 32 x 32 tile each up to order 512: these kernels are latency bound, so many small CTAs)

// Chunked over gridDim.x CTAs per block (blockIdx.y = block). The reductions (||svec||^2, ||svec - wprev||^2) go
// through per-chunk partials in `scr` ([nblk][LARGE_NCH][2] doubles + one ticket per block in `tick`); the last CTA
// to finish sums them in chunk order (deterministic), sets mu and adds it to the diagonal.
template <typename T>
__global__ void __launch_bounds__(256) k_large_smat(PsdTab tab, LargeTab lt, const double* v, const double* v2,
                                                    Hyper<T> H, int k, int use_rho_scale, int shift, T* G, T* Vt, T* mu,
                                                    double* wprev, const T* lmax, T* Splain, double* scr, unsigned* tick, int* flags,
                                                    const int* need) {
  __shared__ double sh[64];
  __shared__ unsigned last;
  if (need && !need[blockIdx.y]) return;        // second ("polish") pass: only the blocks whose first pass ran on a wide shift
  const int lb = blockIdx.y, blk = lt.gblk[lb], nch = gridDim.x, ch = blockIdx.x;
  const int p = tab.p[blk];
  const long long row0 = tab.row0[blk];
  const double sc = use_rho_scale ? H.rho_blk(k, tab.prob[blk], row0) : 0.0;
  T* g = G + lt.moff[lb];
  const double* a = v + row0;
  const double* a2 = v2 ? v2 + row0 : nullptr;
  double* wp = (wprev && shift) ? wprev + lt.soff[lb] : nullptr;
  // 32 x 32 tiles of the lower triangle (tile row bi >= tile column bj): the svec entries of matrix row R, columns
  // Cc <= R are contiguous (idx = R (R + 1) / 2 + Cc), so reads are coalesced along Cc; the tile and its mirror image
  // are written from shared memory, both coalesced.
  __shared__ T tile[32][33];
  const int ntr = (p + 31) >> 5, ntiles = ntr * (ntr + 1) / 2;
  const int lane = threadIdx.x & 31, wy = threadIdx.x >> 5, nwy = blockDim.x >> 5;
  double acc[2] = {0.0, 0.0};
  for (int tl = ch; tl < ntiles; tl += nch) {
    int bi = (int)((sqrt(8.0 * tl + 1.0) - 1.0) * 0.5);
    while (bi * (bi + 1) / 2 > tl) --bi;
    while ((bi + 1) * (bi + 2) / 2 <= tl) ++bi;
    const int bj = tl - bi * (bi + 1) / 2;
    const int Cc = bj * 32 + lane;
    for (int rr = wy; rr < 32; rr += nwy) {
      const int R = bi * 32 + rr;
      T val = (T)0;
      if (R < p && Cc < p && Cc <= R) {
        const int idx = svec_idx(Cc, R);
        double x = a[idx];
        if (a2) x += sc * a2[idx];
        acc[0] += x * x;
        if (wp) { const double d = x - wp[idx]; acc[1] += d * d; wp[idx] = x; }
        val = (T)(R == Cc ? x : x * 0.70710678118654752440);
      }
      tile[rr][lane] = val;
    }
    __syncthreads();
    for (int rr = wy; rr < 32; rr += nwy) {
      const int R = bi * 32 + rr;
      if (R < p && Cc < p && (bi != bj || lane <= rr)) {
        const long long t = (long long)R * p + Cc;
        const T val = tile[rr][lane];
        g[t] = val;
        if (Splain) Splain[lt.moff[lb] + t] = val;
        if (Vt) Vt[lt.moff[lb] + t] = (R == Cc) ? (T)1 : (T)0;
      }
      // mirror image: element (row Cm, column Rm) = tile[lane][rr] with Rm = bi * 32 + lane, Cm = bj * 32 + rr
      const int Rm = bi * 32 + lane, Cm = bj * 32 + rr;
      if (Rm < p && Cm < p && (bi != bj ? true : rr < lane)) {
        const long long t = (long long)Cm * p + Rm;
        const T val = tile[lane][rr];
        g[t] = val;
        if (Splain) Splain[lt.moff[lb] + t] = val;
        if (Vt) Vt[lt.moff[lb] + t] = (T)0;
      }
    }
    __syncthreads();
  }
  if (!shift) return;
  block_sum<2>(acc, sh);
  if (threadIdx.x == 0) {
    scr[((size_t)lb * LARGE_NCH + ch) * 2] = acc[0]; scr[((size_t)lb * LARGE_NCH + ch) * 2 + 1] = acc[1];
    __threadfence();
    last = (atomicAdd(tick + lb, 1u) == (unsigned)nch - 1) ? 1u : 0u;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  double n2 = 0.0, d2 = 0.0;
  for (int c = 0; c < nch; ++c) { n2 += __ldcg(scr + ((size_t)lb * LARGE_NCH + c) * 2); d2 += __ldcg(scr + ((size_t)lb * LARGE_NCH + c) * 2 + 1); }
  double m = sqrt(n2);
  if (!(m <= 1.7e308) && flags && threadIdx.x == 0) atomicOr(flags + tab.prob[blk], FLAG_NONFINITE);   // NaN or Inf in w
  if (shift == 2) {
    const double weyl = 1.5 * (1.02 * (double)lmax[lb] + sqrt(d2)) + 1e-30;
    if (weyl < m) m = weyl;
  }
  const T mT = (T)m;
  if (threadIdx.x == 0) { if (mu) mu[lb] = mT; tick[lb] = 0; }
  for (int i = threadIdx.x; i < p; i += blockDim.x) {
    T* d = g + (long long)i * p + i;
    *d = (T)((double)__ldcg(d) + (double)mT);
  }
}

// Batched row-major GEMM C = op(A) op(B) (p x p x p per block), FMA path. 64x64 tile, 16x16 threads, 4x4 each.
// Optional row scaling of op(A): op(A)(i,k) *= rs[k] (used for U diag(lam+) U').
template <typename T>
__global__ void __launch_bounds__(256) k_gemm_fma(int nblk, const int* pvec, const long long* moff, const int* voff, const T* A, int ta,
                                                  const T* Bm, int tb, T* Cm, const T* kscale, int kscale_relu, const int* need) {
  __shared__ T As[16][64 + 1];
  __shared__ T Bs[16][64 + 1];
  if (need && !need[blockIdx.z]) return;
  const int lb = blockIdx.z, p = pvec[lb];
  const int i0 = blockIdx.y * 64, j0 = blockIdx.x * 64;
  if (i0 >= p || j0 >= p) return;
  const T* a = A + moff[lb];
  const T* b = Bm + moff[lb];
  T* c = Cm + moff[lb];
  const T* ks = kscale ? kscale + voff[lb] : nullptr;
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  T acc[4][4] = {};
  for (int k0 = 0; k0 < p; k0 += 16) {
    for (int t = threadIdx.x; t < 16 * 64; t += 256) {
      int kk, ii;
      if (ta) { kk = t / 64; ii = t % 64; } else { ii = t / 16; kk = t % 16; }   // coalesce along the contiguous axis
      const int gi = i0 + ii, gk = k0 + kk;
      T v = (T)0;
      if (gi < p && gk < p) {
        v = ta ? a[(long long)gk * p + gi] : a[(long long)gi * p + gk];
        if (ks) { T s = ks[gk]; if (kscale_relu && !(s > (T)0)) s = (T)0; v *= s; }
      }
      As[kk][ii] = v;
    }
    for (int t = threadIdx.x; t < 16 * 64; t += 256) {
      int kk, jj;
      if (tb) { jj = t / 16; kk = t % 16; } else { kk = t / 64; jj = t % 64; }
      const int gj = j0 + jj, gk = k0 + kk;
      T v = (T)0;
      if (gj < p && gk < p) v = tb ? b[(long long)gj * p + gk] : b[(long long)gk * p + gj];
      Bs[kk][jj] = v;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < 16; ++kk) {
      T x[4], y[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) { x[u] = As[kk][ty * 4 + u]; y[u] = Bs[kk][tx * 4 + u]; }
#pragma unroll
      for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int w = 0; w < 4; ++w) acc[u][w] += x[u] * y[w];
    }
    __syncthreads();
  }
#pragma unroll
  for (int u = 0; u < 4; ++u)
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const int gi = i0 + ty * 4 + u, gj = j0 + tx * 4 + w;
      if (gi < p && gj < p) c[(long long)gi * p + gj] = acc[u][w];
    }
}

template <typename T>
__global__ void k_large_hadamard(int nblk, const int* pvec, const long long* moff, const int* voff, T* Cm, const T* lam) {
  const int lb = blockIdx.y, p = pvec[lb];
  T* c = Cm + moff[lb];
  const T* l = lam + voff[lb];
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < (long long)p * p; t += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(t / p), j = (int)(t - (long long)i * p);
    c[t] *= gamma_relu<T>(l[i], l[j]);
  }
}

// lam_i = <R_i, v_i> / <v_i, v_i> with R = Vt S (rows): Rayleigh quotients against the UNSHIFTED matrix, so the
// eigenvalues carry an error of eps ||S||, not eps mu, and do not see how the sweeps scaled the rows of G.
template <typename T>
__global__ void __launch_bounds__(256) k_large_rayleigh(const int* pvec, const long long* moff, const int* voff, const T* R,
                                                        const T* Vt, T* lam, const int* need) {
  if (need && !need[blockIdx.y]) return;
  const int lb = blockIdx.y, p = pvec[lb];
  const int lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  const T* r = R + moff[lb];
  const T* v = Vt + moff[lb];
  for (int i = blockIdx.x * nw + (threadIdx.x >> 5); i < p; i += gridDim.x * nw) {
    double a = 0.0, b = 0.0;
    for (int c = lane; c < p; c += 32) { const double x = (double)v[(long long)i * p + c]; a += (double)r[(long long)i * p + c] * x; b += x * x; }
    a = warp_sum(a); b = warp_sum(b);
    if (lane == 0) lam[voff[lb] + i] = (T)(b > 0.0 ? a / b : 0.0);
  }
}

// After an eigendecomposition: scale[k] = max(lam_k, 0) (the rebuild's column scaling) and lmax = max |lam_k|
// (the spectral radius the next warm call's shift is derived from).
template <typename T>
__global__ void __launch_bounds__(256) k_large_post(const int* pvec, const int* voff, const T* lam, T* scale, T* lmax, const T* mu,
                                                    const int* need, int* need_out) {
  __shared__ double sh[32];
  if (need && !need[blockIdx.x]) { if (need_out && threadIdx.x == 0) need_out[blockIdx.x] = 0; return; }
  const int lb = blockIdx.x, p = pvec[lb];
  const T* l = lam + voff[lb];
  double mx = 0.0;
  for (int i = threadIdx.x; i < p; i += blockDim.x) {
    const T x = l[i];
    scale[voff[lb] + i] = x > (T)0 ? x : (T)0;
    mx = fmax(mx, fabs((double)x));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = mx;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) mx = fmax(mx, sh[w]);
    lmax[lb] = (T)mx;
    // the rounding errors of the one-sided Jacobi scale with its shift: a decomposition that ran on a shift well above the
    // spectral radius (cold start: ||S||_F; early iterations: the Weyl bound with ||dS||_F) is polished by a second pass
    if (need_out) need_out[lb] = (!need && (double)mu[lb] > 3.0 * mx) ? 1 : 0;
  }
}

// svec of the symmetric part of a p x p row-major matrix M, tile by tile: 32 x 32 tiles of the lower triangle (tile row bi >=
// tile column bj). The tile and its mirror image are read coalesced into shared memory; element (R, Cc <= R) is
// 1/2 (M[R][Cc] + M[Cc][R]) (x sqrt 2 off the diagonal) and goes to f(svec index, value) with the index contiguous along the
// lanes (idx = R (R + 1) / 2 + Cc), so whatever f reads or writes at that index is coalesced too. CTA ch of nch.
template <typename T, typename F>
__device__ __forceinline__ void svec_of_sym_tiles(int p, const T* M, int ch, int nch, F f) {
  __shared__ T ta[32][33];
  __shared__ T tb[32][33];
  const int ntr = (p + 31) >> 5, ntiles = ntr * (ntr + 1) / 2;
  const int lane = threadIdx.x & 31, wy = threadIdx.x >> 5, nwy = blockDim.x >> 5;
  for (int tl = ch; tl < ntiles; tl += nch) {
    int bi = (int)((sqrt(8.0 * tl + 1.0) - 1.0) * 0.5);
    while (bi * (bi + 1) / 2 > tl) --bi;
    while ((bi + 1) * (bi + 2) / 2 <= tl) ++bi;
    const int bj = tl - bi * (bi + 1) / 2;
    for (int rr = wy; rr < 32; rr += nwy) {
      const int R = bi * 32 + rr, Cc = bj * 32 + lane;         // tile (bi, bj): row R, column Cc
      ta[rr][lane] = (R < p && Cc < p) ? M[(long long)R * p + Cc] : (T)0;
      const int Rm = bj * 32 + rr, Cm = bi * 32 + lane;        // tile (bj, bi): row Rm, column Cm
      tb[rr][lane] = (Rm < p && Cm < p) ? M[(long long)Rm * p + Cm] : (T)0;
    }
    __syncthreads();
    for (int rr = wy; rr < 32; rr += nwy) {
      const int R = bi * 32 + rr, Cc = bj * 32 + lane;
      if (R < p && Cc <= R) {
        const double v = (R == Cc) ? (double)ta[rr][lane] : 0.5 * ((double)ta[rr][lane] + (double)tb[lane][rr]) * 1.41421356237309504880;
        f(svec_idx(Cc, R), v);
      }
    }
    __syncthreads();
  }
}

// s+ = svec(Tm), y+ = rho (s+ - w); also copies Vt, lam into the checkpoint store.
template <typename T>
__global__ void __launch_bounds__(256) k_large_finish_fwd(PsdTab tab, LargeTab lt, Hyper<T> H, int k, const T* Tm,
                                                           const T* Vt, const T* lam, PsdFwdArgs A) {
  const int lb = blockIdx.y, blk = lt.gblk[lb];
  const int p = tab.p[blk];
  const long long row0 = tab.row0[blk];
  const double rho = H.rho_blk(k, tab.prob[blk], row0);
  const T* tm = Tm + lt.moff[lb];
  const double* w = A.W + row0;
  double *s1 = A.S1 + row0, *y1 = A.Y1 + row0;
  T* U = reinterpret_cast<T*>(A.Ustore) + tab.uoff[blk];
  T* L = reinterpret_cast<T*>(A.Lstore) + tab.loff[blk];
  const long long stride = (long long)gridDim.x * blockDim.x, t0 = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (U != Vt + lt.moff[lb])
    for (long long t = t0; t < (long long)p * p; t += stride) U[t] = Vt[lt.moff[lb] + t];
  svec_of_sym_tiles<T>(p, tm, (int)blockIdx.x, (int)gridDim.x, [&](int idx, double o) {
    s1[idx] = o;
    y1[idx] = rho * (o - w[idx]);
  });
  for (long long t = t0; t < p; t += stride) L[t] = lam[lt.voff[lb] + t];
}

// FULL-checkpoint backward: bring (Vt, lam) of step k from the store into the large-path scratch layout.
template <typename T>
__global__ void k_large_fetch(PsdTab tab, LargeTab lt, const T* Ustore, const T* Lstore, T* Vt, T* lam) {
  const int lb = blockIdx.y, blk = lt.gblk[lb];
  const int p = tab.p[blk];
  const T* U = Ustore + tab.uoff[blk];
  const T* L = Lstore + tab.loff[blk];
  const long long stride = (long long)gridDim.x * blockDim.x, t0 = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  for (long long t = t0; t < (long long)p * p; t += stride) Vt[lt.moff[lb] + t] = U[t];
  for (long long t = t0; t < p; t += stride) lam[lt.voff[lb] + t] = L[t];
}

// g_w = -rho g_y + svec(Out); partial dots for g_rho. Chunked like k_large_smat; the last CTA of a block sums the
// chunk partials in order into A.part.
template <typename T>
__global__ void __launch_bounds__(256) k_large_finish_bwd(PsdTab tab, LargeTab lt, Hyper<T> H, int k, const T* Out,
                                                          PsdBwdArgs A, double* scr, unsigned* tick) {
  __shared__ double sh[64];
  __shared__ unsigned last;
  const int lb = blockIdx.y, blk = lt.gblk[lb], nch = gridDim.x, ch = blockIdx.x;
  const int p = tab.p[blk];
  const long long row0 = tab.row0[blk];
  const double rho = H.rho_blk(k, tab.prob[blk], row0);
  const T* o = Out + lt.moff[lb];
  const double *w = A.W + row0, *yk = A.Yk + row0, *s1 = A.S1 + row0, *gy = A.Gy + row0;
  double* gw = A.GW + row0;
  double acc[2] = {0.0, 0.0};
  svec_of_sym_tiles<T>(p, o, ch, nch, [&](int idx, double ov) {
    const double gyv = gy[idx];
    const double g = -rho * gyv + ov;
    gw[idx] = g;
    acc[0] += gyv * (s1[idx] - w[idx]);
    acc[1] += g * yk[idx];
  });
  block_sum<2>(acc, sh);
  if (threadIdx.x == 0) {
    scr[((size_t)lb * LARGE_NCH + ch) * 2] = acc[0]; scr[((size_t)lb * LARGE_NCH + ch) * 2 + 1] = acc[1];
    __threadfence();
    last = (atomicAdd(tick + lb, 1u) == (unsigned)nch - 1) ? 1u : 0u;
  }
  __syncthreads();
  if (!last || threadIdx.x != 0) return;
  __threadfence();
  double p0 = 0.0, p1 = 0.0;
  for (int c = 0; c < nch; ++c) { p0 += __ldcg(scr + ((size_t)lb * LARGE_NCH + c) * 2); p1 += __ldcg(scr + ((size_t)lb * LARGE_NCH + c) * 2 + 1); }
  A.part[2 * blk] = p0; A.part[2 * blk + 1] = p1;
  tick[lb] = 0;
}

}  // namespace cdu

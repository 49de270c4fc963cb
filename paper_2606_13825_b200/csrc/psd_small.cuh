// psd_small.cuh - PSD-cone projection and its Dalecki-Krein VJP for blocks that fit in shared memory.
//
//   forward : S = smat(w);  S = U L U' by two-sided cyclic Jacobi (round-robin parallel ordering, one CTA per
//             matrix, everything resident in shared memory);  s+ = svec(U max(L,0) U')   (Eq. 7)
//   backward: g_w = svec( U ((U' smat(G) U) o Gamma) U' )                                  (Eq. 9-10)
//             with Gamma the first divided differences of max(.,0) written without differences of close
//             eigenvalues, so it stays finite at repeated eigenvalues (L119).
// Not a tensor-core shape: the rotations are rank-2 updates with ~p dependent steps per sweep.
#pragma once
#include "common.cuh"
#include "lin.cuh"

namespace cdu {

struct PsdTab {
  int nblk;
  const int* prob;       // owning problem
  const int* row0;       // global index of the first svec row
  const int* p;          // matrix order
  const long long* uoff; // offset of the block's U in the eigenvector store (elements)
  const int* loff;       // offset of lambda
};

// Pair (i, j), i < j, met in round r at table q of a round-robin tournament over pe (even) players.
__device__ __forceinline__ void rr_pair(int r, int q, int pe, int& i, int& j) {
  const int mod = pe - 1;
  int a, b;
  if (q == 0) { a = pe - 1; b = r; }
  else { a = r + q; if (a >= mod) a -= mod; b = r - q; if (b < 0) b += mod; }
  i = a < b ? a : b; j = a < b ? b : a;
}

template <typename T> __device__ __forceinline__ T gamma_relu(T li, T lj) {
  const bool pi = li > (T)0, pj = lj > (T)0;
  if (pi && pj) return (T)1;
  if (!pi && !pj) return (T)0;
  const T mx = li > lj ? li : lj;
  return mx / (fabs(li) + fabs(lj));
}

// Two-sided Jacobi on the pe x pe matrix S (leading dimension ld, zero-padded if p is odd); V accumulates the
// rotations (columns = eigenvectors). On exit diag(S) holds the eigenvalues. Returns the number of sweeps.
template <typename T>
__device__ int jacobi_smem(int pe, int ld, T* S, T* V, T* cs, double* shred, int max_sweeps, int* flag) {
  const int tid = threadIdx.x, nt = blockDim.x;
  const int h = pe >> 1;
  double acc[1] = {0.0};
  for (int t = tid; t < pe * pe; t += nt) {
    const int a = t / pe, b = t - a * pe;
    const T v = S[a * ld + b];
    acc[0] += (double)v * (double)v;
    V[a * ld + b] = (a == b) ? (T)1 : (T)0;
  }
  block_sum<1>(acc, shred);
  const double normF2 = acc[0];
  if (!(normF2 > 0.0)) { if (normF2 != normF2) *flag |= FLAG_NONFINITE; return 0; }
  const double tol2 = 16.0 * (double)Eps<T>::v() * (double)Eps<T>::v() * normF2;
  const T skip = (T)(0.01 * sqrt(tol2) / pe);
  int sweep = 0;
  for (; sweep < max_sweeps; ++sweep) {
    acc[0] = 0.0;
    for (int t = tid; t < pe * pe; t += nt) {
      const int a = t / pe, b = t - a * pe;
      if (a < b) { const T v = S[a * ld + b]; acc[0] += 2.0 * (double)v * (double)v; }
    }
    block_sum<1>(acc, shred);
    if (!(acc[0] > tol2)) break;
    for (int r = 0; r < pe - 1; ++r) {
      for (int q = tid; q < h; q += nt) {
        int i, j; rr_pair(r, q, pe, i, j);
        const T aij = S[i * ld + j];
        // Rutishauser form: x' = x - s (y + tau x), y' = y + s (x - tau y), tau = s / (1 + c). The deviation from
        // orthogonality is O((1-c) eps) per rotation instead of O(eps), so V stays orthogonal to a few eps.
        T sn = (T)0, tau = (T)0, tt = (T)0;
        if (fabs(aij) > skip) {
          const double th = ((double)S[j * ld + j] - (double)S[i * ld + i]) / (2.0 * (double)aij);
          const double t = (th >= 0.0 ? 1.0 : -1.0) / (fabs(th) + sqrt(1.0 + th * th));
          const double c = 1.0 / sqrt(1.0 + t * t);
          sn = (T)(t * c); tau = (T)(t * c / (1.0 + c)); tt = (T)t;
        }
        cs[3 * q] = sn; cs[3 * q + 1] = tau; cs[3 * q + 2] = tt;
      }
      __syncthreads();
      for (int t = tid; t < h * h; t += nt) {
        const int q1 = t / h, q2 = t - q1 * h;
        int i1, j1, i2, j2;
        rr_pair(r, q1, pe, i1, j1); rr_pair(r, q2, pe, i2, j2);
        const T s1 = cs[3 * q1], t1 = cs[3 * q1 + 1], s2 = cs[3 * q2], t2 = cs[3 * q2 + 1];
        T a = S[i1 * ld + i2], b = S[i1 * ld + j2], c = S[j1 * ld + i2], d = S[j1 * ld + j2];
        if (q1 == q2) {
          const T g = cs[3 * q1 + 2] * b;                        // t * a_ij
          a -= g; d += g; b = (T)0; c = (T)0;
        } else {
          const T ra = a - s1 * (c + t1 * a), rc = c + s1 * (a - t1 * c);   // rows:  J' S
          const T rb = b - s1 * (d + t1 * b), rd = d + s1 * (b - t1 * d);
          a = ra - s2 * (rb + t2 * ra); b = rb + s2 * (ra - t2 * rb);       // cols:  (.) J
          c = rc - s2 * (rd + t2 * rc); d = rd + s2 * (rc - t2 * rd);
        }
        S[i1 * ld + i2] = a; S[i1 * ld + j2] = b; S[j1 * ld + i2] = c; S[j1 * ld + j2] = d;
      }
      for (int t = tid; t < pe * h; t += nt) {
        const int row = t / h, q2 = t - row * h;
        int i2, j2; rr_pair(r, q2, pe, i2, j2);
        const T s2 = cs[3 * q2], t2 = cs[3 * q2 + 1];
        const T a = V[row * ld + i2], b = V[row * ld + j2];
        V[row * ld + i2] = a - s2 * (b + t2 * a);
        V[row * ld + j2] = b + s2 * (a - t2 * b);
      }
      __syncthreads();
    }
  }
  if (sweep >= max_sweeps) *flag |= FLAG_EIG_CAP;
  return sweep;
}

// C(i,j) = sum_k A(i,k) B(k,j), all pe x pe in shared memory with generic strides; 2x2 register tiles.
template <typename T>
__device__ __forceinline__ void smem_gemm(int pe, const T* A, int sai, int sak, const T* B, int sbk, int sbj, T* C,
                                          int ldc) {
  const int h = pe >> 1;
  for (int t = threadIdx.x; t < h * h; t += blockDim.x) {
    const int i = (t / h) * 2, j = (t % h) * 2;
    T c00 = 0, c01 = 0, c10 = 0, c11 = 0;
    const T *a0 = A + i * sai, *a1 = a0 + sai, *b0 = B + j * sbj, *b1 = b0 + sbj;
#pragma unroll 4
    for (int k = 0; k < pe; ++k) {
      const T x0 = a0[k * sak], x1 = a1[k * sak], y0 = b0[k * sbk], y1 = b1[k * sbk];
      c00 += x0 * y0; c01 += x0 * y1; c10 += x1 * y0; c11 += x1 * y1;
    }
    C[i * ldc + j] = c00; C[i * ldc + j + 1] = c01; C[(i + 1) * ldc + j] = c10; C[(i + 1) * ldc + j + 1] = c11;
  }
}

template <typename T>
__device__ __forceinline__ void load_smat(int p, int pe, int ld, T* S, const double* v, double scale_add,
                                          const double* v2) {
  // S = smat(v + scale_add * v2) (v2 may be NULL), zero padded to pe
  for (int t = threadIdx.x; t < pe * pe; t += blockDim.x) {
    const int a = t / pe, b = t - a * pe;
    T val = (T)0;
    if (a < p && b < p) {
      const int idx = a <= b ? svec_idx(a, b) : svec_idx(b, a);
      double x = v[idx];
      if (v2) x += scale_add * v2[idx];
      val = (T)(a == b ? x : x * 0.70710678118654752440);
    } else if (a == b) {
      val = (T)0;
    }
    S[a * ld + b] = val;
  }
}

struct PsdFwdArgs {
  const double* W;   // projection argument, all rows
  double* S1;        // s^{k+1} base (rows)
  double* Y1;        // y^{k+1} base (rows)
  void* Ustore;      // eigenvector store of this iteration (or scratch)
  void* Lstore;
  int* sweeps_max; int* flags;
  unsigned long long* sweeps_sum;   // total Jacobi sweeps over blocks (statistics for the ALU roofline)
};

template <typename T>
__global__ void __launch_bounds__(512) k_psd_fwd_small(PsdTab tab, Hyper<T> H, int k, PsdFwdArgs A, const int* list) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int blk = list[blockIdx.x];
  const int p = tab.p[blk], pe = (p + 1) & ~1, ld = pe;
  const int prob = tab.prob[blk];
  const long long row0 = tab.row0[blk];
  double* shred = reinterpret_cast<double*>(smem_raw);
  T* S = reinterpret_cast<T*>(shred + 32);
  T* V = S + pe * ld;
  T* cs = V + pe * ld;
  T* lp = cs + 2 * pe;
  const double rho = H.rho_at(k, prob);
  const double* w = A.W + row0;
  load_smat<T>(p, pe, ld, S, w, 0.0, nullptr);
  __syncthreads();
  int flag = 0;
  const int sweeps = jacobi_smem<T>(pe, ld, S, V, cs, shred, 40, &flag);
  for (int i = threadIdx.x; i < pe; i += blockDim.x) { const T l = S[i * ld + i]; lp[i] = l > (T)0 ? l : (T)0; }
  __syncthreads();
  T* U = reinterpret_cast<T*>(A.Ustore) + tab.uoff[blk];
  T* L = reinterpret_cast<T*>(A.Lstore) + tab.loff[blk];
  for (int t = threadIdx.x; t < p * p; t += blockDim.x) { const int a = t / p, i = t - a * p; U[t] = V[a * ld + i]; }
  for (int i = threadIdx.x; i < p; i += blockDim.x) L[i] = S[i * ld + i];
  // rebuild + svec + dual update
  const int nsv = p * (p + 1) / 2;
  double* s1 = A.S1 + row0;
  double* y1 = A.Y1 + row0;
  for (int t = threadIdx.x; t < nsv; t += blockDim.x) {
    int b = (int)((sqrt(8.0 * t + 1.0) - 1.0) * 0.5);
    while (b * (b + 1) / 2 > t) --b;
    while ((b + 1) * (b + 2) / 2 <= t) ++b;
    const int a = t - b * (b + 1) / 2;
    const T *va = V + a * ld, *vb = V + b * ld;
    T acc = (T)0;
#pragma unroll 4
    for (int i = 0; i < pe; ++i) acc += va[i] * lp[i] * vb[i];
    const double sp = (a == b) ? (double)acc : (double)acc * 1.41421356237309504880;
    s1[t] = sp;
    y1[t] = rho * (sp - w[t]);
  }
  if (threadIdx.x == 0) {
    atomicMax(A.sweeps_max, sweeps);
    if (A.sweeps_sum) atomicAdd(A.sweeps_sum, (unsigned long long)sweeps);
    if (flag) atomicOr(A.flags + prob, flag);
  }
}

struct PsdBwdArgs {
  const double* W;     // w of step k, all rows
  const double* Yk;    // y^k rows
  const double* S1;    // s^{k+1} rows
  const double* Gs;    // cotangent of s^{k+1} rows
  const double* Gy;    // cotangent of y^{k+1} rows
  double* GW;          // out: g_w rows
  double* part;        // out: [nblk][2]
  const void* Ustore; const void* Lstore;
  int recompute;       // LEAN: eigendecompose smat(w) again
  int* flags;
};

template <typename T>
__global__ void __launch_bounds__(512) k_psd_bwd_small(PsdTab tab, Hyper<T> H, int k, PsdBwdArgs A, const int* list) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int blk = list[blockIdx.x];
  const int p = tab.p[blk], pe = (p + 1) & ~1, ld = pe;
  const int prob = tab.prob[blk];
  const long long row0 = tab.row0[blk];
  double* shred = reinterpret_cast<double*>(smem_raw);
  T* V = reinterpret_cast<T*>(shred + 64);
  T* G = V + pe * ld;       // S during a recompute, then smat(G), then C
  T* Tm = G + pe * ld;      // V accumulates here during recompute? no: scratch product
  T* cs = Tm + pe * ld;
  T* lam = cs + 2 * pe;
  const double rho = H.rho_at(k, prob);
  const double* w = A.W + row0;
  int flag = 0;
  if (A.recompute) {
    load_smat<T>(p, pe, ld, G, w, 0.0, nullptr);
    __syncthreads();
    jacobi_smem<T>(pe, ld, G, V, cs, shred, 40, &flag);
    for (int i = threadIdx.x; i < pe; i += blockDim.x) lam[i] = G[i * ld + i];
    __syncthreads();
  } else {
    const T* U = reinterpret_cast<const T*>(A.Ustore) + tab.uoff[blk];
    const T* L = reinterpret_cast<const T*>(A.Lstore) + tab.loff[blk];
    for (int t = threadIdx.x; t < pe * pe; t += blockDim.x) {
      const int a = t / pe, i = t - a * pe;
      V[a * ld + i] = (a < p && i < p) ? U[a * p + i] : ((a == i) ? (T)1 : (T)0);
    }
    for (int i = threadIdx.x; i < pe; i += blockDim.x) lam[i] = i < p ? L[i] : (T)0;
    __syncthreads();
  }
  const double* gs = A.Gs + row0;
  const double* gy = A.Gy + row0;
  load_smat<T>(p, pe, ld, G, gs, rho, gy);                 // G = smat(g_s+ + rho g_y+)
  __syncthreads();
  smem_gemm<T>(pe, G, ld, 1, V, ld, 1, Tm, ld);            // Tm = G V
  __syncthreads();
  smem_gemm<T>(pe, V, 1, ld, Tm, ld, 1, G, ld);            // C  = V' Tm
  __syncthreads();
  for (int t = threadIdx.x; t < pe * pe; t += blockDim.x) {
    const int i = t / pe, j = t - i * pe;
    G[i * ld + j] *= gamma_relu<T>(lam[i], lam[j]);
  }
  __syncthreads();
  smem_gemm<T>(pe, V, ld, 1, G, ld, 1, Tm, ld);            // Tm = V C
  __syncthreads();
  smem_gemm<T>(pe, Tm, ld, 1, V, 1, ld, G, ld);            // out = Tm V'
  __syncthreads();
  const int nsv = p * (p + 1) / 2;
  const double* yk = A.Yk + row0;
  const double* s1 = A.S1 + row0;
  double* gw = A.GW + row0;
  double acc[2] = {0.0, 0.0};
  for (int t = threadIdx.x; t < nsv; t += blockDim.x) {
    int b = (int)((sqrt(8.0 * t + 1.0) - 1.0) * 0.5);
    while (b * (b + 1) / 2 > t) --b;
    while ((b + 1) * (b + 2) / 2 <= t) ++b;
    const int a = t - b * (b + 1) / 2;
    const double o = (a == b) ? (double)G[a * ld + a]
                              : 0.5 * ((double)G[a * ld + b] + (double)G[b * ld + a]) * 1.41421356237309504880;
    const double gyv = gy[t];
    const double g = -rho * gyv + o;
    gw[t] = g;
    acc[0] += gyv * (s1[t] - w[t]);
    acc[1] += g * yk[t];
  }
  block_sum<2>(acc, shred);
  if (threadIdx.x == 0) {
    A.part[2 * blk] = acc[0]; A.part[2 * blk + 1] = acc[1];
    if (flag) atomicOr(A.flags + prob, flag);
  }
}

static inline size_t psd_small_smem_fwd(int p, size_t sz) { const int pe = (p + 1) & ~1; return 32 * 8 + (2 * (size_t)pe * pe + 3 * pe) * sz; }
static inline size_t psd_small_smem_bwd(int p, size_t sz) { const int pe = (p + 1) & ~1; return 64 * 8 + (3 * (size_t)pe * pe + 3 * pe) * sz; }

}  // namespace cdu

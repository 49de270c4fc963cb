// eq12.cuh - residuals of an iterate, the training loss of PAPER.md Eq. 12 (L146-148) with its cotangents on every
// iterate, and the policy features of App. E (L321-339). SURVEY.md 8(f) F2.
//
//   r_p = A x + s - b,  r_d = P x + q + A'y                     (as printed in Eq. 12 and L323)
//   L   = sum_{k=1..K} log( ||r_d^k||^2 / det(||r_d^0||^2) + ||r_p^k||^2 / det(||r_p^0||^2) )     (Eq. 12; det = stop-gradient,
//                                                                                                  DESIGN.md reading A12)
//   dL/dx^k = (2 / D_k) (P r_d^k / a_0 + A' r_p^k / b_0),  dL/ds^k = (2 / D_k) r_p^k / b_0,  dL/dy^k = (2 / D_k) A r_d^k / a_0,
//   a_k = ||r_d^k||^2, b_k = ||r_p^k||^2, D_k = a_k / a_0 + b_k / b_0  (a term whose denominator is 0 is dropped).
// The cotangent of z^k is formed when the reverse sweep reaches k, from the stored iterate: nothing of size K (n + 2m) is
// ever held (O(n) memory per unrolled iteration, L92).
// Grid-wide passes over the chunk table of lin_diag.cuh (one CTA = one chunk of rows / columns of one problem, fp64);
// per-problem sums and maxima are combined by the last CTA of a problem in chunk order (bit-reproducible).
#pragma once
#include "lin_diag.cuh"

namespace cdu {

constexpr int RES_NV = 8;   // a = ||r_d||^2, b = ||r_p||^2, max|Ax|, max|s|, max|b|, max|Px|, max|q|, max|A'y|

template <typename T, typename IT>
__device__ __forceinline__ double csr_row_dot(const int* rp, const IT* ci, const T* v, long long row, const double* x) {
  double a = 0.0;
  for (int e = rp[row]; e < rp[row + 1]; ++e) a += (double)v[e] * x[(int)ci[e]];
  return a;
}
template <typename T, typename IT>
__device__ __forceinline__ double p_row_dot(const BatchDev<T, IT>& D, int b, long long v0, int n, int j, const double* x) {
  if (D.P_dense) {
    const T* pr = D.P_v + D.P_off[b] + (long long)j * n;
    double a = 0.0;
    for (int i = 0; i < n; ++i) a += (double)pr[i] * x[i];
    return a;
  }
  return csr_row_dot<T, IT>(D.P_rp, D.P_ci, D.P_v, v0 + j, x);
}

__device__ __forceinline__ double block_max(double v, double* sh) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  const int w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  if ((threadIdx.x & 31) == 0) sh[w] = v;
  __syncthreads();
  double m = 0.0;
  for (int i = 0; i < nw; ++i) m = fmax(m, sh[i]);
  __syncthreads();
  return m;
}

// r_p, r_d of the iterate Z = (x | s | y) and the per-problem scalars nrm[b][RES_NV].
template <typename T, typename IT>
__global__ void __launch_bounds__(DIAG_THREADS) k_residuals(BatchDev<T, IT> D, DiagTab G, const double* Z, double* rp, double* rd,
                                                            double* nrm) {
  __shared__ double sh[2 * 32];
  __shared__ int is_last;
  const int4 ch = G.chunk[blockIdx.x];
  const int b = ch.x, tid = threadIdx.x;
  const long long v0 = D.var_off[b], r0 = D.row_off[b];
  const int n = D.var_off[b + 1] - (int)v0, m = D.row_off[b + 1] - (int)r0;
  const double *x = Z + v0, *s = Z + D.N + r0, *y = Z + D.N + D.Mtot + r0;
  double sum[2] = {0.0, 0.0}, mx[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  for (int j = ch.y + tid; j < min(ch.z, n); j += DIAG_THREADS) {
    const double px = p_row_dot(D, b, v0, n, j, x), q = (double)D.q[v0 + j];
    const double aty = csr_row_dot<T, IT>(D.AT_rp, D.AT_ci, D.AT_v, v0 + j, y);
    const double r = px + q + aty;
    rd[v0 + j] = r;
    sum[0] += r * r;
    mx[3] = fmax(mx[3], fabs(px)); mx[4] = fmax(mx[4], fabs(q)); mx[5] = fmax(mx[5], fabs(aty));
  }
  for (int r = ch.y + tid; r < min(ch.z, m); r += DIAG_THREADS) {
    const double ax = csr_row_dot<T, IT>(D.A_rp, D.A_ci, D.A_v, r0 + r, x), bv = (double)D.b[r0 + r];
    const double v = ax + s[r] - bv;
    rp[r0 + r] = v;
    sum[1] += v * v;
    mx[0] = fmax(mx[0], fabs(ax)); mx[1] = fmax(mx[1], fabs(s[r])); mx[2] = fmax(mx[2], fabs(bv));
  }
  block_sum<2>(sum, sh);
#pragma unroll
  for (int i = 0; i < 6; ++i) mx[i] = block_max(mx[i], sh);
  const int c0 = G.chunk_off[b], nch = G.chunk_off[b + 1] - c0;
  if (tid == 0) {
    double* p = G.part + (size_t)blockIdx.x * RES_NV;
    p[0] = sum[0]; p[1] = sum[1];
#pragma unroll
    for (int i = 0; i < 6; ++i) p[2 + i] = mx[i];
    __threadfence();
    const unsigned t = atomicAdd(G.ticket + b, 1u);
    is_last = (t == (unsigned)nch - 1u);
    if (is_last) { G.ticket[b] = 0u; __threadfence(); }
  }
  __syncthreads();
  if (is_last && tid < RES_NV) {
    double t = 0.0;
    for (int c = 0; c < nch; ++c) {
      const double v = __ldcg(G.part + (size_t)(c0 + c) * RES_NV + tid);
      t = tid < 2 ? t + v : fmax(t, v);
    }
    nrm[(size_t)b * RES_NV + tid] = t;
  }
}

// Gz (cotangent of z^k, x | s | y) += dL/dz^k of Eq. 12; rp, rd, nk: k_residuals of z^k; n0: of z^0.
template <typename T, typename IT>
__global__ void __launch_bounds__(DIAG_THREADS) k_eq12_cot(BatchDev<T, IT> D, DiagTab G, const double* rp, const double* rd,
                                                           const double* nk, const double* n0, double* Gz) {
  const int4 ch = G.chunk[blockIdx.x];
  const int b = ch.x, tid = threadIdx.x;
  const long long v0 = D.var_off[b], r0 = D.row_off[b];
  const int n = D.var_off[b + 1] - (int)v0, m = D.row_off[b + 1] - (int)r0;
  const double a0 = n0[(size_t)b * RES_NV], b0 = n0[(size_t)b * RES_NV + 1];
  const double ak = nk[(size_t)b * RES_NV], bk = nk[(size_t)b * RES_NV + 1];
  const double Dk = (a0 > 0.0 ? ak / a0 : 0.0) + (b0 > 0.0 ? bk / b0 : 0.0);
  if (!(Dk > 0.0)) return;
  const double c1 = a0 > 0.0 ? 2.0 / (Dk * a0) : 0.0, c2 = b0 > 0.0 ? 2.0 / (Dk * b0) : 0.0;
  double *gx = Gz + v0, *gs = Gz + D.N + r0, *gy = Gz + D.N + D.Mtot + r0;
  for (int j = ch.y + tid; j < min(ch.z, n); j += DIAG_THREADS)
    gx[j] += c1 * p_row_dot(D, b, v0, n, j, rd + v0) + c2 * csr_row_dot<T, IT>(D.AT_rp, D.AT_ci, D.AT_v, v0 + j, rp + r0);
  for (int r = ch.y + tid; r < min(ch.z, m); r += DIAG_THREADS) {
    gs[r] += c2 * rp[r0 + r];
    gy[r] += c1 * csr_row_dot<T, IT>(D.A_rp, D.A_ci, D.A_v, r0 + r, rd + v0);
  }
}

// loss[b] = sum_{k=1..K} log(a_k / a_0 + b_k / b_0) from nrm_all[k][b][RES_NV], k = 0..K
template <typename T>
__global__ void k_eq12_loss(const double* nrm_all, int K, int B, T* loss) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  const double a0 = nrm_all[(size_t)b * RES_NV], b0 = nrm_all[(size_t)b * RES_NV + 1];
  double L = 0.0;
  for (int k = 1; k <= K; ++k) {
    const double* p = nrm_all + ((size_t)k * B + b) * RES_NV;
    const double Dk = (a0 > 0.0 ? p[0] / a0 : 0.0) + (b0 > 0.0 ? p[1] / b0 : 0.0);
    if (Dk > 0.0) L += log(Dk);
  }
  loss[b] = (T)L;
}

// App. E features of iterate k: r_p / max(|Ax|, |s|, |b|)_inf, r_d / max(|Px|, |q|, |A'y|)_inf, delta_d = s^k - s^{k-1},
// delta_p = s^k - s-tilde^k, and per problem log(||.||_inf + 1e-12) of the three that the alpha policy reads.
template <typename T, typename IT>
__global__ void __launch_bounds__(DIAG_THREADS) k_features(BatchDev<T, IT> D, DiagTab G, const double* rp, const double* rd, const double* nrm,
                                                           const double* s_k, const double* s_km1, const double* st_k, T* rp_bar, T* rd_bar,
                                                           T* delta_p, T* delta_d, double* fmax_part) {
  __shared__ double sh[32];
  const int4 ch = G.chunk[blockIdx.x];
  const int b = ch.x, tid = threadIdx.x;
  const long long v0 = D.var_off[b], r0 = D.row_off[b];
  const int n = D.var_off[b + 1] - (int)v0, m = D.row_off[b + 1] - (int)r0;
  const double* q = nrm + (size_t)b * RES_NV;
  const double dp = fmax(q[2], fmax(q[3], q[4])), dd = fmax(q[5], fmax(q[6], q[7]));
  const double ip = dp > 0.0 ? 1.0 / dp : 1.0, id = dd > 0.0 ? 1.0 / dd : 1.0;
  double m3[3] = {0.0, 0.0, 0.0};   // |rp_bar|, |rd_bar|, |delta_p|
  for (int j = ch.y + tid; j < min(ch.z, n); j += DIAG_THREADS) {
    const double v = rd[v0 + j] * id;
    if (rd_bar) rd_bar[v0 + j] = (T)v;
    m3[1] = fmax(m3[1], fabs(v));
  }
  for (int r = ch.y + tid; r < min(ch.z, m); r += DIAG_THREADS) {
    const double v = rp[r0 + r] * ip, sk = s_k[r0 + r];
    const double d1 = st_k ? sk - st_k[r0 + r] : 0.0, d2 = s_km1 ? sk - s_km1[r0 + r] : 0.0;
    if (rp_bar) rp_bar[r0 + r] = (T)v;
    if (delta_p) delta_p[r0 + r] = (T)d1;
    if (delta_d) delta_d[r0 + r] = (T)d2;
    m3[0] = fmax(m3[0], fabs(v)); m3[2] = fmax(m3[2], fabs(d1));
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) m3[i] = block_max(m3[i], sh);
  if (tid == 0) { double* p = fmax_part + (size_t)blockIdx.x * 4; p[0] = m3[0]; p[1] = m3[1]; p[2] = m3[2]; }
}
template <typename T>
__global__ void k_features_fin(DiagTab G, int B, const double* fmax_part, T* scal) {   // scal[b][3] = log(max + 1e-12)
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  double m3[3] = {0.0, 0.0, 0.0};
  for (int c = G.chunk_off[b]; c < G.chunk_off[b + 1]; ++c)
    for (int i = 0; i < 3; ++i) m3[i] = fmax(m3[i], fmax_part[(size_t)c * 4 + i]);
  for (int i = 0; i < 3; ++i) scal[(size_t)b * 3 + i] = (T)log(m3[i] + 1e-12);
}

template <typename T>
__global__ void k_add_vec(double* dst, const T* src, long long n) {   // dst += src
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) dst[i] += (double)src[i];
}

}  // namespace cdu

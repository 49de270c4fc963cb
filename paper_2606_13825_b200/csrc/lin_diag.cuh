// lin_diag.cuh - the linear-system step when M = P + sigma I + rho A'A is DIAGONAL (every row of A holds at most one
// entry and P only diagonal entries: the max-cut SDPs of BASELINE.json configs 1, 2, 5, where A = [E_diag; -I], P = 0).
//
// Jacobi-preconditioned CG (Eq. 4) on a diagonal M ends after its first iteration with
// xt = xi / diag(M) - the preconditioned residual IS the solution - so this path evaluates that one iteration in closed
// form, in fp64, and nothing couples the entries of a problem any more: S1-S5, S7 (forward) and S9-S13 (reverse, with
// the adjoint solve lam = g_xt / diag(M), Eq. 5, and Eq. 6 L90 in the cancellation-free form of lin.cuh) become
// one grid-wide pass each, with no per-problem team, no cluster barrier and no CG work vectors. Same arithmetic as
// lin.cuh in exact arithmetic; cdu_stats counts one CG iteration per solve.
//   * a CTA owns one chunk of one problem: columns [lo, hi) and rows [lo, hi) (local indices);
//   * a row needs xt (or lam) of its column, which another thread (possibly another CTA) owns: it is recomputed from
//     the column's entries of A' (cdu_create admits the path only if no column holds more than DIAG_MAXCOL entries);
//   * per-problem dot products (g_rho, g_alpha, g_sigma and the two partials handed from the pre to the post phase):
//     block sums into part[chunk][], the last CTA of a problem to arrive (ticket) adds them in a fixed order, so the
//     results are bit-reproducible.
#pragma once
#include "lin.cuh"

namespace cdu {

constexpr int DIAG_MAXCOL = 8;        // admitted entries per column of A
constexpr int DIAG_CHUNK = 512;       // local indices per CTA (two per thread: the gathers are dependent loads, parallelism hides them)
constexpr int DIAG_THREADS = 256;

template <typename T, typename IT>
struct DiagCtx {   // one problem as seen by one thread
  const BatchDev<T, IT>& D;
  int b, n, m;
  long long v0, r0;
  double rho, alpha, sigma;
  const T* rrow;                     // per-row rho of this problem at this iteration, or NULL
  __device__ DiagCtx(const BatchDev<T, IT>& D_, const Hyper<T>& H, int k, int b_) : D(D_), b(b_) {
    v0 = D.var_off[b]; r0 = D.row_off[b];
    n = D.var_off[b + 1] - (int)v0; m = D.row_off[b + 1] - (int)r0;
    rho = H.rho_row ? 0.0 : H.rho_at(k, b); alpha = H.alpha_at(k, b); sigma = H.sigma;
    rrow = H.rows_of(k, r0);
  }
  __device__ __forceinline__ double rh(int row) const { return rrow ? (double)rrow[row] : rho; }
  // t_j = sum_e v_e f(row_e) over column j of A, and diag(M)_j (exact: the squares are summed here, in fp64)
  template <typename F> __device__ __forceinline__ double col_gather(int j, double& dM, F f) const {
    double a = 0.0, sq = 0.0;
    for (int e = D.AT_rp[v0 + j]; e < D.AT_rp[v0 + j + 1]; ++e) {
      const double v = (double)D.AT_v[e];
      const int r = (int)D.AT_ci[e];
      a += v * f(r);
      sq += v * v * rh(r);
    }
    dM = (double)D.diagP[v0 + j] + sigma + sq;
    return a;
  }
  // S1 + S2: xt_j = (sigma x_j - q_j + [A'(rho (b - s) - y)]_j) / diag(M)_j
  __device__ __forceinline__ double xt_of(int j, const double* x, const double* s, const double* y) const {
    double dM;
    const double a = col_gather(j, dM, [&](int r) { return rh(r) * ((double)D.b[r0 + r] - s[r]) - y[r]; });
    return (sigma * x[j] - (double)D.q[v0 + j] + a) / dM;
  }
  // S10 + S11: lam_j = alpha (g_x+_j - [A' g_w]_j) / diag(M)_j
  __device__ __forceinline__ double lam_of(int j, const double* gx1, const double* gw) const {
    double dM;
    const double a = col_gather(j, dM, [&](int r) { return gw[r]; });
    return alpha * (gx1[j] - a) / dM;
  }
};

// Sum of NV doubles over the chunks of a problem: every CTA leaves its block sums in part[chunk]; the last one to arrive
// adds the problem's chunks in a fixed order and returns true (to all its threads) with the totals in v.
template <int NV>
__device__ __forceinline__ bool diag_problem_sum(double (&v)[NV], double* sh, double* part, unsigned* ticket, int chunk0, int nch,
                                                 int chunk) {
  __shared__ int is_last;
  block_sum<NV>(v, sh);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int i = 0; i < NV; ++i) part[(size_t)chunk * 4 + i] = v[i];
    __threadfence();
    const unsigned t = atomicAdd(ticket, 1u);
    is_last = (t == (unsigned)nch - 1u);
    if (is_last) { *ticket = 0u; __threadfence(); }
  }
  __syncthreads();
  if (!is_last) return false;
  // thread t adds the chunks t, t + blockDim.x, ... and the block sums those: a fixed order, whatever CTA arrives last
#pragma unroll
  for (int i = 0; i < NV; ++i) v[i] = 0.0;
  for (int c = threadIdx.x; c < nch; c += blockDim.x) {
#pragma unroll
    for (int i = 0; i < NV; ++i) v[i] += __ldcg(part + (size_t)(chunk0 + c) * 4 + i);
  }
  __syncthreads();
  block_sum<NV>(v, sh);
  return true;
}

struct DiagTab {
  int nchunk;
  const int4* chunk;        // (problem, lo, hi, index of the chunk inside its problem)
  const int* chunk_off;     // [B+1]
  const int* acol;          // [Mtot] local column of the row's entry, -1: empty row
  double* part;             // [nchunk][4]
  unsigned* ticket;         // [B], zero between launches
};

// relaxation, zero / nonneg projection and dual update of one row (S3-S5, S7); PSD rows only leave w
template <typename T, typename IT>
__device__ __forceinline__ double diag_row_st(const DiagCtx<T, IT>& c, const DiagTab& G, const T* aval, int r, const double* x,
                                              const double* s, const double* y) {
  const int jc = G.acol[c.r0 + r];
  const double a = jc >= 0 ? (double)aval[c.r0 + r] * c.xt_of(jc, x, s, y) : 0.0;
  return (double)c.D.b[c.r0 + r] - a;
}

template <typename T, typename IT>
__global__ void __launch_bounds__(DIAG_THREADS) k_dfwd(BatchDev<T, IT> D, DiagTab G, const T* aval, Hyper<T> H, IterPtrs I, int k) {
  const int4 ch = G.chunk[blockIdx.x];
  const DiagCtx<T, IT> c(D, H, k, ch.x);
  const int tid = threadIdx.x;
  const double *x = I.Zk + c.v0, *s = I.Zk + D.N + c.r0, *y = I.Zk + D.N + D.Mtot + c.r0;
  double *x1 = I.Zk1 + c.v0, *s1 = I.Zk1 + D.N + c.r0, *y1 = I.Zk1 + D.N + D.Mtot + c.r0;
  double *xt = I.XT + c.v0, *st = I.ST + c.r0;
  const double al = c.alpha;
  bool bad = false;
  for (int j = ch.y + tid; j < min(ch.z, c.n); j += DIAG_THREADS) {
    const double v = c.xt_of(j, x, s, y);
    bad |= (v != v);
    xt[j] = v;
    x1[j] = al * v + (1.0 - al) * x[j];
  }
  const uint8_t* kind = D.rowkind + c.r0;
  for (int r = ch.y + tid; r < min(ch.z, c.m); r += DIAG_THREADS) {
    const double stv = diag_row_st(c, G, aval, r, x, s, y);
    st[r] = stv;
    const double rho = c.rh(r);
    const double w = al * stv + (1.0 - al) * s[r] - y[r] / rho;
    D.W[c.r0 + r] = w;
    const int kd = kind[r];
    if (kd <= KIND_NONNEG) {
      const double sp = (kd == KIND_NONNEG && w > 0.0) ? w : 0.0;
      s1[r] = sp;
      y1[r] = rho * (sp - w);
    }
  }
  if (bad) atomicOr(D.flags + c.b, FLAG_NONFINITE);
  if (ch.w == 0 && tid == 0) { D.cg_iters[c.b] += 1; D.cg_iters0[c.b] += 1; if (D.cg_max[c.b] < 1) D.cg_max[c.b] = 1; }
}

// Reverse step, phase 1: (LEAN: xt, st again), w, and the zero / nonneg rows of g_w with the two partial dots.
template <typename T, typename IT>
__global__ void __launch_bounds__(DIAG_THREADS) k_dbwd_pre(BatchDev<T, IT> D, DiagTab G, const T* aval, Hyper<T> H, BwdPtrs Q, int k) {
  __shared__ double sh[2 * 32];
  const int4 ch = G.chunk[blockIdx.x];
  const DiagCtx<T, IT> c(D, H, k, ch.x);
  const int tid = threadIdx.x;
  const double *x = Q.Zk + c.v0, *s = Q.Zk + D.N + c.r0, *y = Q.Zk + D.N + D.Mtot + c.r0;
  const double* s1 = Q.Zk1 + D.N + c.r0;
  const double *gs = Q.Gin + D.N + c.r0, *gy = Q.Gin + D.N + D.Mtot + c.r0;
  double *xt = Q.XT + c.v0, *st = Q.ST + c.r0;
  const double al = c.alpha;
  if (Q.recompute)
    for (int j = ch.y + tid; j < min(ch.z, c.n); j += DIAG_THREADS) xt[j] = c.xt_of(j, x, s, y);
  const uint8_t* kind = D.rowkind + c.r0;
  double acc[2] = {0.0, 0.0};   // <gy, s+ - w>, <gw, y> over the zero / nonneg rows
  for (int r = ch.y + tid; r < min(ch.z, c.m); r += DIAG_THREADS) {
    double stv;
    if (Q.recompute) { stv = diag_row_st(c, G, aval, r, x, s, y); st[r] = stv; } else stv = st[r];
    const double yv = y[r], rho = c.rh(r);
    const double w = al * stv + (1.0 - al) * s[r] - yv / rho;
    D.W[c.r0 + r] = w;
    const int kd = kind[r];
    if (kd <= KIND_NONNEG) {
      const double gyv = gy[r];
      const double Gv = gs[r] + rho * gyv;
      const double gw = -rho * gyv + ((kd == KIND_NONNEG && w > 0.0) ? Gv : 0.0);
      D.GW[c.r0 + r] = gw;
      acc[0] += gyv * (s1[r] - w);
      acc[1] += gw * yv;
    }
  }
  const int c0 = G.chunk_off[c.b], nch = G.chunk_off[c.b + 1] - c0;
  if (diag_problem_sum<2>(acc, sh, G.part, G.ticket + c.b, c0, nch, blockIdx.x) && tid == 0) {
    Q.part_pre[2 * c.b] = acc[0]; Q.part_pre[2 * c.b + 1] = acc[1];
    if (Q.recompute) { D.cg_iters[c.b] += 1; D.cg_iters0[c.b] += 1; }
  }
}

// Reverse step, phase 2: adjoint solve, Eq. 6 and the cotangent of z^k; needs g_w on every row (PSD rows: PSD kernels).
template <typename T, typename IT>
__global__ void __launch_bounds__(DIAG_THREADS) k_dbwd_post(BatchDev<T, IT> D, DiagTab G, const T* aval, Hyper<T> H, BwdPtrs Q, int k) {
  __shared__ double sh[3 * 32];
  const int4 ch = G.chunk[blockIdx.x];
  const DiagCtx<T, IT> c(D, H, k, ch.x);
  const int tid = threadIdx.x;
  const double *x = Q.Zk + c.v0, *s = Q.Zk + D.N + c.r0;
  const double* gx1 = Q.Gin + c.v0;
  double *gx = Q.Gout + c.v0, *gs = Q.Gout + D.N + c.r0, *gy = Q.Gout + D.N + D.Mtot + c.r0;
  const double *xt = Q.XT + c.v0, *st = Q.ST + c.r0;
  const double* gw = D.GW + c.r0;
  const double al = c.alpha, sg = c.sigma;
  const double* gy1 = Q.Gin + D.N + D.Mtot + c.r0;
  const double* s1 = Q.Zk1 + D.N + c.r0;
  const double* yk = Q.Zk + D.N + D.Mtot + c.r0;
  double* grow = Q.g_rho_row ? Q.g_rho_row + (size_t)k * D.Mtot + c.r0 : nullptr;
  double acc[3] = {0.0, 0.0, 0.0};   // rho, alpha, sigma
  for (int j = ch.y + tid; j < min(ch.z, c.n); j += DIAG_THREADS) {
    const double l = c.lam_of(j, gx1, gw), g1 = gx1[j], dx = xt[j] - x[j];
    acc[1] += g1 * dx;                                  // B5: <g_x+, xt - x>
    acc[2] -= l * dx;                                   // B7+B8: <lam, x - xt>
    gx[j] = (1.0 - al) * g1 + sg * l;                   // B5 + B8
  }
  for (int r = ch.y + tid; r < min(ch.z, c.m); r += DIAG_THREADS) {
    const int jc = G.acol[c.r0 + r];
    const double u = jc >= 0 ? (double)aval[c.r0 + r] * c.lam_of(jc, gx1, gw) : 0.0;   // u = A lam
    const double g = gw[r], ds = st[r] - s[r], rho = c.rh(r);
    acc[0] += u * ds;                                   // B7+B9: <u, st - s>
    acc[1] += g * ds;                                   // B5: <g_vhat, st - s>
    if (grow) grow[r] = u * ds + gy1[r] * (s1[r] - D.W[c.r0 + r]) + g * yk[r] / (rho * rho);   // per-row rho: B1 + B4 + (B7+B9) row by row
    gs[r] = (1.0 - al) * g - rho * u;                   // B5 + B9
    gy[r] = -g / rho - u;                               // B4 + B9
  }
  const int c0 = G.chunk_off[c.b], nch = G.chunk_off[c.b + 1] - c0;
  if (diag_problem_sum<3>(acc, sh, G.part, G.ticket + c.b, c0, nch, blockIdx.x) && tid == 0) {
    double d_gy_sw = Q.part_pre[2 * c.b], d_gw_y = Q.part_pre[2 * c.b + 1];
    for (int j = D.psdblk_off[c.b]; j < D.psdblk_off[c.b + 1]; ++j) { d_gy_sw += D.psd_part[2 * j]; d_gw_y += D.psd_part[2 * j + 1]; }
    const size_t o = (size_t)k * D.B + c.b;
    Q.g_rho_pb[o] = grow ? 0.0 : acc[0] + d_gy_sw + d_gw_y / (c.rho * c.rho);   // B1 + B4 + (B7+B9)
    Q.g_alpha_pb[o] = acc[1];
    Q.g_sigma_pb[o] = acc[2];
    D.cg_iters[c.b] += 1; D.cg_iters0[c.b] += 1;
  }
}

}  // namespace cdu

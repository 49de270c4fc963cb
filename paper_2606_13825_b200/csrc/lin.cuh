// lin.cuh - per-problem linear-system step, relaxation, separable/SOC cones, and their reverse.
//
// One CTA owns one problem instance of the batch ("super-batch" of PAPER.md L306 held as batched CSR with
// per-problem offsets; CG convergence is decided per problem on the device, never by the host).
//   forward  : S1 xi assembly, S2 PCG on M = P + sigma I + rho A'A (Eq. 4, Jacobi preconditioner L294),
//              S3 st = b - A xt, S4 relaxation (Eq. 3c-3d), S5 zero/nonneg/SOC projection, S7 dual
//              update (Eq. 3e) - SURVEY.md 8(a).
//   backward : S9 (separable + SOC part), S10, S11 adjoint PCG (Eq. 5), S12 Eq. 6 (L90) and the RHS terms.
// The iterate and every reduction are fp64; matrices, CG vectors and the preconditioner are T.
#pragma once
#include "common.cuh"

namespace cdu {

template <typename T>
struct BatchDev {
  int B;
  const int *var_off, *row_off;                       // [B+1]
  const int *A_rp, *A_ci;   const T* A_v;   int A_G;   // A   : rows = constraints, local column index
  const int *AT_rp, *AT_ci; const T* AT_v;  int AT_G;  // A^T : rows = variables,   local row index
  const int *P_rp, *P_ci;   const T* P_v;   int P_G;   // P   : full symmetric storage
  const T *q, *b, *diagP, *colsq;
  const uint8_t* rowkind;                              // per row: cone kind
  const int *soc_off, *soc_start, *soc_dim;            // per problem SOC list (start = local row)
  const int *psdblk_off;                               // [B+1] PSD blocks of each problem
  double *xi, *xt_scr, *rd, *tm, *st_scr, *W, *GW, *lam;   // fp64 scratch, sized sum n / sum m
  T *r, *p, *Ap, *d, *dinv, *tA;                        // CG vectors
  double tol, tol_ref;
  int maxit, refine;
  int *cg_iters, *cg_max, *flags;                      // [B] statistics
  double* psd_part;                                    // [nblk][2] partial dots written by the PSD backward
  long long N, Mtot;
};

template <typename T>
struct Hyper {  // per-iteration hyper-parameters as the caller laid them out (cdu_rho_mode)
  const T* rho; const T* alpha; int kstride, pstride; double sigma;
  __device__ double rho_at(int k, int b) const { return (double)rho[(size_t)k * kstride + (size_t)b * pstride]; }
  __device__ double alpha_at(int k, int b) const { return (double)alpha[(size_t)k * kstride + (size_t)b * pstride]; }
};

// y = op(rows) . x with a group of G (power of two <= 32) lanes per row; emit(row, dot) runs on lane 0 of the group.
template <typename TACC, typename TV, typename TX, typename F>
__device__ __forceinline__ void spmv_rows(int nrows, const int* __restrict__ rp, const int* __restrict__ ci,
                                          const TV* __restrict__ v, const TX* x, int G, F emit) {
  const int tid = threadIdx.x;
  const int gl = tid & (G - 1);
  const int gid = tid / G, ng = blockDim.x / G;
  for (int row0 = 0; row0 < nrows; row0 += ng) {
    const int row = row0 + gid;
    TACC acc = (TACC)0;
    if (row < nrows) {
      const int e0 = __ldg(rp + row), e1 = __ldg(rp + row + 1);
#pragma unroll 4
      for (int e = e0 + gl; e < e1; e += G) acc += (TACC)__ldg(v + e) * (TACC)x[__ldg(ci + e)];
    }
    for (int o = G >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (row < nrows && gl == 0) emit(row, acc);
  }
}

template <typename T>
struct Prob {  // one problem's view of the batch
  int n, m, b;
  const int *A_rp, *AT_rp, *P_rp;
  const T *q, *bv, *diagP, *colsq;
  double *xi, *rd, *tm, *W, *GW, *lam;
  T *r, *p, *Ap, *d, *dinv, *tA;
  double rho, alpha, sigma;
  double* sh;
  __device__ Prob(const BatchDev<T>& D, int b_, double* sh_) : b(b_), sh(sh_) {
    const int v0 = D.var_off[b], r0 = D.row_off[b];
    n = D.var_off[b + 1] - v0; m = D.row_off[b + 1] - r0;
    A_rp = D.A_rp + r0; AT_rp = D.AT_rp + v0; P_rp = D.P_rp + v0;
    q = D.q + v0; bv = D.b + r0; diagP = D.diagP + v0; colsq = D.colsq + v0;
    xi = D.xi + v0; rd = D.rd + v0; lam = D.lam + v0; tm = D.tm + r0; W = D.W + r0; GW = D.GW + r0;
    r = D.r + v0; p = D.p + v0; Ap = D.Ap + v0; d = D.d + v0; dinv = D.dinv + v0; tA = D.tA + r0;
  }
};

// Jacobi-preconditioned CG on M d = r, d0 = 0. r (T) holds the right-hand side on entry. rr0 = ||r||^2.
// Stops when the recursive residual satisfies ||r|| <= thresh. Returns iterations.
template <typename T>
__device__ int pcg(const BatchDev<T>& D, const Prob<T>& c, double thresh, double rr0, int* flag) {
  const int tid = threadIdx.x, nt = blockDim.x;
  double acc[2];
  acc[0] = 0.0;
  for (int i = tid; i < c.n; i += nt) {
    const T ri = c.r[i], z = ri * c.dinv[i];
    c.d[i] = (T)0; c.p[i] = z;
    acc[0] += (double)ri * (double)z;
  }
  acc[1] = 0.0;
  block_sum<2>(acc, c.sh);
  double rz = acc[0];
  const double th2 = thresh * thresh;
  int it = 0;
  if (!(rr0 > th2)) return 0;
  const T rhoT = (T)c.rho, sigT = (T)c.sigma;
  while (it < D.maxit) {
    spmv_rows<T>(c.m, c.A_rp, D.A_ci, D.A_v, c.p, D.A_G, [&](int row, T a) { c.tA[row] = rhoT * a; });
    __syncthreads();
    spmv_rows<T>(c.n, c.AT_rp, D.AT_ci, D.AT_v, c.tA, D.AT_G, [&](int row, T a) { c.Ap[row] = a; });
    __syncthreads();
    double pap[1] = {0.0};
    spmv_rows<T>(c.n, c.P_rp, D.P_ci, D.P_v, c.p, D.P_G, [&](int row, T a) {
      const T pi = c.p[row];
      const T ap = c.Ap[row] + a + sigT * pi;
      c.Ap[row] = ap;
      pap[0] += (double)pi * (double)ap;
    });
    block_sum<1>(pap, c.sh);
    if (!(pap[0] > 0.0)) { *flag |= FLAG_CG_CURV; break; }
    const T a = (T)(rz / pap[0]);
    acc[0] = 0.0; acc[1] = 0.0;
    for (int i = tid; i < c.n; i += nt) {
      const T pi = c.p[i];
      c.d[i] += a * pi;
      const T ri = c.r[i] - a * c.Ap[i];
      c.r[i] = ri;
      const T z = ri * c.dinv[i];
      acc[0] += (double)ri * (double)ri;
      acc[1] += (double)ri * (double)z;
    }
    block_sum<2>(acc, c.sh);
    ++it;
    if (!(acc[0] > th2)) break;
    const T beta = (T)(acc[1] / rz);
    rz = acc[1];
    for (int i = tid; i < c.n; i += nt) c.p[i] = c.r[i] * c.dinv[i] + beta * c.p[i];
    __syncthreads();
  }
  if (it >= D.maxit) *flag |= FLAG_CG_CAP;
  return it;
}

// out = M^-1 rhs with start xbase (NULL = 0): pass 0 is PCG to tol ||rhs|| on the fp64 residual of the start
// (identical to CG started at xbase); each further pass re-evaluates the residual in fp64 and corrects
// (iterative refinement). Guards ||rhs|| = 0 => out = 0 (reading A5).
template <typename T>
__device__ int solve_M(const BatchDev<T>& D, const Prob<T>& c, const double* rhs, const double* xbase, double* out,
                       int* flag) {
  const int tid = threadIdx.x, nt = blockDim.x;
  double acc[1] = {0.0};
  for (int i = tid; i < c.n; i += nt) {
    c.dinv[i] = (T)(1.0 / ((double)c.diagP[i] + c.sigma + c.rho * (double)c.colsq[i]));
    const double v = rhs[i];
    acc[0] += v * v;
    out[i] = xbase ? xbase[i] : 0.0;
  }
  block_sum<1>(acc, c.sh);
  const double nr2 = acc[0];
  if (!(nr2 > 0.0)) {
    for (int i = tid; i < c.n; i += nt) out[i] = 0.0;
    if (nr2 != nr2) *flag |= FLAG_NONFINITE;
    __syncthreads();
    return 0;
  }
  int total = 0;
  for (int pass = 0; pass <= D.refine; ++pass) {
    double rr0;
    if (pass == 0 && !xbase) {
      for (int i = tid; i < c.n; i += nt) c.r[i] = (T)rhs[i];
      rr0 = nr2;
      __syncthreads();
    } else {  // r = rhs - M out, fp64
      spmv_rows<double>(c.m, c.A_rp, D.A_ci, D.A_v, out, D.A_G, [&](int row, double a) { c.tm[row] = c.rho * a; });
      __syncthreads();
      spmv_rows<double>(c.n, c.AT_rp, D.AT_ci, D.AT_v, c.tm, D.AT_G, [&](int row, double a) { c.rd[row] = a; });
      __syncthreads();
      acc[0] = 0.0;
      spmv_rows<double>(c.n, c.P_rp, D.P_ci, D.P_v, out, D.P_G, [&](int row, double a) {
        const double res = rhs[row] - (c.rd[row] + a + c.sigma * out[row]);
        c.r[row] = (T)res;
        acc[0] += res * res;
      });
      block_sum<1>(acc, c.sh);
      rr0 = acc[0];
    }
    double thresh = D.tol * sqrt(nr2);
    if (pass > 0) {
      if (!(rr0 > 1e-28 * nr2)) break;
      thresh = D.tol_ref * sqrt(rr0);
    }
    const int it = pcg(D, c, thresh, rr0, flag);
    total += it;
    if (it == 0 && pass == 0 && D.refine == 0) break;
    for (int i = tid; i < c.n; i += nt) out[i] += (double)c.d[i];
    __syncthreads();
  }
  return total;
}

// xi and x-tilde of one step from z^k = (x, s, y): S1 + S2. Writes xt; st is produced by the caller's A pass.
template <typename T>
__device__ int lin_solve_step(const BatchDev<T>& D, const Prob<T>& c, const double* x, const double* s,
                              const double* y, double* xt, int* flag) {
  const int tid = threadIdx.x, nt = blockDim.x;
  for (int i = tid; i < c.m; i += nt) c.tm[i] = c.rho * ((double)c.bv[i] - s[i]) - y[i];
  __syncthreads();
  spmv_rows<double>(c.n, c.AT_rp, D.AT_ci, D.AT_v, c.tm, D.AT_G,
                    [&](int row, double a) { c.xi[row] = c.sigma * x[row] - (double)c.q[row] + a; });
  __syncthreads();
  return solve_M(D, c, c.xi, x, xt, flag);
}

// SOC projection of one cone held by a warp: w -> s+; returns branch (0 inside, 1 polar, 2 boundary), nu.
__device__ __forceinline__ int soc_branch(double t, double nu) { return (nu <= t) ? 0 : ((nu <= -t) ? 1 : 2); }

struct IterPtrs {
  const double* Zk;   // z^k  (x | s | y), sizes N, Mtot, Mtot
  double* Zk1;        // z^{k+1}
  double* XT;         // x-tilde store (checkpoint slot or scratch), size N
  double* ST;         // s-tilde store, size Mtot
};

template <typename T>
__global__ void __launch_bounds__(1024) k_fwd(BatchDev<T> D, Hyper<T> H, IterPtrs I, int k) {
  __shared__ double sh[3 * 32];
  const int b = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
  Prob<T> c(D, b, sh);
  c.rho = H.rho_at(k, b); c.alpha = H.alpha_at(k, b); c.sigma = H.sigma;
  const long long v0 = D.var_off[b], r0 = D.row_off[b];
  const double *x = I.Zk + v0, *s = I.Zk + D.N + r0, *y = I.Zk + D.N + D.Mtot + r0;
  double *x1 = I.Zk1 + v0, *s1 = I.Zk1 + D.N + r0, *y1 = I.Zk1 + D.N + D.Mtot + r0;
  double *xt = I.XT + v0, *st = I.ST + r0;
  int flag = 0;
  const int iters = lin_solve_step(D, c, x, s, y, xt, &flag);
  const double al = c.alpha, rho = c.rho;
  const uint8_t* kind = D.rowkind + r0;
  spmv_rows<double>(c.m, c.A_rp, D.A_ci, D.A_v, xt, D.A_G, [&](int row, double a) {
    const double stv = (double)c.bv[row] - a;
    st[row] = stv;
    const double yv = y[row];
    const double w = al * stv + (1.0 - al) * s[row] - yv / rho;
    c.W[row] = w;
    const int kd = kind[row];
    if (kd <= KIND_NONNEG) {
      const double sp = (kd == KIND_NONNEG && w > 0.0) ? w : 0.0;
      s1[row] = sp;
      y1[row] = rho * (sp - w);
    }
  });
  for (int i = tid; i < c.n; i += nt) x1[i] = al * xt[i] + (1.0 - al) * x[i];
  __syncthreads();
  // second-order cones of this problem: one warp per cone
  const int lane = tid & 31, wid = tid >> 5, nw = nt >> 5;
  for (int j = D.soc_off[b] + wid; j < D.soc_off[b + 1]; j += nw) {
    const int st0 = D.soc_start[j], dim = D.soc_dim[j];
    const double* w = c.W + st0;
    double nu2 = 0.0;
    for (int i = 1 + lane; i < dim; i += 32) nu2 += w[i] * w[i];
    nu2 = warp_sum(nu2);
    const double t = w[0], nu = sqrt(nu2);
    const int br = soc_branch(t, nu);
    const double cf = (br == 2) ? 0.5 * (t + nu) : 0.0;
    for (int i = lane; i < dim; i += 32) {
      const double wi = w[i];
      double sp;
      if (br == 0) sp = wi; else if (br == 1) sp = 0.0; else sp = (i == 0) ? cf : cf * wi / nu;
      s1[st0 + i] = sp;
      y1[st0 + i] = rho * (sp - wi);
    }
  }
  if (tid == 0) {
    D.cg_iters[b] += iters;
    if (iters > D.cg_max[b]) D.cg_max[b] = iters;
    if (flag) D.flags[b] |= flag;
  }
}

// ---------------------------------------------------------------------------------------------------------
// backward
// ---------------------------------------------------------------------------------------------------------
struct BwdPtrs {
  const double* Zk;    // z^k
  const double* Zk1;   // z^{k+1} (s+ is read from it)
  double* XT;          // x-tilde of step k (FULL: checkpoint; LEAN: scratch, recomputed here)
  double* ST;          // s-tilde of step k
  const double* Gin;   // cotangent of z^{k+1}: (g_x | g_s | g_y)
  double* Gout;        // cotangent of z^k
  double* g_rho_pb;    // [K][B] per-problem partials
  double* g_alpha_pb;
  double* g_sigma_pb;
  double* part_pre;    // [B][2] partials handed from the pre to the post phase
  int recompute;       // LEAN: re-solve for xt, st
};

// Phase 1 of the reverse step: (LEAN: re-solve), w, and B1/B2/B4 for zero, nonneg and SOC rows.
template <typename T>
__device__ void bwd_pre(const BatchDev<T>& D, Prob<T>& c, const BwdPtrs& Q, double* out_part, int* flag, int* iters) {
  const int b = c.b, tid = threadIdx.x, nt = blockDim.x;
  const long long v0 = D.var_off[b], r0 = D.row_off[b];
  const double *x = Q.Zk + v0, *s = Q.Zk + D.N + r0, *y = Q.Zk + D.N + D.Mtot + r0;
  const double* s1 = Q.Zk1 + D.N + r0;
  const double *gs = Q.Gin + D.N + r0, *gy = Q.Gin + D.N + D.Mtot + r0;
  double *xt = Q.XT + v0, *st = Q.ST + r0;
  const double al = c.alpha, rho = c.rho;
  if (Q.recompute) {
    *iters += lin_solve_step(D, c, x, s, y, xt, flag);
    spmv_rows<double>(c.m, c.A_rp, D.A_ci, D.A_v, xt, D.A_G, [&](int row, double a) { st[row] = (double)c.bv[row] - a; });
    __syncthreads();
  }
  const uint8_t* kind = D.rowkind + r0;
  double acc[2] = {0.0, 0.0};   // [0]: <gy, s+ - w>, [1]: <gw, y>
  for (int i = tid; i < c.m; i += nt) {
    const double yv = y[i];
    const double w = al * st[i] + (1.0 - al) * s[i] - yv / rho;
    c.W[i] = w;
    const int kd = kind[i];
    if (kd <= KIND_NONNEG) {
      const double gyv = gy[i];
      const double G = gs[i] + rho * gyv;
      const double gw = -rho * gyv + ((kd == KIND_NONNEG && w > 0.0) ? G : 0.0);
      c.GW[i] = gw;
      acc[0] += gyv * (s1[i] - w);
      acc[1] += gw * yv;
    }
  }
  __syncthreads();
  const int lane = tid & 31, wid = tid >> 5, nw = nt >> 5;
  for (int j = D.soc_off[b] + wid; j < D.soc_off[b + 1]; j += nw) {
    const int st0 = D.soc_start[j], dim = D.soc_dim[j];
    const double* w = c.W + st0;
    double nu2 = 0.0, dot = 0.0;   // dot = u . G_u
    for (int i = 1 + lane; i < dim; i += 32) {
      const double wi = w[i];
      nu2 += wi * wi;
      dot += wi * (gs[st0 + i] + rho * gy[st0 + i]);
    }
    nu2 = warp_sum(nu2); dot = warp_sum(dot);
    const double t = w[0], nu = sqrt(nu2);
    const int br = soc_branch(t, nu);
    const double Gt = gs[st0] + rho * gy[st0];
    const double dh = (br == 2) ? dot / nu : 0.0;       // uhat . G_u
    const double tn = (br == 2) ? t / nu : 0.0;
    for (int i = lane; i < dim; i += 32) {
      const double gyv = gy[st0 + i];
      const double G = gs[st0 + i] + rho * gyv;
      double v;
      if (br == 0) v = G;
      else if (br == 1) v = 0.0;
      else if (i == 0) v = 0.5 * (Gt + dh);
      else { const double uh = w[i] / nu; v = 0.5 * (Gt * uh + (1.0 + tn) * G - tn * dh * uh); }
      const double gw = -rho * gyv + v;
      c.GW[st0 + i] = gw;
      acc[0] += gyv * (s1[st0 + i] - w[i]);
      acc[1] += gw * y[st0 + i];
    }
  }
  block_sum<2>(acc, c.sh);
  out_part[0] = acc[0]; out_part[1] = acc[1];
}

// Phase 2: B5-B9 with the adjoint solve; needs GW complete on every row (PSD rows written by the PSD kernels).
template <typename T>
__device__ void bwd_post(const BatchDev<T>& D, Prob<T>& c, const BwdPtrs& Q, const double* part, int k, int* flag,
                         int* iters) {
  const int b = c.b, tid = threadIdx.x, nt = blockDim.x;
  const long long v0 = D.var_off[b], r0 = D.row_off[b];
  const double *x = Q.Zk + v0, *s = Q.Zk + D.N + r0;
  const double* gx1 = Q.Gin + v0;
  double *gx = Q.Gout + v0, *gs = Q.Gout + D.N + r0, *gy = Q.Gout + D.N + D.Mtot + r0;
  const double *xt = Q.XT + v0, *st = Q.ST + r0;
  const double al = c.alpha, rho = c.rho, sg = c.sigma;
  double d_gy_sw = part[0], d_gw_y = part[1];
  for (int j = D.psdblk_off[b]; j < D.psdblk_off[b + 1]; ++j) { d_gy_sw += D.psd_part[2 * j]; d_gw_y += D.psd_part[2 * j + 1]; }
  // B6: rhs = alpha g_x+ - A'(alpha g_w)   (g_st = alpha g_w)
  spmv_rows<double>(c.n, c.AT_rp, D.AT_ci, D.AT_v, c.GW, D.AT_G,
                    [&](int row, double a) { c.xi[row] = al * (gx1[row] - a); });
  __syncthreads();
  // B7: adjoint solve M lam = g_xt (Eq. 5), zero start
  *iters += solve_M(D, c, c.xi, (const double*)nullptr, c.lam, flag);
  // u = A lam; B7+B9 combined: g_rho += <u, st - s> (cancellation-free form of Eq. 6 + RHS term)
  double acc[3] = {0.0, 0.0, 0.0};   // rho, alpha, sigma
  spmv_rows<double>(c.m, c.A_rp, D.A_ci, D.A_v, c.lam, D.A_G, [&](int row, double u) {
    const double gw = c.GW[row];
    const double ds = st[row] - s[row];
    acc[0] += u * ds;
    acc[1] += gw * ds;                                  // B5: <g_vhat, st - s>
    gs[row] = (1.0 - al) * gw - rho * u;                // B5 + B9
    gy[row] = -gw / rho - u;                            // B4 + B9
  });
  for (int i = tid; i < c.n; i += nt) {
    const double g1 = gx1[i], l = c.lam[i], dx = xt[i] - x[i];
    acc[1] += g1 * dx;                                  // B5: <g_x+, xt - x>
    acc[2] -= l * dx;                                   // B7+B8: <lam, x - xt>
    gx[i] = (1.0 - al) * g1 + sg * l;                   // B5 + B8
  }
  block_sum<3>(acc, c.sh);
  if (tid == 0) {
    const size_t o = (size_t)k * D.B + b;
    Q.g_rho_pb[o] = acc[0] + d_gy_sw + d_gw_y / (rho * rho);   // B1 + B4 + (B7+B9)
    Q.g_alpha_pb[o] = acc[1];
    Q.g_sigma_pb[o] = acc[2];
  }
}

template <typename T>
__global__ void __launch_bounds__(1024) k_bwd(BatchDev<T> D, Hyper<T> H, BwdPtrs Q, int k, int phase) {
  // phase 0: pre + post fused (no PSD blocks anywhere); 1: pre only; 2: post only
  __shared__ double sh[3 * 32];
  const int b = blockIdx.x;
  Prob<T> c(D, b, sh);
  c.rho = H.rho_at(k, b); c.alpha = H.alpha_at(k, b); c.sigma = H.sigma;
  int flag = 0, iters = 0;
  double part[2];
  if (phase != 2) {
    bwd_pre(D, c, Q, part, &flag, &iters);
    if (phase == 1 && threadIdx.x == 0) { Q.part_pre[2 * b] = part[0]; Q.part_pre[2 * b + 1] = part[1]; }
  } else {
    part[0] = Q.part_pre[2 * b]; part[1] = Q.part_pre[2 * b + 1];
  }
  if (phase != 1) bwd_post(D, c, Q, part, k, &flag, &iters);
  if (threadIdx.x == 0) {
    D.cg_iters[b] += iters;
    if (flag) D.flags[b] |= flag;
  }
}

// ---- small utility kernels -------------------------------------------------------------------------------
template <typename T>
__global__ void k_load_vec(double* dst, const T* src, long long n) {   // dst = src (NULL -> 0)
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
    dst[i] = src ? (double)src[i] : 0.0;
}
template <typename T>
__global__ void k_store_vec(T* dst, const double* src, long long n) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
    dst[i] = (T)src[i];
}
// Single-block reduction of the per-problem partials into the caller's layout (deterministic order).
// PER_ITER: g[k] = sum_b pb[k][b], g_sigma[0] = sum_{k,b}; PER_PROBLEM: g[k][b] = pb[k][b], g_sigma[b] = sum_k.
template <typename T>
__global__ void __launch_bounds__(256) k_reduce_grads(const double* rho_pb, const double* alpha_pb,
                                                      const double* sigma_pb, int K, int B, int per_problem,
                                                      T* g_rho, T* g_alpha, T* g_sigma) {
  __shared__ double sh[32];
  const int tid = threadIdx.x, nt = blockDim.x;
  if (!per_problem) {
    double sg[1] = {0.0};
    for (int k = tid; k < K; k += nt) {
      double a = 0.0, c = 0.0, e = 0.0;
      for (int b = 0; b < B; ++b) {
        a += rho_pb[(size_t)k * B + b]; c += alpha_pb[(size_t)k * B + b]; e += sigma_pb[(size_t)k * B + b];
      }
      if (g_rho) g_rho[k] = (T)a;
      if (g_alpha) g_alpha[k] = (T)c;
      sg[0] += e;
    }
    block_sum<1>(sg, sh);
    if (tid == 0 && g_sigma) g_sigma[0] = (T)sg[0];
  } else {
    for (int t = tid; t < K * B; t += nt) {
      if (g_rho) g_rho[t] = (T)rho_pb[t];
      if (g_alpha) g_alpha[t] = (T)alpha_pb[t];
    }
    for (int b = tid; b < B; b += nt) {
      double e = 0.0;
      for (int k = 0; k < K; ++k) e += sigma_pb[(size_t)k * B + b];
      if (g_sigma) g_sigma[b] = (T)e;
    }
  }
}

}  // namespace cdu

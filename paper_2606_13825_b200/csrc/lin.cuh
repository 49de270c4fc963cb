// lin.cuh - per-problem linear-system step, relaxation, separable/SOC cones, and their reverse.
//
// One TEAM owns one problem instance at a time ("super-batch" of PAPER.md L306 held as batched CSR with per-problem
// offsets; CG convergence is decided per problem on the device, never by the host). A team is one CTA, or - when
// the batch has fewer problems than the GPU has SMs - a thread-block cluster of C CTAs that split the rows of every
// pass and reduce dot products through distributed shared memory. Teams are persistent: the grid is sized so that the
// matrices of the problems in flight stay resident in the 126 MB L2 across the CG iterations, and loops over the batch.
//   forward  : S1 xi assembly, S2 PCG on M = P + sigma I + rho A'A (Eq. 4, Jacobi preconditioner L294),
//              S3 st = b - A xt, S4 relaxation (Eq. 3c-3d), S5 zero/nonneg/SOC projection, S7 dual
//              update (Eq. 3e) - SURVEY.md 8(a).
//   backward : S9 (separable + SOC part), S10, S11 adjoint PCG (Eq. 5), S12 Eq. 6 (L90) and the RHS terms.
// The iterate and every reduction are fp64; matrices, CG vectors and the preconditioner are T. Column indices are IT
// (uint16_t when every n_b, m_b < 65536). A fully dense P is stored without indices and, if it fits, cached in shared
// memory together with the CG vectors.
#pragma once
#include <cooperative_groups.h>
#include "common.cuh"

namespace cdu {
namespace cg = cooperative_groups;

// Sliced ELL with row chunks: every row is cut into chunks of at most 32 elements; the chunks of a problem are sorted
// by length and packed 32 to a slab, one per lane, stored lane-interleaved in element PAIRS (pair k of the 32 chunks
// is contiguous: 32 x (v0, v1) and 32 x (c0, c1)), so a warp walks a slab with one coalesced 8-byte value load and one
// index load per two elements, 16 elements of every lane in flight at a time, plus one gather and one FMA per element. A row of one chunk is finished in its lane (crow >= 0); the chunks of a longer row leave partial sums in
// consecutive scratch slots (crow = -(slot + 1)) that are summed in chunk order afterwards (mrow). Padding is
// value 0 / column 0. Fixed summation order: bit-reproducible.
constexpr int SELL_NONE = -2147483647 - 1;
template <typename TV, typename IT>
struct Sell {
  const int* sl_base;    // [B+1] first slab of each problem
  const int* slab_off;   // [nslab+1] first pair column of each slab (a column = 32 lanes x 2 elements)
  const TV* val; const IT* idx;
  const int* crow;       // [nslab*32]
  const int* mr_base;    // [B+1] first multi-chunk row of each problem
  const int4* mrow;      // (row, first slot, number of slots, -)
};

// wide teams (Team<2> below): CTAs of a cooperative launch that meet at a global counter
struct WideTab {
  int C;                 // CTAs per wide team
  unsigned* bar;         // [teams] arrival counters, zeroed by the host before every launch
  double* slots;         // [teams][2][C][4]
};

template <typename T, typename IT>
struct BatchDev {
  int B;
  const int *var_off, *row_off;                        // [B+1]
  const int *A_rp;  const IT* A_ci;  const T* A_v;  int A_G;   // A   : rows = constraints, local column index
  const int *AT_rp; const IT* AT_ci; const T* AT_v; int AT_G;  // A^T : rows = variables,   local row index
  const int *P_rp;  const IT* P_ci;  const T* P_v;  int P_G;   // P   : full symmetric storage (CSR), or
  int P_dense; const long long* P_off;                 //       dense row-major n_b x n_b blocks at P_v + P_off[b]
  int P_smem, vec_smem;                                // dense P / CG vectors live in dynamic shared memory
  // sliced-ELL chunk format (single-CTA teams), built by cdu_create - see Sell below.
  int batched, nmax, mmax, sell_slots;
  Sell<T, IT> SA, SAT, SP;
  const T *q, *b, *diagP, *colsq;
  const uint8_t* rowkind;                              // per row: cone kind
  const int *soc_off, *soc_start, *soc_dim;            // per problem SOC list (start = local row)
  const int *psdblk_off;                               // [B+1] PSD blocks of each problem
  double *xi, *rd, *tm, *W, *GW, *lam;                 // fp64 scratch, sized sum n / sum m
  T *r, *p, *Ap, *d, *dinv, *tA;                       // CG vectors (global copies; unused parts when vec_smem)
  double tol, tol_ref;
  int maxit, refine;
  int *cg_iters, *cg_iters0, *cg_max, *flags;          // [B] statistics (cg_iters0: iterations of pass 0 only, i.e. without refinement)
  double* psd_part;                                    // [nblk][2] partial dots written by the PSD backward
  long long N, Mtot;
  WideTab wide;                                        // wide teams (MULTI == 2)
};

template <typename T>
struct Hyper {  // per-iteration hyper-parameters as the caller laid them out (cdu_rho_mode)
  const T* rho; const T* alpha; int kstride, pstride; double sigma;
  const T* rho_row = nullptr; long long mstride = 0;   // CDU_RHO_PER_ROW: rho_row[k][sum m_b] (constant inside SOC / PSD blocks)
  __device__ double rho_at(int k, int b) const { return (double)rho[(size_t)k * kstride + (size_t)b * pstride]; }
  // rho of the cone block that starts at global row `grow` of problem b
  __device__ double rho_blk(int k, int b, long long grow) const { return rho_row ? (double)rho_row[(size_t)k * mstride + grow] : rho_at(k, b); }
  __device__ const T* rows_of(int k, long long r0) const { return rho_row ? rho_row + (size_t)k * mstride + r0 : nullptr; }
  __device__ double alpha_at(int k, int b) const { return (double)alpha[(size_t)k * kstride + (size_t)b * pstride]; }
};

// ---- team = CTA (MULTI 0), thread-block cluster (1) or "wide" team (2) ---------------------------------------
// A wide team is any number of co-resident CTAs (cooperative launch) that meet at a counter in global memory and
// exchange partial sums through global memory: for the few-large-problems regime (Fig. 2 workload, L247-255), where a
// 16-CTA cluster would leave most of the GPU idle and the matrices do not fit L2.
template <int MULTI>
struct Team {
  int C, rank, parity;
  double* sh;       // [3*32] block_sum scratch
  double* slots;    // [2][4] partials exchanged through DSMEM
  double* bc;       // [4] broadcast
  unsigned* wbar; unsigned wgen; double* wslots;     // wide teams
  __device__ void init(double* sh_, double* slots_, double* bc_, const WideTab& W) {
    sh = sh_; slots = slots_; bc = bc_; parity = 0; wbar = nullptr; wgen = 0; wslots = nullptr;
    if (MULTI == 1) { cg::cluster_group cl = cg::this_cluster(); C = (int)cl.num_blocks(); rank = (int)cl.block_rank(); }
    else if (MULTI == 2) {
      C = W.C; rank = (int)blockIdx.x % C;
      const int team = (int)blockIdx.x / C;
      wbar = W.bar + team; wslots = W.slots + (size_t)team * 2 * C * 4;
    } else { C = 1; rank = 0; }
  }
  __device__ __forceinline__ void sync() {
    if (MULTI == 1) cg::this_cluster().sync();
    else if (MULTI == 2) {
      __syncthreads();
      if (threadIdx.x == 0) {
        ++wgen;
        __threadfence();
        atomicAdd(wbar, 1u);
        const unsigned target = wgen * (unsigned)C;
        unsigned v;
        do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(wbar) : "memory"); } while (v < target);
      }
      __syncthreads();
    } else __syncthreads();
  }
  __device__ __forceinline__ void range(int len, int& lo, int& hi) const {
    if (MULTI) { lo = (int)((long long)len * rank / C); hi = (int)((long long)len * (rank + 1) / C); }
    else { lo = 0; hi = len; }
  }
  // Deterministic team-wide sum; every thread of every CTA returns the same bits.
  template <int NV> __device__ void sum(double (&v)[NV]) {
    block_sum<NV>(v, sh);
    if (MULTI == 1) {
      double* slot = slots + parity * 4;
      if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < NV; ++i) slot[i] = v[i];
      }
      cg::cluster_group cl = cg::this_cluster();
      cl.sync();
      if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        const double* rs = cl.map_shared_rank(slot, lane < C ? lane : 0);
#pragma unroll
        for (int i = 0; i < NV; ++i) {
          const double mine = lane < C ? rs[i] : 0.0;
          double t = 0.0;
          for (int r = 0; r < C; ++r) t += __shfl_sync(0xffffffffu, mine, r);
          if (lane == 0) bc[i] = t;
        }
      }
      __syncthreads();
#pragma unroll
      for (int i = 0; i < NV; ++i) v[i] = bc[i];
      __syncthreads();
      parity ^= 1;
    } else if (MULTI == 2) {
      double* mine = wslots + ((size_t)parity * C + rank) * 4;
      if (threadIdx.x == 0) {
#pragma unroll
        for (int i = 0; i < NV; ++i) mine[i] = v[i];
      }
      sync();
      if (threadIdx.x < 32) {       // lane l adds ranks l, l + 32, ... in order, then a fixed shuffle tree
        const int lane = threadIdx.x;
#pragma unroll
        for (int i = 0; i < NV; ++i) {
          double t = 0.0;
          for (int r = lane; r < C; r += 32) t += __ldcg(wslots + ((size_t)parity * C + r) * 4 + i);
          t = warp_sum(t);
          if (lane == 0) bc[i] = t;
        }
      }
      __syncthreads();
#pragma unroll
      for (int i = 0; i < NV; ++i) v[i] = bc[i];
      __syncthreads();
      parity ^= 1;
    }
  }
};

template <int MULTI, typename TX> __device__ __forceinline__ TX ldv(const TX* x) {
  if (MULTI == 1) return __ldcg(x);   // written by another CTA of the cluster during this launch: read at L2
  return *x;                          // wide teams: every phase ends in Team::sync, whose gpu-scope fence drops the SM's L1 lines
}

// y = op(rows [lo,hi)) . x with a group of G (power of two <= 32) lanes per row; emit(row, dot) runs on lane 0.
template <typename TACC, int MULTI, typename TV, typename IT, typename TX, typename F>
__device__ __forceinline__ void spmv_rows(int lo, int hi, const int* __restrict__ rp, const IT* __restrict__ ci,
                                          const TV* __restrict__ v, const TX* x, int G, F emit) {
  const int tid = threadIdx.x;
  const int gl = tid & (G - 1);
  const int gid = tid / G, ng = blockDim.x / G;
  for (int row0 = lo; row0 < hi; row0 += ng) {
    const int row = row0 + gid;
    TACC acc = (TACC)0;
    if (row < hi) {
      const int e0 = __ldg(rp + row), e1 = __ldg(rp + row + 1);
      // eight independent (value, index) loads in flight per lane, then the eight gathers; out-of-row slots read element
      // e0 with weight 0, so a row of any length costs ceil(len / 8G) round trips and no serial tail
      for (int e = e0 + gl; e < e1; e += 8 * G) {
        TV vv[8]; int cc[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          const int idx = e + u * G;
          const bool ok = idx < e1;
          vv[u] = ok ? __ldg(v + idx) : (TV)0;
          cc[u] = ok ? (int)__ldg(ci + idx) : (int)__ldg(ci + e0);
        }
        TX xx[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) xx[u] = ldv<MULTI>(x + cc[u]);
#pragma unroll
        for (int u = 0; u < 8; ++u) acc += (TACC)vv[u] * (TACC)xx[u];
      }
    }
    for (int o = G >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (row < hi && gl == 0) emit(row, acc);
  }
}

// Dense row-major block (n x n, global or shared): one warp per row.
template <typename TACC, int MULTI, typename TV, typename TX, typename F>
__device__ __forceinline__ void dense_rows(int lo, int hi, int n, const TV* __restrict__ Pm, const TX* x, F emit) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  for (int row = lo + wid; row < hi; row += nw) {
    const TV* pr = Pm + (size_t)row * n;
    TACC a0 = (TACC)0, a1 = (TACC)0;
    int j = lane;
    for (; j + 32 < n; j += 64) {
      a0 += (TACC)pr[j] * (TACC)ldv<MULTI>(x + j);
      a1 += (TACC)pr[j + 32] * (TACC)ldv<MULTI>(x + j + 32);
    }
    if (j < n) a0 += (TACC)pr[j] * (TACC)ldv<MULTI>(x + j);
    a0 += a1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a0 += __shfl_xor_sync(0xffffffffu, a0, o);
    if (lane == 0) emit(row, a0);
  }
}

// two consecutive elements of a lane's chunk in one load (read-only path)
__device__ __forceinline__ void ld_pair(const float* p, float& a, float& b) { const float2 t = __ldg(reinterpret_cast<const float2*>(p)); a = t.x; b = t.y; }
__device__ __forceinline__ void ld_pair(const double* p, double& a, double& b) { const double2 t = __ldg(reinterpret_cast<const double2*>(p)); a = t.x; b = t.y; }
__device__ __forceinline__ void ld_pair(const int* p, int& a, int& b) { const int2 t = __ldg(reinterpret_cast<const int2*>(p)); a = t.x; b = t.y; }
__device__ __forceinline__ void ld_pair(const uint16_t* p, int& a, int& b) {
  const unsigned t = __ldg(reinterpret_cast<const unsigned*>(p)); a = (int)(t & 0xffffu); b = (int)(t >> 16);
}

// ---- sliced-ELL rows: one warp per slab ---------------------------------------------------------------------
// emit(row, dot) runs exactly once per row (any thread). Contains CTA barriers: every thread of the CTA must call.
template <typename TACC, typename TV, typename IT, typename TX, typename F>
__device__ __forceinline__ void sell_rows(const Sell<TV, IT>& S, int b, const TX* x, TACC* scratch, F emit) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int s0 = __ldg(S.sl_base + b), s1 = __ldg(S.sl_base + b + 1);
  for (int sl = s0 + warp; sl < s1; sl += nw) {
    const int e0 = __ldg(S.slab_off + sl), lp = __ldg(S.slab_off + sl + 1) - e0;     // element PAIRS per lane
    const TV* __restrict__ v = S.val + ((size_t)e0 * 32 + lane) * 2;
    const IT* __restrict__ ci = S.idx + ((size_t)e0 * 32 + lane) * 2;
    TACC a0 = (TACC)0, a1 = (TACC)0;
    int k = 0;
    for (; k + 8 <= lp; k += 8) {            // 16 elements of the chunk in flight per lane
      TV v0[8], v1[8]; int c0[8], c1[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) { ld_pair(v + (size_t)(k + j) * 64, v0[j], v1[j]); ld_pair(ci + (size_t)(k + j) * 64, c0[j], c1[j]); }
#pragma unroll
      for (int j = 0; j < 8; ++j) { a0 += (TACC)v0[j] * (TACC)x[c0[j]]; a1 += (TACC)v1[j] * (TACC)x[c1[j]]; }
    }
    for (; k < lp; ++k) {
      TV v0, v1; int c0, c1;
      ld_pair(v + (size_t)k * 64, v0, v1); ld_pair(ci + (size_t)k * 64, c0, c1);
      a0 += (TACC)v0 * (TACC)x[c0]; a1 += (TACC)v1 * (TACC)x[c1];
    }
    a0 += a1;
    const int cr = __ldg(S.crow + (size_t)sl * 32 + lane);
    if (cr >= 0) emit(cr, a0);
    else if (cr != SELL_NONE) scratch[-cr - 1] = a0;
  }
  __syncthreads();
  const int m0 = __ldg(S.mr_base + b), m1 = __ldg(S.mr_base + b + 1);
  for (int j = m0 + threadIdx.x; j < m1; j += blockDim.x) {
    const int4 d = __ldg(S.mrow + j);
    TACC a = (TACC)0;
    for (int q = 0; q < d.z; ++q) a += scratch[d.y + q];
    emit(d.x, a);
  }
  __syncthreads();
}

template <typename T, typename IT, int MULTI>
struct Prob {  // one problem's view of the batch, as seen by one CTA of its team
  int n, m, b;
  int nlo, nhi, mlo, mhi;             // this CTA's share of the variables / rows
  const int *A_rp, *AT_rp, *P_rp;
  const T* Pd;                        // dense P block (global or shared) or NULL
  const T *q, *bv, *diagP, *colsq;
  double *xi, *rd, *tm, *W, *GW, *lam;
  T *r, *p, *Ap, *d, *dinv, *tA;
  double rho, alpha, sigma;
  const T* rrow = nullptr;            // per-row rho of this problem at this iteration (NULL: the scalar rho)
  __device__ __forceinline__ double rh(int row) const { return rrow ? (double)rrow[row] : rho; }
  Team<MULTI>* team;
  double* scratch;                    // partial sums of multi-chunk rows (sell_rows), D.sell_slots doubles
  __device__ Prob(const BatchDev<T, IT>& D, int b_, Team<MULTI>* tm_, unsigned char* dsm) : b(b_), team(tm_) {
    const int v0 = D.var_off[b], r0 = D.row_off[b];
    n = D.var_off[b + 1] - v0; m = D.row_off[b + 1] - r0;
    team->range(n, nlo, nhi); team->range(m, mlo, mhi);
    A_rp = D.A_rp + r0; AT_rp = D.AT_rp + v0; P_rp = D.P_rp + v0;
    q = D.q + v0; bv = D.b + r0; diagP = D.diagP + v0; colsq = D.colsq + v0;
    xi = D.xi + v0; rd = D.rd + v0; lam = D.lam + v0; tm = D.tm + r0; W = D.W + r0; GW = D.GW + r0;
    Pd = D.P_dense ? D.P_v + D.P_off[b] : nullptr;
    scratch = nullptr;
    if (D.batched) {
      scratch = reinterpret_cast<double*>(dsm);
      dsm += (((size_t)D.sell_slots + 1) & ~(size_t)1) * sizeof(double);
    }
    T* sv = reinterpret_cast<T*>(dsm);
    if (D.P_smem) {   // cache the dense P of this problem (single-CTA teams only)
      const size_t nn = (size_t)n * n;
      __syncthreads();   // the previous problem's readers are done
      for (size_t t = threadIdx.x; t < nn; t += blockDim.x) sv[t] = Pd[t];
      Pd = sv; sv += (nn + 3) & ~(size_t)3;
    }
    if (D.vec_smem) {
      const int ns = (n + 3) & ~3;
      r = sv; p = r + ns; Ap = p + ns; d = Ap + ns; dinv = d + ns; tA = dinv + ns;
    } else {
      r = D.r + v0; p = D.p + v0; Ap = D.Ap + v0; d = D.d + v0; dinv = D.dinv + v0; tA = D.tA + r0;
    }
    __syncthreads();
  }
};

// One pass over the rows of A, A^T or P owned by this CTA: warp batches (single-CTA teams) or lane groups per row.
template <typename TACC, typename T, typename IT, int MULTI, typename TX, typename F>
__device__ __forceinline__ void rows_A(const BatchDev<T, IT>& D, const Prob<T, IT, MULTI>& c, const TX* x, F emit) {
  if (D.batched) sell_rows<TACC>(D.SA, c.b, x, reinterpret_cast<TACC*>(c.scratch), emit);
  else spmv_rows<TACC, MULTI>(c.mlo, c.mhi, c.A_rp, D.A_ci, D.A_v, x, D.A_G, emit);
}
template <typename TACC, typename T, typename IT, int MULTI, typename TX, typename F>
__device__ __forceinline__ void rows_AT(const BatchDev<T, IT>& D, const Prob<T, IT, MULTI>& c, const TX* x, F emit) {
  if (D.batched) sell_rows<TACC>(D.SAT, c.b, x, reinterpret_cast<TACC*>(c.scratch), emit);
  else spmv_rows<TACC, MULTI>(c.nlo, c.nhi, c.AT_rp, D.AT_ci, D.AT_v, x, D.AT_G, emit);
}
template <typename TACC, typename T, typename IT, int MULTI, typename TX, typename F>
__device__ __forceinline__ void rows_P(const BatchDev<T, IT>& D, const Prob<T, IT, MULTI>& c, const TX* x, F emit) {
  if (c.Pd) dense_rows<TACC, MULTI>(c.nlo, c.nhi, c.n, c.Pd, x, emit);
  else if (D.batched) sell_rows<TACC>(D.SP, c.b, x, reinterpret_cast<TACC*>(c.scratch), emit);
  else spmv_rows<TACC, MULTI>(c.nlo, c.nhi, c.P_rp, D.P_ci, D.P_v, x, D.P_G, emit);
}

// q = M p for the CG: tA = rho A p ; Ap = A' tA + P p + sigma p ; returns the team-wide <p, Ap>.
template <typename T, typename IT, int MULTI>
__device__ __forceinline__ double apply_M(const BatchDev<T, IT>& D, const Prob<T, IT, MULTI>& c) {
  const T sigT = (T)c.sigma;
  rows_A<T>(D, c, c.p, [&](int row, T a) { c.tA[row] = (T)c.rh(row) * a; });
  c.team->sync();
  rows_AT<T>(D, c, c.tA, [&](int row, T a) { c.Ap[row] = a; });
  __syncthreads();   // Ap rows are owned by this CTA
  double pap[1] = {0.0};
  auto fin = [&](int row, T a) {
    const T pi = c.p[row];
    const T ap = c.Ap[row] + a + sigT * pi;
    c.Ap[row] = ap;
    pap[0] += (double)pi * (double)ap;
  };
  rows_P<T>(D, c, c.p, fin);
  c.team->sum(pap);
  return pap[0];
}

// Jacobi-preconditioned CG on M d = r, d0 = 0. r (T) holds the right-hand side on entry (owner rows).
// Stops when the recursive residual satisfies ||r|| <= thresh (reading A5). Returns iterations.
template <typename T, typename IT, int MULTI>
__device__ int pcg(const BatchDev<T, IT>& D, const Prob<T, IT, MULTI>& c, double thresh, double rr0, int* flag) {
  const int tid = threadIdx.x, nt = blockDim.x;
  double acc[2] = {0.0, 0.0};
  for (int i = c.nlo + tid; i < c.nhi; i += nt) {
    const T ri = c.r[i], z = ri * c.dinv[i];
    c.d[i] = (T)0; c.p[i] = z;
    acc[0] += (double)ri * (double)z;
  }
  c.team->sum(acc);          // also orders the p writes before the first A pass
  double rz = acc[0];
  const double th2 = thresh * thresh;
  int it = 0;
  if (!(rr0 > th2)) return 0;
  while (it < D.maxit) {
    const double pap = apply_M(D, c);
    if (!(pap > 0.0)) { *flag |= FLAG_CG_CURV; break; }
    const T a = (T)(rz / pap);
    acc[0] = 0.0; acc[1] = 0.0;
    for (int i = c.nlo + tid; i < c.nhi; i += nt) {
      const T pi = c.p[i];
      c.d[i] += a * pi;
      const T ri = c.r[i] - a * c.Ap[i];
      c.r[i] = ri;
      const T z = ri * c.dinv[i];
      acc[0] += (double)ri * (double)ri;
      acc[1] += (double)ri * (double)z;
    }
    c.team->sum(acc);
    ++it;
    if (!(acc[0] > th2)) break;
    const T beta = (T)(acc[1] / rz);
    rz = acc[1];
    for (int i = c.nlo + tid; i < c.nhi; i += nt) c.p[i] = c.r[i] * c.dinv[i] + beta * c.p[i];
    c.team->sync();
  }
  if (it >= D.maxit) *flag |= FLAG_CG_CAP;
  return it;
}

// out = M^-1 rhs with start xbase (NULL = 0): pass 0 is PCG to tol ||rhs|| on the fp64 residual of the start
// (identical to CG started at xbase); each further pass re-evaluates the residual in fp64 and corrects
// (iterative refinement). Guards ||rhs|| = 0 => out = 0 (reading A5).
// rhs: owner rows valid. out: every row valid team-wide on return (after a team sync).
template <typename T, typename IT, int MULTI>
__device__ int solve_M(const BatchDev<T, IT>& D, const Prob<T, IT, MULTI>& c, const double* rhs, const double* xbase,
                       double* out, int* flag, int* it0) {
  const int tid = threadIdx.x, nt = blockDim.x;
  double acc[1] = {0.0};
  for (int i = c.nlo + tid; i < c.nhi; i += nt) {
    double dA = c.rho * (double)c.colsq[i];
    if (c.rrow) {        // diag(A' D(rho) A)_i = sum_r a_ri^2 rho_r
      dA = 0.0;
      for (int e = c.AT_rp[i]; e < c.AT_rp[i + 1]; ++e) { const double v = (double)D.AT_v[e]; dA += v * v * (double)c.rrow[(int)D.AT_ci[e]]; }
    }
    c.dinv[i] = (T)(1.0 / ((double)c.diagP[i] + c.sigma + dA));
    const double v = rhs[i];
    acc[0] += v * v;
    out[i] = xbase ? xbase[i] : 0.0;
  }
  c.team->sum(acc);
  const double nr2 = acc[0];
  if (!(nr2 > 0.0)) {
    for (int i = c.nlo + tid; i < c.nhi; i += nt) out[i] = 0.0;
    if (nr2 != nr2) *flag |= FLAG_NONFINITE;
    c.team->sync();
    return 0;
  }
  int total = 0;
  for (int pass = 0; pass <= D.refine; ++pass) {
    double rr0;
    if (pass == 0 && !xbase) {
      for (int i = c.nlo + tid; i < c.nhi; i += nt) c.r[i] = (T)rhs[i];
      rr0 = nr2;
      __syncthreads();
    } else {  // r = rhs - M out, fp64
      rows_A<double>(D, c, out, [&](int row, double a) { c.tm[row] = c.rh(row) * a; });
      c.team->sync();
      rows_AT<double>(D, c, c.tm, [&](int row, double a) { c.rd[row] = a; });
      __syncthreads();
      acc[0] = 0.0;
      auto fin = [&](int row, double a) {
        const double res = rhs[row] - (c.rd[row] + a + c.sigma * out[row]);
        c.r[row] = (T)res;
        acc[0] += res * res;
      };
      rows_P<double>(D, c, out, fin);
      c.team->sum(acc);
      rr0 = acc[0];
    }
    double thresh = D.tol * sqrt(nr2);
    if (pass > 0) {
      if (!(rr0 > 1e-28 * nr2)) break;
      thresh = D.tol_ref * sqrt(rr0);
    }
    const int it = pcg(D, c, thresh, rr0, flag);
    total += it;
    if (pass == 0) *it0 += it;
    if (it == 0 && pass == 0 && D.refine == 0) break;
    for (int i = c.nlo + tid; i < c.nhi; i += nt) out[i] += (double)c.d[i];
    c.team->sync();
  }
  c.team->sync();
  return total;
}

// xi and x-tilde of one step from z^k = (x, s, y): S1 + S2. Writes xt; st is produced by the caller's A pass.
template <typename T, typename IT, int MULTI>
__device__ int lin_solve_step(const BatchDev<T, IT>& D, const Prob<T, IT, MULTI>& c, const double* x, const double* s,
                              const double* y, double* xt, int* flag, int* it0, const double* xstart = nullptr) {
  const int tid = threadIdx.x, nt = blockDim.x;
  for (int i = c.mlo + tid; i < c.mhi; i += nt) c.tm[i] = c.rh(i) * ((double)c.bv[i] - s[i]) - y[i];
  c.team->sync();
  rows_AT<double>(D, c, c.tm, [&](int row, double a) { c.xi[row] = c.sigma * x[row] - (double)c.q[row] + a; });
  c.team->sync();   // tm is reused by solve_M's residual pass
  return solve_M(D, c, c.xi, xstart ? xstart : x, xt, flag, it0);
}

__device__ __forceinline__ int soc_branch(double t, double nu) { return (nu <= t) ? 0 : ((nu <= -t) ? 1 : 2); }

struct IterPtrs {
  const double* Zk;   // z^k  (x | s | y), sizes N, Mtot, Mtot
  double* Zk1;        // z^{k+1}
  double* XT;         // x-tilde store (checkpoint slot or scratch), size N
  double* ST;         // s-tilde store, size Mtot
  const double* XTprev = nullptr;   // x-tilde of the previous step (CG start), NULL: start from x^k
};

#define CDU_TEAM_PROLOGUE()                                                                   \
  __shared__ double sh_[3 * 32];                                                               \
  __shared__ double slots_[8];                                                                 \
  __shared__ double bc_[4];                                                                    \
  extern __shared__ __align__(16) unsigned char dsm_[];                                        \
  Team<MULTI> team;                                                                            \
  team.init(sh_, slots_, bc_, D.wide);                                                         \
  const int nteams = (int)gridDim.x / team.C, team_id = (int)blockIdx.x / team.C;

template <typename T, typename IT, int MULTI>
__global__ void __launch_bounds__(1024) k_fwd(BatchDev<T, IT> D, Hyper<T> H, IterPtrs I, int k) {
  CDU_TEAM_PROLOGUE();
  const int tid = threadIdx.x, nt = blockDim.x;
  for (int b = team_id; b < D.B; b += nteams) {
    Prob<T, IT, MULTI> c(D, b, &team, dsm_);
    c.rho = H.rho_row ? 0.0 : H.rho_at(k, b); c.alpha = H.alpha_at(k, b); c.sigma = H.sigma;
    const long long v0 = D.var_off[b], r0 = D.row_off[b];
    c.rrow = H.rows_of(k, r0);
    const double *x = I.Zk + v0, *s = I.Zk + D.N + r0, *y = I.Zk + D.N + D.Mtot + r0;
    double *x1 = I.Zk1 + v0, *s1 = I.Zk1 + D.N + r0, *y1 = I.Zk1 + D.N + D.Mtot + r0;
    double *xt = I.XT + v0, *st = I.ST + r0;
    int flag = 0, it0 = 0;
    const int iters = lin_solve_step(D, c, x, s, y, xt, &flag, &it0, I.XTprev ? I.XTprev + v0 : nullptr);
    const double al = c.alpha;
    const uint8_t* kind = D.rowkind + r0;
    rows_A<double>(D, c, xt, [&](int row, double a) {
      const double stv = (double)c.bv[row] - a;
      st[row] = stv;
      const double yv = y[row], rho = c.rh(row);
      const double w = al * stv + (1.0 - al) * s[row] - yv / rho;
      c.W[row] = w;
      const int kd = kind[row];
      if (kd <= KIND_NONNEG) {
        const double sp = (kd == KIND_NONNEG && w > 0.0) ? w : 0.0;
        s1[row] = sp;
        y1[row] = rho * (sp - w);
      }
    });
    for (int i = c.nlo + tid; i < c.nhi; i += nt) x1[i] = al * xt[i] + (1.0 - al) * x[i];
    const int nsoc = D.soc_off[b + 1] - D.soc_off[b];
    if (nsoc) {
      team.sync();   // W complete on every row of the problem
      // second-order cones of this problem: one warp per cone, cones dealt round-robin over the team's warps
      const int lane = tid & 31, nw = nt >> 5, gw = team.rank * nw + (tid >> 5), wtot = team.C * nw;
      for (int j = D.soc_off[b] + gw; j < D.soc_off[b + 1]; j += wtot) {
        const int st0 = D.soc_start[j], dim = D.soc_dim[j];
        const double* w = c.W + st0;
        const double rho = c.rh(st0);
        double nu2 = 0.0;
        for (int i = 1 + lane; i < dim; i += 32) { const double wi = ldv<MULTI>(w + i); nu2 += wi * wi; }
        nu2 = warp_sum(nu2);
        const double t = ldv<MULTI>(w), nu = sqrt(nu2);
        const int br = soc_branch(t, nu);
        const double cf = (br == 2) ? 0.5 * (t + nu) : 0.0;
        for (int i = lane; i < dim; i += 32) {
          const double wi = ldv<MULTI>(w + i);
          double sp;
          if (br == 0) sp = wi; else if (br == 1) sp = 0.0; else sp = (i == 0) ? cf : cf * wi / nu;
          s1[st0 + i] = sp;
          y1[st0 + i] = rho * (sp - wi);
        }
      }
    }
    if (tid == 0 && team.rank == 0) {
      D.cg_iters[b] += iters;
      D.cg_iters0[b] += it0;
      if (iters > D.cg_max[b]) D.cg_max[b] = iters;
      if (flag) D.flags[b] |= flag;
    }
    team.sync();   // scratch (tm, xi, CG vectors, shared memory) is reused by the team's next problem
  }
  if (MULTI) team.sync();   // no CTA leaves while a peer may still read its shared memory
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
  double* g_rho_row = nullptr;   // CDU_RHO_PER_ROW: [K][sum m_b] row-wise g_rho (Eq. 6 verbatim plus the RHS terms)
  int recompute;       // LEAN: re-solve for xt, st
  int warm_adjoint;    // not the first reverse step: D.lam holds the previous step's adjoint solution
};

// Phase 1 of the reverse step: (LEAN: re-solve), w, and B1/B2/B4 for zero, nonneg and SOC rows.
template <typename T, typename IT, int MULTI>
__device__ void bwd_pre(const BatchDev<T, IT>& D, Prob<T, IT, MULTI>& c, const BwdPtrs& Q, double* out_part, int* flag,
                        int* iters, int* it0) {
  const int b = c.b, tid = threadIdx.x, nt = blockDim.x;
  const long long v0 = D.var_off[b], r0 = D.row_off[b];
  const double *x = Q.Zk + v0, *s = Q.Zk + D.N + r0, *y = Q.Zk + D.N + D.Mtot + r0;
  const double* s1 = Q.Zk1 + D.N + r0;
  const double *gs = Q.Gin + D.N + r0, *gy = Q.Gin + D.N + D.Mtot + r0;
  double *xt = Q.XT + v0, *st = Q.ST + r0;
  const double al = c.alpha;
  if (Q.recompute) {
    *iters += lin_solve_step(D, c, x, s, y, xt, flag, it0);
    rows_A<double>(D, c, xt, [&](int row, double a) { st[row] = (double)c.bv[row] - a; });
    __syncthreads();
  }
  const uint8_t* kind = D.rowkind + r0;
  double acc[2] = {0.0, 0.0};   // [0]: <gy, s+ - w>, [1]: <gw, y>
  for (int i = c.mlo + tid; i < c.mhi; i += nt) {
    const double yv = y[i], rho = c.rh(i);
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
  const int nsoc = D.soc_off[b + 1] - D.soc_off[b];
  if (nsoc) {
    c.team->sync();
    const int lane = tid & 31, nw = nt >> 5, gwp = c.team->rank * nw + (tid >> 5), wtot = c.team->C * nw;
    for (int j = D.soc_off[b] + gwp; j < D.soc_off[b + 1]; j += wtot) {
      const int st0 = D.soc_start[j], dim = D.soc_dim[j];
      const double* w = c.W + st0;
      const double rho = c.rh(st0);
      double nu2 = 0.0, dot = 0.0;   // dot = u . G_u
      for (int i = 1 + lane; i < dim; i += 32) {
        const double wi = ldv<MULTI>(w + i);
        nu2 += wi * wi;
        dot += wi * (gs[st0 + i] + rho * gy[st0 + i]);
      }
      nu2 = warp_sum(nu2); dot = warp_sum(dot);
      const double t = ldv<MULTI>(w), nu = sqrt(nu2);
      const int br = soc_branch(t, nu);
      const double Gt = gs[st0] + rho * gy[st0];
      const double dh = (br == 2) ? dot / nu : 0.0;       // uhat . G_u
      const double tn = (br == 2) ? t / nu : 0.0;
      for (int i = lane; i < dim; i += 32) {
        const double gyv = gy[st0 + i];
        const double G = gs[st0 + i] + rho * gyv;
        const double wi = ldv<MULTI>(w + i);
        double v;
        if (br == 0) v = G;
        else if (br == 1) v = 0.0;
        else if (i == 0) v = 0.5 * (Gt + dh);
        else { const double uh = wi / nu; v = 0.5 * (Gt * uh + (1.0 + tn) * G - tn * dh * uh); }
        const double gw = -rho * gyv + v;
        c.GW[st0 + i] = gw;
        acc[0] += gyv * (s1[st0 + i] - wi);
        acc[1] += gw * y[st0 + i];
      }
    }
  }
  c.team->sum(acc);
  out_part[0] = acc[0]; out_part[1] = acc[1];
}

// Phase 2: B5-B9 with the adjoint solve; needs GW complete on every row (PSD rows written by the PSD kernels).
template <typename T, typename IT, int MULTI>
__device__ void bwd_post(const BatchDev<T, IT>& D, Prob<T, IT, MULTI>& c, const BwdPtrs& Q, const double* part, int k,
                         int* flag, int* iters, int* it0) {
  const int b = c.b, tid = threadIdx.x, nt = blockDim.x;
  const long long v0 = D.var_off[b], r0 = D.row_off[b];
  const double *x = Q.Zk + v0, *s = Q.Zk + D.N + r0;
  const double* gx1 = Q.Gin + v0;
  double *gx = Q.Gout + v0, *gs = Q.Gout + D.N + r0, *gy = Q.Gout + D.N + D.Mtot + r0;
  const double *xt = Q.XT + v0, *st = Q.ST + r0;
  const double al = c.alpha, sg = c.sigma;
  const double* gy1 = Q.Gin + D.N + D.Mtot + r0;         // per-row rho: the terms of g_rho that the scalar modes take from dots
  const double* s1 = Q.Zk1 + D.N + r0;
  const double* yk = Q.Zk + D.N + D.Mtot + r0;
  double* grow = Q.g_rho_row ? Q.g_rho_row + (size_t)k * D.Mtot + r0 : nullptr;
  double d_gy_sw = part[0], d_gw_y = part[1];
  for (int j = D.psdblk_off[b]; j < D.psdblk_off[b + 1]; ++j) { d_gy_sw += D.psd_part[2 * j]; d_gw_y += D.psd_part[2 * j + 1]; }
  // B6: rhs = alpha g_x+ - A'(alpha g_w)   (g_st = alpha g_w)
  rows_AT<double>(D, c, c.GW, [&](int row, double a) { c.xi[row] = al * (gx1[row] - a); });
  __syncthreads();
  // B7: adjoint solve M lam = g_xt (Eq. 5), zero start
  // Start: 0 (reading A5) or, when the forward solves of this problem needed many CG iterations, the lam of the previous
  // reverse step: the start costs one extra fp64 operator application, which only pays for long solves. Same solution to
  // the same tolerance either way; the choice depends on this unroll's forward only (results stay history independent).
  const bool warm = Q.warm_adjoint && D.cg_max[b] >= 12;
  *iters += solve_M(D, c, c.xi, warm ? (const double*)c.lam : (const double*)nullptr, c.lam, flag, it0);
  // u = A lam; B7+B9 combined: g_rho += <u, st - s> (cancellation-free form of Eq. 6 + RHS term)
  double acc[3] = {0.0, 0.0, 0.0};   // rho, alpha, sigma
  rows_A<double>(D, c, c.lam, [&](int row, double u) {
    const double gw = ldv<MULTI>(c.GW + row);   // SOC rows may have been written by a peer CTA
    const double ds = st[row] - s[row], rho = c.rh(row);
    acc[0] += u * ds;
    acc[1] += gw * ds;                                  // B5: <g_vhat, st - s>
    if (grow) grow[row] = u * ds + gy1[row] * (s1[row] - ldv<MULTI>(c.W + row)) + gw * yk[row] / (rho * rho);   // B1 + B4 + (B7+B9), row by row
    gs[row] = (1.0 - al) * gw - rho * u;                // B5 + B9
    gy[row] = -gw / rho - u;                            // B4 + B9
  });
  for (int i = c.nlo + tid; i < c.nhi; i += nt) {
    const double g1 = gx1[i], l = c.lam[i], dx = xt[i] - x[i];
    acc[1] += g1 * dx;                                  // B5: <g_x+, xt - x>
    acc[2] -= l * dx;                                   // B7+B8: <lam, x - xt>
    gx[i] = (1.0 - al) * g1 + sg * l;                   // B5 + B8
  }
  c.team->sum(acc);
  if (tid == 0 && c.team->rank == 0) {
    const size_t o = (size_t)k * D.B + b;
    Q.g_rho_pb[o] = grow ? 0.0 : acc[0] + d_gy_sw + d_gw_y / (c.rho * c.rho);   // B1 + B4 + (B7+B9)
    Q.g_alpha_pb[o] = acc[1];
    Q.g_sigma_pb[o] = acc[2];
  }
}

template <typename T, typename IT, int MULTI>
__global__ void __launch_bounds__(1024) k_bwd(BatchDev<T, IT> D, Hyper<T> H, BwdPtrs Q, int k, int phase) {
  // phase 0: pre + post fused (no PSD blocks anywhere); 1: pre only; 2: post only
  CDU_TEAM_PROLOGUE();
  for (int b = team_id; b < D.B; b += nteams) {
    Prob<T, IT, MULTI> c(D, b, &team, dsm_);
    c.rho = H.rho_row ? 0.0 : H.rho_at(k, b); c.alpha = H.alpha_at(k, b); c.sigma = H.sigma;
    c.rrow = H.rows_of(k, D.row_off[b]);
    int flag = 0, iters = 0, it0 = 0;
    double part[2];
    if (phase != 2) {
      bwd_pre(D, c, Q, part, &flag, &iters, &it0);
      if (phase == 1 && threadIdx.x == 0 && team.rank == 0) { Q.part_pre[2 * b] = part[0]; Q.part_pre[2 * b + 1] = part[1]; }
    } else {
      part[0] = Q.part_pre[2 * b]; part[1] = Q.part_pre[2 * b + 1];
    }
    if (phase != 1) bwd_post(D, c, Q, part, k, &flag, &iters, &it0);
    if (threadIdx.x == 0 && team.rank == 0) {
      D.cg_iters[b] += iters;
      D.cg_iters0[b] += it0;
      if (flag) D.flags[b] |= flag;
    }
    team.sync();
  }
  if (MULTI) team.sync();
}

// ---- small utility kernels -------------------------------------------------------------------------------
// Device-side validation of device-resident hyper-parameters (cdu.h): rho > 0, alpha in (0, 2). per_problem = B when the
// arrays are [K][B] (the flag goes to that problem), 0 when they are [K] (shared: every problem is flagged).
template <typename T>
__global__ void k_check_hyper(const T* rho, const T* alpha, long long cnt, int per_problem, int B, int* flags) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < cnt; i += (long long)gridDim.x * blockDim.x) {
    const T r = rho[i], a = alpha[i];
    if (!(r > (T)0) || !(a > (T)0) || !(a < (T)2)) {
      if (per_problem) atomicOr(flags + (int)(i % per_problem), FLAG_BAD_HYPER);
      else for (int b = 0; b < B; ++b) atomicOr(flags + b, FLAG_BAD_HYPER);
    }
  }
}
// per-row rho (CDU_RHO_PER_ROW): rho[k][row] > 0, flag on the problem that owns the row
template <typename T>
__global__ void k_check_hyper_rows(const T* rho, long long cnt, long long Mtot, const int* row_off, int B, int* flags) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < cnt; i += (long long)gridDim.x * blockDim.x) {
    if (!(rho[i] > (T)0)) {
      const int row = (int)(i % Mtot);
      int lo = 0, hi = B;
      while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (row_off[mid] <= row) lo = mid; else hi = mid; }
      atomicOr(flags + lo, FLAG_BAD_HYPER);
    }
  }
}

// Rectification of PAPER.md App. E (L343): a per-row rho is averaged over every SOC / PSD block and the mean is broadcast
// back over the block (the operation is its own adjoint, so the same kernel rectifies g_rho). One warp per (block, k).
template <typename T>
__global__ void k_rectify(T* rho, long long Mtot, const long long* blk_row0, const int* blk_rows, int nblk) {
  const int j = blockIdx.x, lane = threadIdx.x;
  if (j >= nblk) return;
  T* r = rho + (size_t)blockIdx.y * Mtot + blk_row0[j];
  const int n = blk_rows[j];
  double a = 0.0;
  for (int i = lane; i < n; i += 32) a += (double)r[i];
  a = warp_sum(a) / (double)n;
  for (int i = lane; i < n; i += 32) r[i] = (T)a;
}

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

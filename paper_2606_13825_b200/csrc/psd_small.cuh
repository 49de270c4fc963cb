// psd_small.cuh - PSD-cone projection and its Dalecki-Krein VJP for blocks that fit in shared memory.
//
//   forward : S = smat(w);  S = U L U' by two-sided cyclic Jacobi (round-robin parallel ordering, one CTA per
//             matrix, everything resident in shared memory, fixed-position tournament layout - see
//             jacobi_planes);  s+ = svec(U max(L,0) U')                                    (Eq. 7)
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

// ---------------------------------------------------------------------------------------------------------
// Two-sided cyclic Jacobi in shared memory, "fixed-position tournament" layout.
//
// The pe (even) indices sit on pe positions; positions 2q ("top") and 2q+1 ("bottom") are the pair rotated in
// every round, and after each round the rows/columns physically move one seat of the round-robin circle
// (top q -> top q+1, top h-1 -> bottom h-1, bottom q -> bottom q-1, bottom 0 -> top 1, top 0 fixed), so pe-1
// consecutive rounds meet every pair once. The matrix is held as h x h blocks of 2 x 2, split in four planes
//     plane 0: (top,top)  1: (top,bottom)  2: (bottom,top)  3: (bottom,bottom),   each h x ldh, ldh odd,
// double-buffered: block (q1,q2) is read from the current buffer with unit-stride, conflict-free loads, rotated
// (rows by pair q1, columns by pair q2) and its four entries are scattered to their next-round seats in the
// other buffer; only q1 <= q2 is computed, the mirror image is written too. Eigenvectors are kept transposed
// (Vt[player][coordinate], "player" = initial position), updated in place with lanes along the coordinate, and
// found through the small position->player table plr. No index arithmetic of the pairing is left in the loop.
// ---------------------------------------------------------------------------------------------------------
template <typename T> struct JacobiWs {
  T* P0; int pstride;    // 2 x (4 planes x h x ldh); buffer c at P0 + c * pstride
  T* Vt;                 // pe x pe
  T* cs;                 // 3 h  (sin, tau = sin/(1+cos), tan)
  int* plr0; int pe;     // 2 x pe   player at position; buffer c at plr0 + c * pe
  int4* mv;              // h        next-round seat offsets of pair q: (row-top, row-bottom, col-top, col-bottom)
  unsigned short* blk;   // h(h+1)/2 (q1 << 8 | q2), q1 <= q2, row after row
};
template <typename T> __host__ __device__ inline size_t jacobi_ws_bytes(int pe) {
  const size_t h = pe >> 1, ldh = h | 1;
  size_t b = (2 * 4 * h * ldh + (size_t)pe * pe + 3 * h) * sizeof(T);
  b = (b + 15) & ~(size_t)15;
  b += h * sizeof(int4) + 2 * (size_t)pe * sizeof(int) + ((h * (h + 1) / 2 + 1) & ~(size_t)1) * sizeof(unsigned short);
  return (b + 15) & ~(size_t)15;
}
template <typename T> __device__ __forceinline__ JacobiWs<T> jacobi_ws_carve(unsigned char* base, int pe) {
  const size_t h = pe >> 1, ldh = h | 1;
  JacobiWs<T> w;
  T* t = reinterpret_cast<T*>(base);
  w.P0 = t; w.pstride = (int)(4 * h * ldh); w.Vt = t + 8 * h * ldh; w.cs = w.Vt + (size_t)pe * pe;
  size_t off = ((2 * 4 * h * ldh + (size_t)pe * pe + 3 * h) * sizeof(T) + 15) & ~(size_t)15;
  w.mv = reinterpret_cast<int4*>(base + off); off += h * sizeof(int4);
  w.plr0 = reinterpret_cast<int*>(base + off); w.pe = pe; off += 2 * (size_t)pe * sizeof(int);
  w.blk = reinterpret_cast<unsigned short*>(base + off);
  return w;
}

__device__ __forceinline__ int seat_after(int pos, int h) {   // position after one round of the circle
  const int q = pos >> 1;
  if (!(pos & 1)) return q == 0 ? 0 : (q < h - 1 ? pos + 2 : 2 * (h - 1) + 1);
  return q == 0 ? (h > 1 ? 2 : 1) : pos - 2;
}

template <typename T> __device__ __forceinline__ void jacobi_angle(T aii, T ajj, T aij, T skip, T& sn, T& tau, T& tt) {
  sn = (T)0; tau = (T)0; tt = (T)0;
  if (fabs(aij) > skip) {
    // Rutishauser form: x' = x - s (y + tau x), y' = y + s (x - tau y), tau = s / (1 + c). The deviation from
    // orthogonality is O((1-c) eps) per rotation instead of O(eps), so V stays orthogonal to a few eps.
    const T th = (ajj - aii) / ((T)2 * aij);
    const T t = ((th >= (T)0) ? (T)1 : (T)-1) / (fabs(th) + sqrt((T)1 + th * th));
    const T c = (T)1 / sqrt((T)1 + t * t);
    sn = t * c; tau = sn / ((T)1 + c); tt = t;
  }
}

// smat(v [+ sc v2]) -> planes of buffer 0, zero padded to pe. v, v2: svec (fp64).
template <typename T>
__device__ __forceinline__ void load_smat_planes(int p, int pe, T* P0, const double* v, double sc, const double* v2) {
  const int h = pe >> 1, ldh = h | 1, psz = h * ldh;
  for (int t = threadIdx.x; t < pe * pe; t += blockDim.x) {
    const int b = t / pe, a = t - b * pe;   // column b, row a: consecutive threads walk down a column of the upper triangle
    T val = (T)0;
    if (a < p && b < p) {
      const int idx = a <= b ? svec_idx(a, b) : svec_idx(b, a);
      double x = v[idx];
      if (v2) x += sc * v2[idx];
      val = (T)(a == b ? x : x * 0.70710678118654752440);
    }
    P0[((a & 1) * 2 + (b & 1)) * psz + (a >> 1) * ldh + (b >> 1)] = val;
  }
}

// On entry buffer 0 holds the matrix. On exit: *cur_out = buffer holding the (numerically diagonal) matrix,
// plr[*cur_out][pos] = player whose eigenvalue sits on the diagonal at pos, Vt[player][:] = its eigenvector.
template <typename T>
__device__ int jacobi_planes(int pe, const JacobiWs<T>& w, double* shred, int max_sweeps, int* flag, int* cur_out) {
  const int tid = threadIdx.x, nt = blockDim.x;
  const int h = pe >> 1, ldh = h | 1, psz = h * ldh, nblk = h * (h + 1) / 2;
  // ---- one-time tables ----
  for (int t = tid; t < pe * pe; t += nt) { const int i = t / pe, a = t - i * pe; w.Vt[t] = (i == a) ? (T)1 : (T)0; }
  for (int pos = tid; pos < pe; pos += nt) w.plr0[pos] = pos;
  for (int q = tid; q < h; q += nt) {
    const int nt_ = seat_after(2 * q, h), nb_ = seat_after(2 * q + 1, h);
    int4 m;
    m.x = 2 * (nt_ & 1) * psz + (nt_ >> 1) * ldh;   // as a row
    m.y = 2 * (nb_ & 1) * psz + (nb_ >> 1) * ldh;
    m.z = (nt_ & 1) * psz + (nt_ >> 1);             // as a column
    m.w = (nb_ & 1) * psz + (nb_ >> 1);
    w.mv[q] = m;
  }
  for (int q1 = tid; q1 < h; q1 += nt) {
    int o = q1 * h - q1 * (q1 - 1) / 2;
    for (int q2 = q1; q2 < h; ++q2) w.blk[o++] = (unsigned short)((q1 << 8) | q2);
  }
  double acc[1] = {0.0};
  for (int t = tid; t < 4 * psz; t += nt) {
    const int r = t % ldh;
    if (r < h) { const double x = (double)w.P0[t]; acc[0] += x * x; }
  }
  block_sum<1>(acc, shred);   // also publishes the tables
  const double normF2 = acc[0];
  *cur_out = 0;
  if (!(normF2 > 0.0)) { if (normF2 != normF2) *flag |= FLAG_NONFINITE; return 0; }
  const double tol2 = 16.0 * (double)Eps<T>::v() * (double)Eps<T>::v() * normF2;
  const T skip = (T)(0.01 * sqrt(tol2) / pe);
  // V-update items (pair q, coordinate a), t = q pe + a, stepped incrementally
  const int vq0 = tid / pe, va0 = tid - vq0 * pe, dq = nt / pe, da = nt - dq * pe;
  int cur = 0, sweep = 0;
  for (; sweep < max_sweeps; ++sweep) {
    {   // off-diagonal mass
      const T* Pc = w.P0 + cur * w.pstride;
      acc[0] = 0.0;
      for (int t = tid; t < h * h; t += nt) {
        const int q1 = t / h, q2 = t - q1 * h, o = q1 * ldh + q2;
        const double b = (double)Pc[psz + o], c = (double)Pc[2 * psz + o];
        acc[0] += b * b + c * c;
        if (q1 != q2) { const double a = (double)Pc[o], d = (double)Pc[3 * psz + o]; acc[0] += a * a + d * d; }
      }
      block_sum<1>(acc, shred);
      if (!(acc[0] > tol2)) break;
    }
    for (int r = 0; r < pe - 1; ++r) {
      const T* Pc = w.P0 + cur * w.pstride;
      T* Pn = w.P0 + (cur ^ 1) * w.pstride;
      const int* plc = w.plr0 + cur * pe;
      int* pln = w.plr0 + (cur ^ 1) * pe;
      for (int q = tid; q < h; q += nt) {
        const int o = q * ldh + q;
        T sn, tau, tt;
        jacobi_angle<T>(Pc[o], Pc[3 * psz + o], Pc[psz + o], skip, sn, tau, tt);
        w.cs[3 * q] = sn; w.cs[3 * q + 1] = tau; w.cs[3 * q + 2] = tt;
      }
      __syncthreads();
      for (int t = tid; t < nblk; t += nt) {
        const int qq = w.blk[t], q1 = qq >> 8, q2 = qq & 255, o = q1 * ldh + q2;
        const int4 m1 = w.mv[q1], m2 = w.mv[q2];
        T a = Pc[o], d = Pc[3 * psz + o];
        if (q1 == q2) {
          const T g = w.cs[3 * q1 + 2] * Pc[psz + o];   // tan * a_ij
          a -= g; d += g;
          Pn[m1.x + m1.z] = a; Pn[m1.y + m1.w] = d; Pn[m1.x + m1.w] = (T)0; Pn[m1.y + m1.z] = (T)0;
        } else {
          const T b = Pc[psz + o], c = Pc[2 * psz + o];
          const T s1 = w.cs[3 * q1], t1 = w.cs[3 * q1 + 1], s2 = w.cs[3 * q2], t2 = w.cs[3 * q2 + 1];
          const T ra = a - s1 * (c + t1 * a), rc = c + s1 * (a - t1 * c);   // rows:  J1' S
          const T rb = b - s1 * (d + t1 * b), rd = d + s1 * (b - t1 * d);
          const T na = ra - s2 * (rb + t2 * ra), nb = rb + s2 * (ra - t2 * rb);   // cols: (.) J2
          const T nc = rc - s2 * (rd + t2 * rc), nd = rd + s2 * (rc - t2 * rd);
          Pn[m1.x + m2.z] = na; Pn[m1.x + m2.w] = nb; Pn[m1.y + m2.z] = nc; Pn[m1.y + m2.w] = nd;
          Pn[m2.x + m1.z] = na; Pn[m2.y + m1.z] = nb; Pn[m2.x + m1.w] = nc; Pn[m2.y + m1.w] = nd;   // mirror block
        }
      }
      for (int q = vq0, a = va0; q < h; ) {
        const T s = w.cs[3 * q];
        if (s != (T)0) {
          const T tau = w.cs[3 * q + 1];
          T* vi = w.Vt + plc[2 * q] * pe + a;
          T* vj = w.Vt + plc[2 * q + 1] * pe + a;
          const T x = *vi, y = *vj;
          *vi = x - s * (y + tau * x);
          *vj = y + s * (x - tau * y);
        }
        q += dq; a += da;
        if (a >= pe) { a -= pe; ++q; }
      }
      for (int pos = tid; pos < pe; pos += nt) pln[seat_after(pos, h)] = plc[pos];
      __syncthreads();
      cur ^= 1;
    }
  }
  if (sweep >= max_sweeps) *flag |= FLAG_EIG_CAP;
  *cur_out = cur;
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
  const int p = tab.p[blk], pe = (p + 1) & ~1;
  const int prob = tab.prob[blk];
  const long long row0 = tab.row0[blk];
  double* shred = reinterpret_cast<double*>(smem_raw);                 // 64 doubles
  const JacobiWs<T> ws = jacobi_ws_carve<T>(smem_raw + 512, pe);
  T* lp = reinterpret_cast<T*>(smem_raw + 512 + jacobi_ws_bytes<T>(pe));   // pe: max(lambda, 0) by player
  const double rho = H.rho_at(k, prob);
  const double* w = A.W + row0;
  load_smat_planes<T>(p, pe, ws.P0, w, 0.0, nullptr);
  __syncthreads();
  int flag = 0, cur = 0;
  const int sweeps = jacobi_planes<T>(pe, ws, shred, 40, &flag, &cur);
  const int h = pe >> 1, ldh = h | 1, psz = h * ldh;
  T* U = reinterpret_cast<T*>(A.Ustore) + tab.uoff[blk];   // rows = eigenvectors
  T* L = reinterpret_cast<T*>(A.Lstore) + tab.loff[blk];
  for (int pos = threadIdx.x; pos < pe; pos += blockDim.x) {
    const int q = pos >> 1, pl = ws.plr0[cur * pe + pos];
    const T l = ws.P0[cur * ws.pstride + ((pos & 1) ? 3 * psz : 0) + q * ldh + q];
    lp[pl] = l > (T)0 ? l : (T)0;
    if (pl < p) L[pl] = l;
  }
  for (int t = threadIdx.x; t < p * p; t += blockDim.x) { const int i = t / p, a = t - i * p; U[t] = ws.Vt[i * pe + a]; }
  __syncthreads();
  // rebuild (Eq. 7) + svec + dual update (Eq. 3e); only eigenpairs with lambda > 0 contribute
  const int nsv = p * (p + 1) / 2;
  double* s1 = A.S1 + row0;
  double* y1 = A.Y1 + row0;
  for (int t = threadIdx.x; t < nsv; t += blockDim.x) {
    int b = (int)((sqrt(8.0 * t + 1.0) - 1.0) * 0.5);
    while (b * (b + 1) / 2 > t) --b;
    while ((b + 1) * (b + 2) / 2 <= t) ++b;
    const int a = t - b * (b + 1) / 2;
    const T *va = ws.Vt + a, *vb = ws.Vt + b;
    T acc = (T)0;
    for (int i = 0; i < pe; ++i) {
      const T l = lp[i];
      if (l > (T)0) acc += va[i * pe] * l * vb[i * pe];
    }
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
  double* shred = reinterpret_cast<double*>(smem_raw);                 // 64 doubles
  const JacobiWs<T> ws = jacobi_ws_carve<T>(smem_raw + 512, pe);
  T* lam = reinterpret_cast<T*>(smem_raw + 512 + jacobi_ws_bytes<T>(pe));
  T* Vt = ws.Vt;            // Vt[i*pe + a] = V(a, i)
  T* G = ws.P0;             // the two p x p work matrices alias the Jacobi planes (dead after a recompute)
  T* Tm = G + pe * pe;
  const double rho = H.rho_at(k, prob);
  const double* w = A.W + row0;
  int flag = 0;
  if (A.recompute) {
    load_smat_planes<T>(p, pe, ws.P0, w, 0.0, nullptr);
    __syncthreads();
    int cur = 0;
    jacobi_planes<T>(pe, ws, shred, 40, &flag, &cur);
    const int h = pe >> 1, ldh = h | 1, psz = h * ldh;
    for (int pos = threadIdx.x; pos < pe; pos += blockDim.x)
      lam[ws.plr0[cur * pe + pos]] = ws.P0[cur * ws.pstride + ((pos & 1) ? 3 * psz : 0) + (pos >> 1) * ldh + (pos >> 1)];
    __syncthreads();
  } else {
    const T* U = reinterpret_cast<const T*>(A.Ustore) + tab.uoff[blk];
    const T* L = reinterpret_cast<const T*>(A.Lstore) + tab.loff[blk];
    for (int t = threadIdx.x; t < pe * pe; t += blockDim.x) {
      const int i = t / pe, a = t - i * pe;
      Vt[t] = (a < p && i < p) ? U[i * p + a] : ((a == i) ? (T)1 : (T)0);
    }
    for (int i = threadIdx.x; i < pe; i += blockDim.x) lam[i] = i < p ? L[i] : (T)0;
    __syncthreads();
  }
  const double* gs = A.Gs + row0;
  const double* gy = A.Gy + row0;
  load_smat<T>(p, pe, ld, G, gs, rho, gy);                 // G = smat(g_s+ + rho g_y+)
  __syncthreads();
  smem_gemm<T>(pe, G, ld, 1, Vt, 1, pe, Tm, ld);           // Tm = G V
  __syncthreads();
  smem_gemm<T>(pe, Vt, pe, 1, Tm, ld, 1, G, ld);           // C  = V' Tm
  __syncthreads();
  for (int t = threadIdx.x; t < pe * pe; t += blockDim.x) {
    const int i = t / pe, j = t - i * pe;
    G[i * ld + j] *= gamma_relu<T>(lam[i], lam[j]);
  }
  __syncthreads();
  smem_gemm<T>(pe, Vt, 1, pe, G, ld, 1, Tm, ld);           // Tm = V C
  __syncthreads();
  smem_gemm<T>(pe, Tm, ld, 1, Vt, pe, 1, G, ld);           // out = Tm V'
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

static inline size_t psd_small_smem_bytes(int p, size_t sz) {
  const int pe = (p + 1) & ~1;
  const size_t ws = sz == 4 ? jacobi_ws_bytes<float>(pe) : jacobi_ws_bytes<double>(pe);
  return 512 + ws + (((size_t)pe * sz + 15) & ~(size_t)15);
}
static inline size_t psd_small_smem_fwd(int p, size_t sz) { return psd_small_smem_bytes(p, sz); }
static inline size_t psd_small_smem_bwd(int p, size_t sz) { return psd_small_smem_bytes(p, sz); }

}  // namespace cdu

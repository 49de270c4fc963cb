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
// other buffer; only q1 <= q2 is computed, the mirror image is written too. Because seats never change, every
// thread owns the same <= MAXI blocks and eigenvector slices in every round and keeps their source and
// destination offsets in registers: no index arithmetic of the pairing is left in the loop.
// Eigenvectors are kept transposed (Vt[player][coordinate], "player" = initial position), updated in place
// with 16-byte accesses along the coordinate, and found through the small position->player table plr.
// The last two warps of the CTA are "angle" warps: while the work warps apply round r they evaluate, from the
// three entries involved, the pivots round r+1 will meet and write that round's rotations, so a round costs
// one barrier and the rotation set-up is off the critical path of the updates.
// ---------------------------------------------------------------------------------------------------------
template <typename T> struct VecT;
template <> struct VecT<float> { using type = float4; static constexpr int W = 4; };
template <> struct VecT<double> { using type = double2; static constexpr int W = 2; };
constexpr int JACOBI_ANGLE_THREADS = 64;

template <typename T> struct JacobiWs {
  T* P0; int pstride;    // 2 x (4 planes x h x ldh); buffer c at P0 + c * pstride
  T* Vt; int ldv;        // pe x ldv, ldv = pe rounded up to the 16-byte vector width
  T* cs0;                // 2 x h x 4  (sin, tau = sin/(1+cos), tan, -); buffer c at cs0 + c * 4 h
  int* plr0; int pe;     // 2 x pe   player at position; buffer c at plr0 + c * pe
};
__host__ __device__ inline int jacobi_ldv(int pe, size_t sz) { const int vw = (int)(16 / sz); return (pe + vw - 1) / vw * vw; }
template <typename T> __host__ __device__ inline size_t jacobi_ws_bytes(int pe) {
  const size_t h = pe >> 1, ldh = h | 1, ldv = jacobi_ldv(pe, sizeof(T));
  size_t b = (((2 * 4 * h * ldh) * sizeof(T)) + 15) & ~(size_t)15;
  b += (size_t)pe * ldv * sizeof(T) + 2 * h * 4 * sizeof(T);
  b = (b + 15) & ~(size_t)15;
  b += 2 * (size_t)pe * sizeof(int);
  return (b + 15) & ~(size_t)15;
}
template <typename T> __device__ __forceinline__ JacobiWs<T> jacobi_ws_carve(unsigned char* base, int pe) {
  const size_t h = pe >> 1, ldh = h | 1, ldv = jacobi_ldv(pe, sizeof(T));
  JacobiWs<T> w;
  w.P0 = reinterpret_cast<T*>(base); w.pstride = (int)(4 * h * ldh);
  size_t off = (((2 * 4 * h * ldh) * sizeof(T)) + 15) & ~(size_t)15;
  w.Vt = reinterpret_cast<T*>(base + off); w.ldv = (int)ldv; off += (size_t)pe * ldv * sizeof(T);
  w.cs0 = reinterpret_cast<T*>(base + off); off += 2 * h * 4 * sizeof(T);
  off = (off + 15) & ~(size_t)15;
  w.plr0 = reinterpret_cast<int*>(base + off); w.pe = pe;
  return w;
}

__host__ __device__ inline int seat_after(int pos, int h) {   // position after one round of the circle
  const int q = pos >> 1;
  if (!(pos & 1)) return q == 0 ? 0 : (q < h - 1 ? pos + 2 : 2 * (h - 1) + 1);
  return q == 0 ? (h > 1 ? 2 : 1) : pos - 2;
}
__device__ __forceinline__ int seat_before(int pos, int h) {  // inverse of seat_after
  const int q = pos >> 1;
  if (h == 1) return pos;
  if (!(pos & 1)) return q == 0 ? 0 : (q == 1 ? 1 : pos - 2);          // top 1 <- bottom 0, top q <- top q-1
  return q == h - 1 ? 2 * (h - 1) : pos + 2;                            // bottom h-1 <- top h-1, bottom q <- bottom q+1
}
__device__ __forceinline__ int seat_offset(int rowpos, int colpos, int psz, int ldh) {   // plane offset of entry (rowpos, colpos)
  return ((rowpos & 1) * 2 + (colpos & 1)) * psz + (rowpos >> 1) * ldh + (colpos >> 1);
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
template <typename T> __device__ __forceinline__ void rot2(T s, T tau, T& x, T& y) {
  const T nx = x - s * (y + tau * x), ny = y + s * (x - tau * y);
  x = nx; y = ny;
}
__device__ __forceinline__ void rot_vec(float s, float tau, float4& x, float4& y) {
  rot2(s, tau, x.x, y.x); rot2(s, tau, x.y, y.y); rot2(s, tau, x.z, y.z); rot2(s, tau, x.w, y.w);
}
__device__ __forceinline__ void rot_vec(double s, double tau, double2& x, double2& y) {
  rot2(s, tau, x.x, y.x); rot2(s, tau, x.y, y.y);
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
    P0[seat_offset(a, b, psz, ldh)] = val;
  }
}

// Work threads needed so that every thread owns at most `maxi` blocks / eigenvector slices (host side).
inline int jacobi_need(int pe, size_t sz) {
  const int h = pe >> 1, nblk = h * (h + 1) / 2, nvit = h * (jacobi_ldv(pe, sz) / (int)(16 / sz));
  return nblk > nvit ? nblk : nvit;
}

// On entry buffer 0 holds the matrix. On exit: *cur_out = buffer holding the (numerically diagonal) matrix,
// plr0[*cur_out * pe + pos] = player whose eigenvalue sits on the diagonal at pos, Vt[player][:] = its eigenvector.
// blockDim.x = work threads + JACOBI_ANGLE_THREADS; every thread of the CTA must call.
template <typename T, int MAXI>
__device__ int jacobi_planes(int pe, const JacobiWs<T>& w, double* shred, int max_sweeps, int* flag, int* cur_out,
                             bool keep_vt = false) {
  using V4 = typename VecT<T>::type;
  constexpr int VW = VecT<T>::W;
  const int tid = threadIdx.x, nt = blockDim.x, ntw = nt - JACOBI_ANGLE_THREADS;
  const int h = pe >> 1, ldh = h | 1, psz = h * ldh, ldv = w.ldv, nblk = h * (h + 1) / 2, nvc = ldv / VW, nvit = h * nvc;
  // ---- one-time set-up ----
  if (!keep_vt)   // warm start: Vt already holds an orthonormal basis in which the matrix was expressed
    for (int t = tid; t < pe * ldv; t += nt) { const int i = t / ldv, a = t - i * ldv; w.Vt[t] = (i == a) ? (T)1 : (T)0; }
  for (int pos = tid; pos < pe; pos += nt) w.plr0[pos] = pos;
  double acc[1] = {0.0};
  for (int t = tid; t < 4 * psz; t += nt) {
    const int r = t % ldh;
    if (r < h) { const double x = (double)w.P0[t]; acc[0] += x * x; }
  }
  block_sum<1>(acc, shred);
  const double normF2 = acc[0];
  *cur_out = 0;
  if (!(normF2 > 0.0)) { if (normF2 != normF2) *flag |= FLAG_NONFINITE; return 0; }
  const double tol2 = 256.0 * (double)Eps<T>::v() * (double)Eps<T>::v() * normF2;   // off-diagonal norm <= 16 eps ||S||_F
  const T skip = (T)(0.01 * sqrt(tol2) / pe);

  // per-thread constants (registers): blocks, eigenvector slices, or the pivot an angle thread prepares
  int bsrc[MAXI], bq[MAXI], bdst[MAXI][8];
  int vq[MAXI], va[MAXI];
#pragma unroll
  for (int i = 0; i < MAXI; ++i) { bq[i] = -1; vq[i] = -1; bsrc[i] = 0; va[i] = 0; }
  int qu = 0, qv = 0, su = 0, sv = 0;
  const bool worker = tid < ntw;
  if (worker) {
#pragma unroll
    for (int i = 0; i < MAXI; ++i) {
      const int t = tid + i * ntw;
      if (t < nblk) {
        int q1, q2;
        if (t < h) { q1 = q2 = t; }
        else {   // off-diagonal blocks, row after row: row q1 holds q2 = q1+1 .. h-1
          int e = t - h; q1 = 0;
          while (e >= h - 1 - q1) { e -= h - 1 - q1; ++q1; }
          q2 = q1 + 1 + e;
        }
        const int r_t = seat_after(2 * q1, h), r_b = seat_after(2 * q1 + 1, h), c_t = seat_after(2 * q2, h), c_b = seat_after(2 * q2 + 1, h);
        bq[i] = (q1 << 8) | q2; bsrc[i] = q1 * ldh + q2;
        bdst[i][0] = seat_offset(r_t, c_t, psz, ldh); bdst[i][1] = seat_offset(r_t, c_b, psz, ldh);
        bdst[i][2] = seat_offset(r_b, c_t, psz, ldh); bdst[i][3] = seat_offset(r_b, c_b, psz, ldh);
        bdst[i][4] = seat_offset(c_t, r_t, psz, ldh); bdst[i][5] = seat_offset(c_b, r_t, psz, ldh);   // mirror block
        bdst[i][6] = seat_offset(c_t, r_b, psz, ldh); bdst[i][7] = seat_offset(c_b, r_b, psz, ldh);
      }
      if (t < nvit) { vq[i] = t / nvc; va[i] = (t - vq[i] * nvc) * VW; }
    }
  } else {
    const int j = tid - ntw;
    if (j < h) { const int u = seat_before(2 * j, h), v = seat_before(2 * j + 1, h); qu = u >> 1; su = u & 1; qv = v >> 1; sv = v & 1; }
  }
  // rotations of the first round, straight from the diagonal blocks
  for (int q = tid; q < h; q += nt) {
    const int o = q * ldh + q;
    T sn, tau, tt;
    jacobi_angle<T>(w.P0[o], w.P0[3 * psz + o], w.P0[psz + o], skip, sn, tau, tt);
    w.cs0[4 * q] = sn; w.cs0[4 * q + 1] = tau; w.cs0[4 * q + 2] = tt; w.cs0[4 * q + 3] = (T)0;
  }
  __syncthreads();

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
      const T* __restrict__ Pc = w.P0 + cur * w.pstride;
      T* __restrict__ Pn = w.P0 + (cur ^ 1) * w.pstride;
      const T* __restrict__ csc = w.cs0 + cur * 4 * h;
      const int* __restrict__ plc = w.plr0 + cur * pe;
      if (worker) {
        // ---- eigenvector slices: load everything, then rotate and store (in place, slices are disjoint) ----
        V4 x[MAXI], y[MAXI]; T vs[MAXI], vt[MAXI]; V4 *pi[MAXI], *pj[MAXI];
#pragma unroll
        for (int i = 0; i < MAXI; ++i)
          if (vq[i] >= 0) {
            vs[i] = csc[4 * vq[i]]; vt[i] = csc[4 * vq[i] + 1];
            const int2 pl = *reinterpret_cast<const int2*>(plc + 2 * vq[i]);
            pi[i] = reinterpret_cast<V4*>(w.Vt + pl.x * ldv + va[i]); pj[i] = reinterpret_cast<V4*>(w.Vt + pl.y * ldv + va[i]);
            x[i] = *pi[i]; y[i] = *pj[i];
          }
        // ---- 2 x 2 blocks ----
#pragma unroll
        for (int i = 0; i < MAXI; ++i)
          if (bq[i] >= 0) {
            const int o = bsrc[i], q1 = bq[i] >> 8, q2 = bq[i] & 255;
            const T a = Pc[o], b = Pc[psz + o], d = Pc[3 * psz + o];
            if (q1 == q2) {
              const T g = csc[4 * q1 + 2] * b;   // tan * a_ij
              Pn[bdst[i][0]] = a - g; Pn[bdst[i][3]] = d + g; Pn[bdst[i][1]] = (T)0; Pn[bdst[i][2]] = (T)0;
            } else {
              const T c = Pc[2 * psz + o];
              const T s1 = csc[4 * q1], t1 = csc[4 * q1 + 1], s2 = csc[4 * q2], t2 = csc[4 * q2 + 1];
              const T ra = a - s1 * (c + t1 * a), rc = c + s1 * (a - t1 * c);   // rows:  J1' S
              const T rb = b - s1 * (d + t1 * b), rd = d + s1 * (b - t1 * d);
              const T na = ra - s2 * (rb + t2 * ra), nb = rb + s2 * (ra - t2 * rb);   // cols: (.) J2
              const T nc = rc - s2 * (rd + t2 * rc), nd = rd + s2 * (rc - t2 * rd);
              Pn[bdst[i][0]] = na; Pn[bdst[i][1]] = nb; Pn[bdst[i][2]] = nc; Pn[bdst[i][3]] = nd;
              Pn[bdst[i][4]] = na; Pn[bdst[i][5]] = nb; Pn[bdst[i][6]] = nc; Pn[bdst[i][7]] = nd;
            }
          }
#pragma unroll
        for (int i = 0; i < MAXI; ++i)
          if (vq[i] >= 0 && vs[i] != (T)0) { rot_vec(vs[i], vt[i], x[i], y[i]); *pi[i] = x[i]; *pj[i] = y[i]; }
        for (int pos = tid; pos < pe; pos += ntw) w.plr0[(cur ^ 1) * pe + seat_after(pos, h)] = plc[pos];
      } else {
        // ---- angle threads: pivot of next round's pair j = entries (u,u), (v,v), (u,v) AFTER this round's rotations ----
        const int j = tid - ntw;
        if (j < h) {
          const int ou = qu * ldh + qu, ov = qv * ldh + qv;
          const T su_ = csc[4 * qu], tu_ = csc[4 * qu + 1], gu_ = csc[4 * qu + 2];
          const T sv_ = csc[4 * qv], tv_ = csc[4 * qv + 1], gv_ = csc[4 * qv + 2];
          const T suu = su ? Pc[3 * psz + ou] + gu_ * Pc[psz + ou] : Pc[ou] - gu_ * Pc[psz + ou];
          const T svv = sv ? Pc[3 * psz + ov] + gv_ * Pc[psz + ov] : Pc[ov] - gv_ * Pc[psz + ov];
          T suv = (T)0;
          if (qu != qv) {
            const int o = qu * ldh + qv;
            const T a = Pc[o], b = Pc[psz + o], c = Pc[2 * psz + o], d = Pc[3 * psz + o];
            const T ra = a - su_ * (c + tu_ * a), rc = c + su_ * (a - tu_ * c);
            const T rb = b - su_ * (d + tu_ * b), rd = d + su_ * (b - tu_ * d);
            const T x0 = su ? rc : ra, x1 = su ? rd : rb;                            // row su of J1' S
            suv = sv ? x1 + sv_ * (x0 - tv_ * x1) : x0 - sv_ * (x1 + tv_ * x0);
          }
          T sn, tau, tt;
          jacobi_angle<T>(suu, svv, suv, skip, sn, tau, tt);
          T* csn = w.cs0 + (cur ^ 1) * 4 * h + 4 * j;
          csn[0] = sn; csn[1] = tau; csn[2] = tt;
        }
      }
      __syncthreads();
      cur ^= 1;
    }
  }
  if (sweep >= max_sweeps) *flag |= FLAG_EIG_CAP;
  *cur_out = cur;
  return sweep;
}

// C(i,j) = sum_k A(i,k) B(k,j), all pe x pe in shared memory with generic strides; 2x2 register tiles, consecutive
// threads along j. When B is read transposed (sbk == 1: the rows of B' are k-contiguous with an even stride) the
// threads of a warp would hit the same few banks at every k; they then walk k skewed by their tile column, which
// makes the B loads and the (no longer broadcast) A loads conflict free.
// fp32: the same product on the tensor cores (warp-level mma.sync m16n8k8, 3xTF32 split as in psd_bjacobi.cuh). One warp per
// 16 x 16 tile of C; out-of-range rows / columns / k read element 0 with weight 0. The tensor core adds into its accumulator
// with truncation, so the leading term is accumulated over 32 k at a time and the chunks are added round-to-nearest
// (gemm_tc.cuh has the measurement that made this necessary). ~2x the FMA version at pe = 100 (cfg4).
__device__ __forceinline__ void sg_split(float a, uint32_t& hi, uint32_t& lo) {
  hi = (__float_as_uint(a) + 0x1000u) & 0xffffe000u;
  lo = (__float_as_uint(a - __uint_as_float(hi)) + 0x1000u) & 0xffffe000u;
}
__device__ __forceinline__ void sg_mma(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void smem_gemm_tc(int pe, const float* A, int sai, int sak, const float* B, int sbk, int sbj, float* C,
                                             int ldc) {
  const int warp = threadIdx.x >> 5, nw = blockDim.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int nt = (pe + 15) >> 4;
  for (int tile = warp; tile < nt * nt; tile += nw) {
    const int i0 = (tile / nt) * 16, j0 = (tile % nt) * 16;
    float sum[2][4] = {}, accS[2][4] = {};
    for (int kc = 0; kc < pe; kc += 32) {
      float accM[2][4] = {};
#pragma unroll
      for (int kk = 0; kk < 32; kk += 8) {
        const int k0 = kc + kk;
        if (k0 >= pe) break;
        uint32_t ah[4], al[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {      // a0 (g, t), a1 (g + 8, t), a2 (g, t + 4), a3 (g + 8, t + 4)
          const int i = i0 + g + 8 * (e & 1), k = k0 + t + 4 * (e >> 1);
          const float v = (i < pe && k < pe) ? A[i * sai + k * sak] : 0.f;
          sg_split(v, ah[e], al[e]);
        }
#pragma unroll
        for (int n = 0; n < 2; ++n) {
          uint32_t bh[2], bl[2];
#pragma unroll
          for (int e = 0; e < 2; ++e) {    // b0 (k = t, n = g), b1 (k = t + 4, n = g)
            const int k = k0 + t + 4 * e, j = j0 + 8 * n + g;
            const float v = (k < pe && j < pe) ? B[k * sbk + j * sbj] : 0.f;
            sg_split(v, bh[e], bl[e]);
          }
          sg_mma(accS[n], al, bh[0], bh[1]);
          sg_mma(accS[n], ah, bl[0], bl[1]);
          sg_mma(accM[n], ah, bh[0], bh[1]);
        }
      }
#pragma unroll
      for (int n = 0; n < 2; ++n)
#pragma unroll
        for (int e = 0; e < 4; ++e) sum[n][e] += accM[n][e];
    }
#pragma unroll
    for (int n = 0; n < 2; ++n)
#pragma unroll
      for (int e = 0; e < 4; ++e) {        // c0 (g, 2t), c1 (g, 2t + 1), c2 (g + 8, 2t), c3 (g + 8, 2t + 1)
        const int i = i0 + g + 8 * (e >> 1), j = j0 + 8 * n + 2 * t + (e & 1);
        if (i < pe && j < pe) C[i * ldc + j] = sum[n][e] + accS[n][e];
      }
  }
}

template <typename T>
__device__ __forceinline__ void smem_gemm(int pe, const T* A, int sai, int sak, const T* B, int sbk, int sbj, T* C,
                                          int ldc) {
  if constexpr (sizeof(T) == 4) { smem_gemm_tc(pe, A, sai, sak, B, sbk, sbj, C, ldc); return; }
  const int h = pe >> 1;
  const bool skewed = (sbk == 1 && sbj != 1 && sak == 1);
  for (int t = threadIdx.x; t < h * h; t += blockDim.x) {
    const int jt = t % h;
    const int i = (t / h) * 2, j = jt * 2;
    T c00 = 0, c01 = 0, c10 = 0, c11 = 0;
    const T *a0 = A + i * sai, *a1 = a0 + sai, *b0 = B + j * sbj, *b1 = b0 + sbj;
    if (skewed) {
      int k = jt;                       // pe = 2 h > jt
#pragma unroll 4
      for (int s = 0; s < pe; ++s) {
        const T x0 = a0[k], x1 = a1[k], y0 = b0[k], y1 = b1[k];
        c00 += x0 * y0; c01 += x0 * y1; c10 += x1 * y0; c11 += x1 * y1;
        if (++k == pe) k = 0;
      }
    } else {
#pragma unroll 4
      for (int k = 0; k < pe; ++k) {
        const T x0 = a0[k * sak], x1 = a1[k * sak], y0 = b0[k * sbk], y1 = b1[k * sbk];
        c00 += x0 * y0; c01 += x0 * y1; c10 += x1 * y0; c11 += x1 * y1;
      }
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

// CTA size cap per MAXI (more register-resident items per thread -> fewer threads, more registers each)
__host__ __device__ constexpr int psd_small_max_threads(int maxi) { return maxi <= 1 ? 1024 : (maxi == 2 ? 768 : (maxi == 3 ? 640 : 608)); }

struct PsdFwdArgs {
  const double* W;   // projection argument, all rows
  double* S1;        // s^{k+1} base (rows)
  double* Y1;        // y^{k+1} base (rows)
  void* Ustore;      // eigenvector store of this iteration (or scratch)
  void* Lstore;
  const void* Uprev; // eigenvectors of the previous iterate (same layout as Ustore) or NULL: warm start
  int* sweeps_max; int* flags;
  unsigned long long* sweeps_sum;   // total Jacobi sweeps over blocks (statistics for the ALU roofline)
};

template <typename T, int MAXI>
__global__ void __launch_bounds__(psd_small_max_threads(MAXI)) k_psd_fwd_small(PsdTab tab, Hyper<T> H, int k, PsdFwdArgs A, const int* list) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int blk = list[blockIdx.x];
  const int p = tab.p[blk], pe = (p + 1) & ~1;
  const int prob = tab.prob[blk];
  const long long row0 = tab.row0[blk];
  double* shred = reinterpret_cast<double*>(smem_raw);                 // 64 doubles
  const JacobiWs<T> ws = jacobi_ws_carve<T>(smem_raw + 512, pe);
  T* lp = reinterpret_cast<T*>(smem_raw + 512 + jacobi_ws_bytes<T>(pe));   // pe: max(lambda, 0) by player
  const double rho = H.rho_blk(k, prob, row0);
  const double* w = A.W + row0;
  const int ldv = ws.ldv;
  const int h = pe >> 1, ldh = h | 1, psz = h * ldh;
  const bool warmst = A.Uprev != nullptr;
  if (warmst) {
    // Warm start: consecutive ADMM iterates have nearby eigenbases, so S is first expressed in the previous
    // iterate's basis, A' = U' S U (two shared-memory products), which leaves it almost diagonal; the sweeps then
    // rotate that basis (Vt keeps U instead of the identity) and 2-3 of them suffice instead of 6-8.
    const T* Up = reinterpret_cast<const T*>(A.Uprev) + tab.uoff[blk];
    T* Tm = ws.P0;                    // buffer 0: S U
    T* Sd = ws.P0 + ws.pstride;       // buffer 1: S, then A'
    for (int t = threadIdx.x; t < pe * ldv; t += blockDim.x) {
      const int i = t / ldv, a = t - i * ldv;
      ws.Vt[t] = (i < p && a < p) ? Up[i * p + a] : ((i == a) ? (T)1 : (T)0);
    }
    __syncthreads();
    // One Newton-Schulz step U <- (3/2) U - (1/2) U (U'U) first: the basis is a product of hundreds of fp32 rotations
    // per iterate and is carried from iterate to iterate, so its orthogonality error would grow with k (measured on
    // cfg2: iterate error 8.6e-5 after 50 steps without this step, 1e-5 with it); the step squares that error.
    smem_gemm<T>(pe, ws.Vt, ldv, 1, ws.Vt, 1, ldv, Tm, pe);    // Tm(i,j) = <u_i, u_j>
    __syncthreads();
    smem_gemm<T>(pe, Tm, pe, 1, ws.Vt, ldv, 1, Sd, pe);        // Sd(i,a) = sum_j Tm(i,j) U(a,j)
    __syncthreads();
    for (int t = threadIdx.x; t < pe * pe; t += blockDim.x) {
      const int i = t / pe, a = t - i * pe;
      ws.Vt[i * ldv + a] = (T)1.5 * ws.Vt[i * ldv + a] - (T)0.5 * Sd[i * pe + a];
    }
    __syncthreads();
    load_smat<T>(p, pe, pe, Sd, w, 0.0, nullptr);
    __syncthreads();
    smem_gemm<T>(pe, Sd, pe, 1, ws.Vt, 1, ldv, Tm, pe);        // Tm(a,i) = sum_b S(a,b) U(b,i)
    __syncthreads();
    smem_gemm<T>(pe, ws.Vt, ldv, 1, Tm, pe, 1, Sd, pe);        // A'(i,j) = sum_a U(a,i) Tm(a,j)
    __syncthreads();
    for (int t = threadIdx.x; t < pe * pe; t += blockDim.x) {
      const int b = t / pe, a = t - b * pe;
      ws.P0[seat_offset(a, b, psz, ldh)] = (T)0.5 * (Sd[a * pe + b] + Sd[b * pe + a]);
    }
  } else {
    load_smat_planes<T>(p, pe, ws.P0, w, 0.0, nullptr);
  }
  __syncthreads();
  int flag = 0, cur = 0;
  const int sweeps = jacobi_planes<T, MAXI>(pe, ws, shred, 40, &flag, &cur, warmst);
  T* U = reinterpret_cast<T*>(A.Ustore) + tab.uoff[blk];   // rows = eigenvectors
  T* L = reinterpret_cast<T*>(A.Lstore) + tab.loff[blk];
  for (int pos = threadIdx.x; pos < pe; pos += blockDim.x) {
    const int q = pos >> 1, pl = ws.plr0[cur * pe + pos];
    const T l = ws.P0[cur * ws.pstride + ((pos & 1) ? 3 * psz : 0) + q * ldh + q];
    lp[pl] = l > (T)0 ? l : (T)0;
    if (pl < p) L[pl] = l;
  }
  for (int t = threadIdx.x; t < p * p; t += blockDim.x) { const int i = t / p, a = t - i * p; U[t] = ws.Vt[i * ldv + a]; }
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
      if (l > (T)0) acc += va[i * ldv] * l * vb[i * ldv];
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

template <typename T, int MAXI>
__global__ void __launch_bounds__(psd_small_max_threads(MAXI)) k_psd_bwd_small(PsdTab tab, Hyper<T> H, int k, PsdBwdArgs A, const int* list) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int blk = list[blockIdx.x];
  const int p = tab.p[blk], pe = (p + 1) & ~1, ld = pe;
  const int prob = tab.prob[blk];
  const long long row0 = tab.row0[blk];
  double* shred = reinterpret_cast<double*>(smem_raw);                 // 64 doubles
  const JacobiWs<T> ws = jacobi_ws_carve<T>(smem_raw + 512, pe);
  T* lam = reinterpret_cast<T*>(smem_raw + 512 + jacobi_ws_bytes<T>(pe));
  T* Vt = ws.Vt;            // Vt[i*ldv + a] = V(a, i)
  const int ldv = ws.ldv;
  T* G = ws.P0;             // the two p x p work matrices alias the Jacobi planes (dead after a recompute)
  T* Tm = G + pe * pe;
  const double rho = H.rho_blk(k, prob, row0);
  const double* w = A.W + row0;
  int flag = 0;
  if (A.recompute) {
    load_smat_planes<T>(p, pe, ws.P0, w, 0.0, nullptr);
    __syncthreads();
    int cur = 0;
    jacobi_planes<T, MAXI>(pe, ws, shred, 40, &flag, &cur);
    const int h = pe >> 1, ldh = h | 1, psz = h * ldh;
    for (int pos = threadIdx.x; pos < pe; pos += blockDim.x)
      lam[ws.plr0[cur * pe + pos]] = ws.P0[cur * ws.pstride + ((pos & 1) ? 3 * psz : 0) + (pos >> 1) * ldh + (pos >> 1)];
    __syncthreads();
  } else {
    const T* U = reinterpret_cast<const T*>(A.Ustore) + tab.uoff[blk];
    const T* L = reinterpret_cast<const T*>(A.Lstore) + tab.loff[blk];
    for (int t = threadIdx.x; t < pe * pe; t += blockDim.x) {
      const int i = t / pe, a = t - i * pe;
      Vt[i * ldv + a] = (a < p && i < p) ? U[i * p + a] : ((a == i) ? (T)1 : (T)0);
    }
    for (int i = threadIdx.x; i < pe; i += blockDim.x) lam[i] = i < p ? L[i] : (T)0;
    __syncthreads();
  }
  const double* gs = A.Gs + row0;
  const double* gy = A.Gy + row0;
  load_smat<T>(p, pe, ld, G, gs, rho, gy);                 // G = smat(g_s+ + rho g_y+)
  __syncthreads();
  smem_gemm<T>(pe, G, ld, 1, Vt, 1, ldv, Tm, ld);           // Tm = G V
  __syncthreads();
  smem_gemm<T>(pe, Vt, ldv, 1, Tm, ld, 1, G, ld);           // C  = V' Tm
  __syncthreads();
  for (int t = threadIdx.x; t < pe * pe; t += blockDim.x) {
    const int i = t / pe, j = t - i * pe;
    G[i * ld + j] *= gamma_relu<T>(lam[i], lam[j]);
  }
  __syncthreads();
  smem_gemm<T>(pe, Vt, 1, ldv, G, ld, 1, Tm, ld);           // Tm = V C
  __syncthreads();
  smem_gemm<T>(pe, Tm, ld, 1, Vt, ldv, 1, G, ld);           // out = Tm V'
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

// Launch shape of the small-block kernels for blocks up to order pmax: every work thread owns at most `maxi`
// 2x2 blocks and eigenvector slices (register resident), plus the angle warps. maxi <= PSD_SMALL_MAXI.
constexpr int PSD_SMALL_MAXI = 4;
struct PsdSmallCfg { int maxi, threads; };
static inline PsdSmallCfg psd_small_cfg(int pmax, size_t sz) {
  const int pe = (pmax + 1) & ~1, need = jacobi_need(pe, sz);
  int maxi = 1;
  while (maxi <= PSD_SMALL_MAXI && need > maxi * (psd_small_max_threads(maxi) - JACOBI_ANGLE_THREADS)) ++maxi;
  int ntw = (((need + maxi - 1) / maxi) + 31) & ~31;
  if (ntw < 32) ntw = 32;
  return PsdSmallCfg{maxi, ntw + JACOBI_ANGLE_THREADS};
}

}  // namespace cdu

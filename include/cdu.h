/* cdu.h - C ABI of the conic deep-unfolding hot path (batched, unrolled COSMO ADMM, forward + backward)
 *
 * Problem statement (Eq. 1):   min 1/2 x'Px + q'x   s.t.  Ax + s = b,  s in K,
 * K a Cartesian product of zero / nonnegative / second-order / PSD cones.
 *
 * One iteration (Eq. 3a-3e L60-72 in the indirect form Eq. 4; sign convention "y in K*",
 * DESIGN.md reading A1, so that r_p = Ax+s-b and r_d = Px+q+A'y as printed in Eq. 12):
 *     xi = sigma x - q + A'(rho (b - s) - y)
 *     xt = M^-1 xi,  M = P + sigma I + rho A'A      (matrix-free Jacobi-preconditioned CG, L80, L294)
 *     st = b - A xt
 *     x+ = alpha xt + (1-alpha) x ;  w = alpha st + (1-alpha) s - y/rho
 *     s+ = Pi_K(w)                                   (PSD blocks: eigendecomposition, clamp, rebuild, Eq. 7)
 *     y+ = rho (s+ - w)
 * Backward: BPTT over the stored iterates; adjoint CG on the same M and grad_rho = (A lam) o (A xt)
 * (Eq. 5-6); Dalecki-Krein VJP for the PSD projection (Eq. 9-10).
 *
 * Conventions
 *   - svec: upper triangle, column by column, off-diagonals scaled by sqrt(2).
 *   - SOC_d = {(t,u): ||u||_2 <= t}, t first.
 *   - All floating-point arrays crossing this ABI have the handle's dtype (float for CDU_F32, double for
 *     CDU_F64). Internally the iterate and all reductions are fp64; CG, eig and DK run in the handle's dtype.
 *   - No function throws or aborts; every error is a return code, cdu_last_error() gives the text.
 *   - Thread safety: one handle may be used from one host thread at a time.
 */
#ifndef CDU_H_
#define CDU_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cdu_handle_s* cdu_handle; /* opaque; owns device copies of the problem, scratch and the checkpoint store */

typedef enum { CDU_OK = 0, CDU_EINVAL = 1, CDU_ENOMEM = 2, CDU_ECUDA = 3, CDU_ESTATE = 4, CDU_ENUMERIC = 5 } cdu_status;
typedef enum { CDU_F32 = 0, CDU_F64 = 1 } cdu_dtype;
typedef enum { CDU_ZERO = 0, CDU_NONNEG = 1, CDU_SOC = 2, CDU_PSD = 3 } cdu_cone_kind;
typedef enum { CDU_RHO_PER_ITER = 0,    /* rho[K], alpha[K] shared by the batch; g_rho[K], g_alpha[K], g_sigma[1] are batch sums */
               CDU_RHO_PER_PROBLEM = 1, /* rho[K][B], alpha[K][B]; g_rho[K][B], g_alpha[K][B], g_sigma[B] */
               CDU_RHO_PER_ROW = 2      /* rho[K][sum m_b] (D = diag(rho) in M = P + sigma I + A'DA, L78; Eq. 6 L90 row by row),
                                           alpha[K][B]; g_rho[K][sum m_b], g_alpha[K][B], g_sigma[B]. rho must be constant
                                           inside every SOC / PSD block (the projection of Eq. 3d couples their rows, L343):
                                           cdu_rectify_rho averages a per-row prediction over each block */
} cdu_rho_mode;
typedef enum { CDU_CKPT_FULL = 0, /* store z^k plus x-tilde, s-tilde and (U, lambda) of every PSD block            */
               CDU_CKPT_LEAN = 1  /* store z^k only ((n+2m) doubles per iteration); backward re-solves and re-factors */
} cdu_ckpt_mode;

/* dim = number of rows for ZERO / NONNEG / SOC (SOC: t first); for PSD the matrix order p, rows = p(p+1)/2 */
typedef struct { int32_t kind; int32_t dim; } cdu_cone;

/* A batch of `batch` independent instances, block-diagonal batched CSR (the paper's "super-batch", L306).
 * All arrays below are HOST memory and are copied by cdu_create; the caller may free them on return. */
typedef struct {
  int32_t batch;
  int32_t dtype;            /* cdu_dtype of A_val, P_val, q, b and of every array passed to forward/backward */
  const int64_t* var_off;   /* [batch+1] offsets of x:  n_b = var_off[b+1]-var_off[b]                       */
  const int64_t* row_off;   /* [batch+1] offsets of the constraint rows: m_b                                */
  const int64_t* A_rowptr;  /* [sum m_b + 1] global nnz offsets                                              */
  const int32_t* A_colidx;  /* [nnz A] column index LOCAL to the problem, 0..n_b-1, sorted within a row      */
  const void*    A_val;     /* [nnz A]                                                                       */
  const int64_t* P_rowptr;  /* [sum n_b + 1]; P in FULL symmetric storage (both triangles); may hold 0 nnz   */
  const int32_t* P_colidx;
  const void*    P_val;
  const void*    q;         /* [sum n_b] */
  const void*    b;         /* [sum m_b] */
  const int64_t* cone_off;  /* [batch+1] into cones[]; the cones of a problem tile its rows in order         */
  const cdu_cone* cones;
} cdu_problem;

typedef struct {
  double  cg_tol;           /* stop when ||xi - M xt||_2 <= cg_tol ||xi||_2; <= 0: 1e-10 (F64) / 1e-6 (F32)     */
  int32_t cg_max_iter;      /* <= 0: 2 n + 50                                                                   */
  int32_t K_max;            /* capacity of the checkpoint store (largest K a forward call may use)              */
  int32_t ckpt_mode;        /* cdu_ckpt_mode                                                                    */
  int32_t cg_refine;        /* extra passes of fp64-residual iterative refinement around the CG solve;
                               < 0: default (1 for F32, 0 for F64)                                              */
  double  cg_refine_tol;    /* each refinement pass reduces the true residual by this factor; <= 0: 1e-4        */
  int32_t psd_small_max;    /* PSD blocks of order <= this run in the shared-memory Jacobi kernel, larger ones in
                               the global-memory path; <= 0: default (128 for F32, 88 for F64)                  */
  int32_t use_tensor_cores; /* large-block products on tcgen05 (3xTF32, fp32 handles, block order a multiple of 128):
                               bit 0 = rebuild U max(L,0) U', bit 1 = the four Dalecki-Krein products; 0 = fp32 FMA
                               GEMM for both; < 0: default (3)                                                  */
  int32_t team_size;        /* CTAs (thread-block cluster size, power of two <= 16) that share one problem in the
                               linear-step kernels; <= 0: chosen from the batch size and the problem size         */
  int32_t no_batch;         /* 1: single-CTA teams read rows with lane groups straight from global memory instead of
                               the precomputed warp batches (debug / comparison)                                  */
  int32_t no_diag_path;     /* 1: run the PCG kernels even when M = P + sigma I + rho A'A is diagonal (every row of A
                               holds <= 1 entry, P diagonal, no SOC cones), where by default the single PCG iteration
                               is evaluated in closed form (debug / comparison)                                    */
} cdu_options;

/* Copies and re-packs the batch onto the current CUDA device (transposed copy of A, diag(P), column square
 * sums for the Jacobi preconditioner, cone tables) and allocates scratch and the checkpoint store.
 * `opts` may be NULL (defaults, K_max = 0 is invalid). Returns CDU_EINVAL on malformed input (cones not tiling
 * the rows, indices out of range, non-symmetric pattern is NOT checked), CDU_ENOMEM / CDU_ECUDA otherwise. */
cdu_status cdu_create(const cdu_problem* prob, const cdu_options* opts, void* cuda_stream, cdu_handle* out);

/* K unrolled iterations from (x0, s0, y0) (NULL = zeros). rho, alpha: hyper-parameters, layout per rho_mode.
 * xK, sK, yK (each may be NULL) receive z^K. If io_on_host == 0 all pointers are DEVICE pointers, borrowed for the
 * stream-ordered work, and the call returns without synchronising. If io_on_host != 0 they are HOST pointers
 * (pinned memory recommended); the library stages them through its own device buffers and returns after the
 * results have landed (stream synchronised).
 * Errors: CDU_EINVAL (K < 1, K > K_max, sigma <= 0, NULL rho/alpha; host-side rho <= 0 or alpha outside (0,2)).
 * Device-resident rho / alpha cannot be read without a host sync: they are checked by a kernel that raises flag 16 on
 * the problems they apply to; cdu_get_stats then returns CDU_ENUMERIC. */
cdu_status cdu_forward(cdu_handle h, int32_t K, const void* rho, int32_t rho_mode, double sigma, const void* alpha,
                       const void* x0, const void* s0, const void* y0,
                       void* xK, void* sK, void* yK, int32_t io_on_host, void* cuda_stream);

/* Reverse sweep of the last cdu_forward on this handle (CDU_ESTATE if there was none); may be called repeatedly
 * with different cotangents. g_xK, g_sK, g_yK: dL/d(x_K, s_K, y_K) (NULL = zeros). Outputs (each may be NULL):
 * g_rho, g_alpha (layout of the forward's rho_mode), g_sigma ([1] or [B]), g_x0, g_s0, g_y0. */
cdu_status cdu_backward(cdu_handle h, const void* g_xK, const void* g_sK, const void* g_yK,
                        void* g_rho, void* g_sigma, void* g_alpha, void* g_x0, void* g_s0, void* g_y0,
                        int32_t io_on_host, void* cuda_stream);

/* cdu_backward with a cotangent on every intermediate iterate, for losses that read all iterates (Eq. 12,
 * L146-148): inj_x [K-1][sum n_b], inj_s, inj_y [K-1][sum m_b] (row k-1 = dL/dz^k of the part of the loss that reads z^k,
 * k = 1..K-1; any of the three may be NULL). Same outputs as cdu_backward. */
cdu_status cdu_backward_inject(cdu_handle h, const void* g_xK, const void* g_sK, const void* g_yK,
                               const void* inj_x, const void* inj_s, const void* inj_y,
                               void* g_rho, void* g_sigma, void* g_alpha, void* g_x0, void* g_s0, void* g_y0,
                               int32_t io_on_host, void* cuda_stream);

/* The self-supervised training loss of PAPER.md Eq. 12 (L146) on the iterates of the last cdu_forward,
 *   L_b = sum_{k=1..K} log( ||P x^k + q + A'y^k||^2 / det(||r_d^0||^2) + ||A x^k + s^k - b||^2 / det(||r_p^0||^2) )
 * (det = stop-gradient: the residuals of z^0 enter as constants; a term whose denominator is 0 is dropped), and its reverse
 * sweep: the cotangent of every z^k is formed from the stored iterate when the sweep reaches k, so memory stays O(n + nnz)
 * per unrolled iteration (L92). loss: [batch] (NULL: not wanted); gradient outputs as cdu_backward (sums over the batch in
 * CDU_RHO_PER_ITER mode are gradients of sum_b L_b). */
cdu_status cdu_backward_eq12(cdu_handle h, void* loss, void* g_rho, void* g_sigma, void* g_alpha,
                             void* g_x0, void* g_s0, void* g_y0, int32_t io_on_host, void* cuda_stream);

/* Policy features of PAPER.md App. E (L321-339) for iterate k (0 <= k <= K of the last forward), each output may be NULL:
 *   rp_bar [sum m_b] = (A x^k + s^k - b) / max(|A x^k|_inf, |s^k|_inf, |b|_inf)      (per problem, OSQP-style scaling)
 *   rd_bar [sum n_b] = (P x^k + q + A'y^k) / max(|P x^k|_inf, |q|_inf, |A'y^k|_inf)
 *   delta_p [sum m_b] = s^k - s-tilde^k (k >= 1, FULL checkpoints only: CDU_ESTATE otherwise), delta_d = s^k - s^(k-1) (k >= 1)
 *   scal [batch][3]   = log(|rp_bar|_inf + 1e-12), log(|rd_bar|_inf + 1e-12), log(|delta_p|_inf + 1e-12) */
cdu_status cdu_get_features(cdu_handle h, int32_t k, void* rp_bar, void* rd_bar, void* delta_p, void* delta_d, void* scal,
                            int32_t io_on_host, void* cuda_stream);

/* Rectification of PAPER.md App. E (L343), in place on rho [K][sum m_b] (or on a g_rho of that layout: the operation is its
 * own adjoint): every SOC / PSD block gets the mean of its rows; zero / nonneg rows are left as they are. */
cdu_status cdu_rectify_rho(cdu_handle h, int32_t K, void* rho, int32_t io_on_host, void* cuda_stream);

/* Vanilla COSMO run to tolerance (the baseline workload of PAPER.md Table 1): iterates in chunks of `check_every`
 * (<= K_max) steps through the kernels of cdu_forward with a fixed alpha and one base penalty rho_b per problem, starting at
 * rho0; the equality (ZERO cone) rows run on eq_scale rho_b (COSMO / OSQP use 1e3, L306; eq_scale <= 0 or 1: every row on
 * rho_b). After every chunk the OSQP-scaled residuals of App. E (L323) are read back - the only host synchronisation - and a
 * problem is converged when |rp_bar|_inf <= eps and |rd_bar|_inf <= eps. adapt_rho != 0: residual balancing (L349), rho_b <-
 * rho_b sqrt(|rp_bar|_inf / |rd_bar|_inf) clipped to [1e-6, 1e6] when the two differ by more than 5x. x0, s0, y0 (NULL = zeros)
 * and x, s, y (may be NULL) as in cdu_forward; iters_out [batch] (HOST): iterations at the first check that found the problem
 * converged, or -(iterations done) if it did not converge within max_iter; res_out [batch][2] (HOST): the last scaled
 * residuals. */
cdu_status cdu_solve(cdu_handle h, int32_t max_iter, int32_t check_every, double eps, double rho0, double alpha, double sigma,
                     int32_t adapt_rho, double eq_scale, const void* x0, const void* s0, const void* y0, void* x, void* s, void* y,
                     int32_t* iters_out, double* res_out, int32_t io_on_host, void* cuda_stream);

typedef struct {
  int64_t cg_iters_fwd;      /* CG iterations summed over problems and iterations, last forward            */
  int64_t cg_iters_bwd;      /* same for the adjoint solves (and LEAN re-solves) of the last backward       */
  int32_t cg_iters_max;      /* largest single-solve count                                                  */
  int32_t eig_sweeps_max;    /* largest Jacobi sweep count of a PSD block                                   */
  int32_t n_flagged;         /* problems with a flag set (CG cap hit, non-positive curvature, sweep cap, NaN) */
  int32_t flags_or;          /* OR of all per-problem flag words: 1 CG cap, 2 pAp<=0, 4 eig sweep cap, 8 non-finite,
                                16 rho <= 0 or alpha outside (0,2) (device-side check of device-resident hyper-parameters) */
  int64_t device_bytes;      /* bytes of device memory owned by the handle                                  */
  int64_t ckpt_bytes;        /* of which checkpoint store                                                   */
  int64_t launches;          /* kernel launches issued by the handle since creation                         */
  int64_t eig_sweeps_sum;    /* Jacobi sweeps summed over PSD blocks and iterations of the last forward     */
  int64_t cg_iters_fwd_pass0; /* of cg_iters_fwd: iterations of the first pass (to cg_tol), i.e. without refinement */
  int64_t cg_iters_bwd_pass0; /* same for cg_iters_bwd                                                       */
} cdu_stats;

/* Synchronises the stream of the last call and reads back the per-problem counters. `out` is always filled; the return
 * value is CDU_ENUMERIC when any per-problem flag is set (CG cap, non-positive curvature, eigen-sweep cap, non-finite
 * value, rho <= 0 or alpha outside (0,2) detected on the device), CDU_OK otherwise. */
cdu_status cdu_get_stats(cdu_handle h, cdu_stats* out);

/* Copies iterate z^k (0 <= k <= K of the last forward) into caller buffers (device or host per io_on_host). */
cdu_status cdu_get_iterate(cdu_handle h, int32_t k, void* x, void* s, void* y, int32_t io_on_host, void* cuda_stream);

const char* cdu_last_error(cdu_handle h); /* valid until the next call on h; h may be NULL (create errors) */
cdu_status  cdu_destroy(cdu_handle h);
const char* cdu_version(void);

/* ---- per-kernel-class timing (CUDA events on the launching stream; used by bench.py's roofline leg) ---------
 * Classes: 0 linear step forward (xi, PCG, relaxation, zero/nonneg/SOC), 1 PSD forward small (shared-memory
 * Jacobi + rebuild), 2 large-block eigendecomposition, 3 large-block GEMMs (rebuild / DK), 4 linear step
 * backward (adjoint PCG, Eq. 6), 5 PSD backward small (DK), 6 large-block glue, 7 other. cdu_get_profile
 * synchronises on the recorded events, returns summed milliseconds and launch counts since the last call. */
#define CDU_PROFILE_CLASSES 8
cdu_status cdu_profile(cdu_handle h, int32_t enable);
cdu_status cdu_get_profile(cdu_handle h, int32_t nclass, double* ms, int64_t* count);

/* ---- stand-alone operator entry points (unit tests, micro-benchmarks, ncu isolation) ------------------------
 * Batched PSD projection S -> Pi(S) = U max(L,0) U' (Eq. 7) and its Dalecki-Krein VJP (Eq. 9-10) on `count`
 * dense symmetric p x p matrices (row-major, device pointers, dtype as given). `path`: 0 auto, 1 shared-memory
 * Jacobi, 2 global-memory path. U (row-major, eigenvectors in columns) and lam may be NULL for the projection;
 * the VJP reads them. */
cdu_status cdu_psd_project(int32_t dtype, int32_t count, int32_t p, const void* S, void* PiS, void* U, void* lam,
                           int32_t path, int32_t use_tensor_cores, void* cuda_stream);
cdu_status cdu_psd_vjp(int32_t dtype, int32_t count, int32_t p, const void* U, const void* lam, const void* Gbar,
                       void* Sbar, int32_t path, int32_t use_tensor_cores, void* cuda_stream);

/* ---- the PSD projection for callers that may not allocate ------------------------------------------------------
 * cdu_psd_project (above) keeps its block tables and work arrays in cudaMalloc'ed memory. Code under CUDA graph
 * capture, tight serving loops and harnesses that forbid cudaMalloc get this variant instead: the same operation
 * (Eq. 7, S -> Pi(S) = U max(L,0) U') through the same shared-memory Jacobi code as path 1 above (same arithmetic,
 * same launch shape), with ALL scratch in one file-scope __device__ array of CDU_PSD_STATIC_BYTES that every GPU
 * which loads the library holds until the process exits. It calls no cudaMalloc / cudaFree / allocating library routine
 * and does not synchronise: on `cuda_stream` it enqueues four kernels, a fifth if U != NULL, and one device-to-device
 * copy if lam != NULL.
 *   S, PiS [count][p][p] row-major device pointers (PiS may alias S); U ([count][p][p], eigenvectors in columns)
 *   and lam ([count][p]) may be NULL; dtype CDU_F32 or CDU_F64 (of S, PiS, U, lam and of the Jacobi arithmetic).
 * Limits: 1 <= p <= CDU_PSD_STATIC_MAX_P and the scratch of (count, p) - about count * (8 p (p+1) + (p*p + p) *
 * sizeof(dtype) + 4) bytes, each part rounded up to 256 - must fit the array: e.g. 120 matrices of order 64 or
 * 480 of order 32 in fp64. Anything larger returns CDU_EINVAL with the required size in cdu_last_error(NULL);
 * nothing is launched then. No per-matrix convergence flag is returned (cdu_psd_project does not return one either).
 * The array is shared by every call on a device and keeps the previous call's contents; the call clears what must
 * start at zero itself. Calls that overlap on the GPU (two streams, two threads) race on it: serialise them. */
#define CDU_PSD_STATIC_BYTES (8u << 20)
#define CDU_PSD_STATIC_MAX_P 64
cdu_status cdu_psd_project_static(int32_t dtype, int32_t count, int32_t p, const void* S, void* PiS, void* U, void* lam,
                                  void* cuda_stream);

/* ---- roofline denominators measured in-tree (bench.py) ---------------------------------------
 * Runs a micro-benchmark on the current device and stream and returns its best-of-5 rate in *value:
 *   CDU_PEAK_FP32_FMA / CDU_PEAK_FP64_FMA : dependent-chain-free FMA loops on the plain ALUs, TFLOP/s;
 *   CDU_PEAK_TF32_TENSOR : back-to-back tcgen05.mma kind::tf32 (M128 N256 K8) from shared-memory operands, dense
 *                          TFLOP/s of the tensor pipe (1 x TF32; the 3xTF32 products execute three of these per flop);
 *   CDU_PEAK_HBM_COPY    : device-to-device copy of 1 GiB, GB/s (read + write);
 *   CDU_PEAK_TF32_MMA_SYNC : back-to-back warp-level mma.sync m16n8k8 tf32 (the blocked Jacobi's Gram / apply path), TFLOP/s. */
typedef enum { CDU_PEAK_FP32_FMA = 0, CDU_PEAK_FP64_FMA = 1, CDU_PEAK_TF32_TENSOR = 2, CDU_PEAK_HBM_COPY = 3,
               CDU_PEAK_TF32_MMA_SYNC = 4 } cdu_peak_kind;
cdu_status cdu_measure_peak(int32_t kind, double* value, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* CDU_H_ */

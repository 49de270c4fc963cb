// psd_static.cu - cdu_psd_project_static: the stand-alone batched PSD projection (Eq. 7) for callers that may
// not allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).
//
// cdu_psd_project (handle.cuh, psd_op_t) runs k_dense_to_svec -> k_psd_fwd_small -> k_svec_to_dense with its block tables,
// the svec forms of the argument and of the result, the eigenvector rows, the eigenvalues, the flags and the sweep counters
// in a DevPool (cudaMalloc). The variant here is the cold-start branch of k_psd_fwd_small as a kernel of its own,
// k_psd_project_static: same device functions (load_smat_planes, jacobi_planes, the rebuild loop), same launch shape, same
// arithmetic; the tables are gone (block i is matrix i) and every work array is carved from ONE file-scope __device__ array
// of CDU_PSD_STATIC_BYTES that each GPU which loads the library holds until exit. The entry point issues kernel launches
// and one device-to-device copy and nothing else: no cudaMalloc / cudaFree / allocating library routine, no host
// synchronisation. (A kernel of its own also keeps cudaFuncSetAttribute away from k_psd_fwd_small, whose instantiations are
// shared with the handles' translation units: their dynamic shared-memory limit is state this file must not touch.)
//
// The array is shared by every call and keeps the last call's contents: k_static_clear zeroes what must start at zero
// (flags, sweep counters); every other part is fully overwritten before it is read. Two calls that overlap on the GPU
// (different streams, or two host threads) race on it - callers serialise.
#include <mutex>

#include "handle.cuh"

namespace cdu {
namespace pstatic {

constexpr size_t PSD_STATIC_BYTES = (size_t)CDU_PSD_STATIC_BYTES;
constexpr int PSD_STATIC_MAX_P = CDU_PSD_STATIC_MAX_P;
constexpr int MAX_DEVICES = 64;

static __device__ __align__(256) unsigned char g_psd_static_scratch[PSD_STATIC_BYTES];

// carve-up of the array for (count, p, sizeof(T)); every part starts on a 256-byte boundary
struct Layout {
  size_t head, flags, W, S1, Us, Ls, total;
};
static inline Layout layout_of(int count, int p, size_t sz) {
  Layout L;
  size_t o = 0;
  auto take = [&](size_t bytes) { const size_t at = o; o += (bytes + 255) & ~(size_t)255; return at; };
  const size_t tot = (size_t)p * (p + 1) / 2 * count;
  L.head = take(64);                                   // [0] sweeps_max (int), [8] sweeps_sum (unsigned long long)
  L.flags = take(sizeof(int) * count);                 // FLAG_* of common.cuh per matrix
  L.W = take(sizeof(double) * tot);                    // svec(S)
  L.S1 = take(sizeof(double) * tot);                   // svec(Pi(S))
  L.Us = take(sz * (size_t)count * p * p);             // eigenvectors as rows
  L.Ls = take(sz * (size_t)count * p);                 // eigenvalues
  L.total = o;
  return L;
}

struct StaticArgs {
  const double* W; double* S1; void* Us; void* Ls; int* flags; int* sweeps_max; unsigned long long* sweeps_sum;
};

__global__ void k_static_clear(int count, StaticArgs A) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) { *A.sweeps_max = 0; *A.sweeps_sum = 0ull; }
  if (i < count) A.flags[i] = 0;
}

// One CTA per matrix: smat(w) into the Jacobi planes, cyclic Jacobi in shared memory, eigenpairs out, rebuild
// Pi(S) = sum_{lambda_i > 0} lambda_i u_i u_i' (Eq. 7) in svec form. blockDim.x as psd_small_cfg(p) says.
template <typename T, int MAXI>
__global__ void __launch_bounds__(psd_small_max_threads(MAXI)) k_psd_project_static(int p, StaticArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int blk = blockIdx.x, pe = (p + 1) & ~1, nsv = p * (p + 1) / 2;
  double* shred = reinterpret_cast<double*>(smem_raw);                      // 64 doubles of reduction scratch
  const JacobiWs<T> ws = jacobi_ws_carve<T>(smem_raw + 512, pe);
  T* lp = reinterpret_cast<T*>(smem_raw + 512 + jacobi_ws_bytes<T>(pe));    // max(lambda, 0) by player
  const double* w = A.W + (size_t)blk * nsv;
  const int ldv = ws.ldv, h = pe >> 1, ldh = h | 1, psz = h * ldh;
  load_smat_planes<T>(p, pe, ws.P0, w, 0.0, nullptr);
  __syncthreads();
  int flag = 0, cur = 0;
  const int sweeps = jacobi_planes<T, MAXI>(pe, ws, shred, 40, &flag, &cur, false);
  T* U = reinterpret_cast<T*>(A.Us) + (size_t)blk * p * p;
  T* L = reinterpret_cast<T*>(A.Ls) + (size_t)blk * p;
  for (int pos = threadIdx.x; pos < pe; pos += blockDim.x) {
    const int q = pos >> 1, pl = ws.plr0[cur * pe + pos];
    const T l = ws.P0[cur * ws.pstride + ((pos & 1) ? 3 * psz : 0) + q * ldh + q];
    lp[pl] = l > (T)0 ? l : (T)0;
    if (pl < p) L[pl] = l;
  }
  for (int t = threadIdx.x; t < p * p; t += blockDim.x) { const int i = t / p, a = t - i * p; U[t] = ws.Vt[i * ldv + a]; }
  __syncthreads();
  double* s1 = A.S1 + (size_t)blk * nsv;
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
    s1[t] = (a == b) ? (double)acc : (double)acc * 1.41421356237309504880;
  }
  if (threadIdx.x == 0) {
    atomicMax(A.sweeps_max, sweeps);
    atomicAdd(A.sweeps_sum, (unsigned long long)sweeps);
    if (flag) atomicOr(A.flags + blk, flag);
  }
}

// once per device, with that device current: the array's device address (in host code the array's name is only a stand-in
// for it: a kernel given that would fault) and the dynamic shared-memory limit of this file's own Jacobi kernels
struct PerDevice { unsigned char* base = nullptr; bool attr32 = false, attr64 = false; };
static PerDevice g_dev[MAX_DEVICES];
static std::mutex g_mu;

template <typename T>
static cdu_status device_setup(int dev, unsigned char** base, std::string& err) {
  std::lock_guard<std::mutex> lk(g_mu);
  PerDevice& d = g_dev[dev];
  if (!d.base) {
    unsigned char* ptr = nullptr;
    CU_OK(cudaGetSymbolAddress((void**)&ptr, g_psd_static_scratch));
    if (!ptr) { err = "cdu_psd_project_static: cudaGetSymbolAddress returned NULL"; return CDU_ECUDA; }
    d.base = ptr;
  }
  bool& done = std::is_same<T, float>::value ? d.attr32 : d.attr64;
  if (!done) {
    size_t sb = 0;                                     // not monotone in p (odd leading dimensions): take the maximum
    for (int q = 1; q <= PSD_STATIC_MAX_P; ++q) sb = std::max(sb, psd_small_smem_bytes(q, sizeof(T)));
    const void* fn[2] = {(const void*)k_psd_project_static<T, 1>, (const void*)k_psd_project_static<T, 2>};
    for (const void* f : fn) CU_OK(cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sb));
    done = true;
  }
  *base = d.base;
  return CDU_OK;
}

template <typename T>
static cdu_status project_t(int count, int p, const void* S, void* PiS, void* U, void* lam, cudaStream_t st) {
  std::string& err = create_error();
  if (count < 1 || p < 1 || !S || !PiS) { err = "cdu_psd_project_static: bad arguments"; return CDU_EINVAL; }
  if (p > PSD_STATIC_MAX_P) {
    err = "cdu_psd_project_static: p = " + std::to_string(p) + " exceeds the maximum order " + std::to_string(PSD_STATIC_MAX_P);
    return CDU_EINVAL;
  }
  if (count > (1 << 24)) { err = "cdu_psd_project_static: count too large"; return CDU_EINVAL; }
  const Layout L = layout_of(count, p, sizeof(T));
  if (L.total > PSD_STATIC_BYTES) {
    err = "cdu_psd_project_static: count = " + std::to_string(count) + ", p = " + std::to_string(p) + " needs " + std::to_string(L.total) +
          " bytes of scratch, the static array holds " + std::to_string(PSD_STATIC_BYTES);
    return CDU_EINVAL;
  }
  const PsdSmallCfg cfg = psd_small_cfg(p, sizeof(T));
  const size_t sm = psd_small_smem_bytes(p, sizeof(T));
  if (cfg.maxi > 2) {   // orders up to CDU_PSD_STATIC_MAX_P need at most two register-resident items per thread
     err = "cdu_psd_project_static: order too large for the shared-memory Jacobi"; return CDU_EINVAL; }
  int dev = 0;
  CU_OK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEVICES) { err = "cdu_psd_project_static: device ordinal out of range"; return CDU_EINVAL; }
  unsigned char* base = nullptr;
  const cdu_status s0 = device_setup<T>(dev, &base, err);
  if (s0 != CDU_OK) return s0;

  double *W = reinterpret_cast<double*>(base + L.W), *S1 = reinterpret_cast<double*>(base + L.S1);
  T *Us = reinterpret_cast<T*>(base + L.Us), *Ls = reinterpret_cast<T*>(base + L.Ls);
  StaticArgs A; A.W = W; A.S1 = S1; A.Us = Us; A.Ls = Ls; A.flags = reinterpret_cast<int*>(base + L.flags);
  A.sweeps_max = reinterpret_cast<int*>(base + L.head); A.sweeps_sum = reinterpret_cast<unsigned long long*>(base + L.head + 8);
  k_static_clear<<<(count + 255) / 256, 256, 0, st>>>(count, A);
  impl::k_dense_to_svec<T><<<count, 256, 0, st>>>(p, (const T*)S, W);
  if (cfg.maxi == 1) k_psd_project_static<T, 1><<<count, cfg.threads, sm, st>>>(p, A);
  else k_psd_project_static<T, 2><<<count, cfg.threads, sm, st>>>(p, A);
  impl::k_svec_to_dense<T><<<count, 256, 0, st>>>(p, S1, (T*)PiS);
  if (U) impl::k_transpose_batched<T><<<count, 256, 0, st>>>(p, Us, (T*)U);    // stored as rows, returned in columns
  if (lam) CU_OK(cudaMemcpyAsync(lam, Ls, (size_t)count * p * sizeof(T), cudaMemcpyDeviceToDevice, st));
  CU_OK(cudaGetLastError());
  return CDU_OK;
}

}  // namespace pstatic
}  // namespace cdu

extern "C" cdu_status cdu_psd_project_static(int32_t dtype, int32_t count, int32_t p, const void* S, void* PiS, void* U, void* lam,
                                             void* cuda_stream) {
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
    (void)cudaGetLastError();
    cdu::create_error() = "cdu_psd_project_static: no CUDA device (there is no CPU fallback)";
    return CDU_ECUDA;
  }
  if (dtype == CDU_F32) return cdu::pstatic::project_t<float>(count, p, S, PiS, U, lam, st);
  if (dtype == CDU_F64) return cdu::pstatic::project_t<double>(count, p, S, PiS, U, lam, st);
  cdu::create_error() = "cdu_psd_project_static: bad dtype";
  return CDU_EINVAL;
}

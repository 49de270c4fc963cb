"""paper_2606_13825_b200 - thin Python binding of the cdu C ABI (include/cdu.h).

Argument marshalling only: every step of the hot path (CSR SpMV / PCG, relaxation, cone projections incl.
the PSD eigendecomposition, checkpointing, adjoint CG, Dalecki-Krein VJP) runs in the CUDA kernels of
`csrc/` behind `libcdu.so`. PyTorch is used for device memory and streams only. There is no CPU fallback:
if the library is missing or no CUDA device is present, the calls raise.

Names follow the C ABI: `cdu_create`, `cdu_forward`, `cdu_backward`, `cdu_get_stats`, `cdu_destroy`,
`cdu_psd_project`, `cdu_psd_vjp`, `cdu_psd_project_static`.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libcdu.so")

CDU_OK, CDU_EINVAL, CDU_ENOMEM, CDU_ECUDA, CDU_ESTATE, CDU_ENUMERIC = range(6)
CDU_F32, CDU_F64 = 0, 1
CDU_ZERO, CDU_NONNEG, CDU_SOC, CDU_PSD = 0, 1, 2, 3
CDU_RHO_PER_ITER, CDU_RHO_PER_PROBLEM, CDU_RHO_PER_ROW = 0, 1, 2
CDU_CKPT_FULL, CDU_CKPT_LEAN = 0, 1
_STATUS = {0: "CDU_OK", 1: "CDU_EINVAL", 2: "CDU_ENOMEM", 3: "CDU_ECUDA", 4: "CDU_ESTATE", 5: "CDU_ENUMERIC"}

EXPORTED_SYMBOLS = ("cdu_create", "cdu_forward", "cdu_backward", "cdu_get_stats", "cdu_get_iterate", "cdu_last_error",
                    "cdu_destroy", "cdu_version", "cdu_psd_project", "cdu_psd_vjp", "cdu_profile", "cdu_get_profile",
                    "cdu_measure_peak", "cdu_backward_inject", "cdu_backward_eq12", "cdu_get_features", "cdu_solve", "cdu_rectify_rho",
                    "cdu_psd_project_static")


class CduError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


class _Cone(C.Structure):
    _fields_ = [("kind", C.c_int32), ("dim", C.c_int32)]


class _Problem(C.Structure):
    _fields_ = [("batch", C.c_int32), ("dtype", C.c_int32),
                ("var_off", C.c_void_p), ("row_off", C.c_void_p),
                ("A_rowptr", C.c_void_p), ("A_colidx", C.c_void_p), ("A_val", C.c_void_p),
                ("P_rowptr", C.c_void_p), ("P_colidx", C.c_void_p), ("P_val", C.c_void_p),
                ("q", C.c_void_p), ("b", C.c_void_p), ("cone_off", C.c_void_p), ("cones", C.c_void_p)]


class _Options(C.Structure):
    _fields_ = [("cg_tol", C.c_double), ("cg_max_iter", C.c_int32), ("K_max", C.c_int32), ("ckpt_mode", C.c_int32),
                ("cg_refine", C.c_int32), ("cg_refine_tol", C.c_double), ("psd_small_max", C.c_int32),
                ("use_tensor_cores", C.c_int32), ("team_size", C.c_int32), ("no_batch", C.c_int32), ("no_diag_path", C.c_int32)]


class _Stats(C.Structure):
    _fields_ = [("cg_iters_fwd", C.c_int64), ("cg_iters_bwd", C.c_int64), ("cg_iters_max", C.c_int32),
                ("eig_sweeps_max", C.c_int32), ("n_flagged", C.c_int32), ("flags_or", C.c_int32),
                ("device_bytes", C.c_int64), ("ckpt_bytes", C.c_int64), ("launches", C.c_int64),
                ("eig_sweeps_sum", C.c_int64), ("cg_iters_fwd_pass0", C.c_int64), ("cg_iters_bwd_pass0", C.c_int64)]


_lib = None


def load_library(path: Optional[str] = None) -> C.CDLL:
    """dlopen libcdu.so (no compute happens here; works without a GPU)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise CduError(CDU_ECUDA, f"{p} not found - run `python -m paper_2606_13825_b200.build` (there is no CPU fallback)")
    lib = C.CDLL(p)
    vp, i32, f64 = C.c_void_p, C.c_int32, C.c_double
    lib.cdu_create.restype = i32
    lib.cdu_create.argtypes = [C.POINTER(_Problem), C.POINTER(_Options), vp, C.POINTER(vp)]
    lib.cdu_forward.restype = i32
    lib.cdu_forward.argtypes = [vp, i32, vp, i32, f64, vp, vp, vp, vp, vp, vp, vp, i32, vp]
    lib.cdu_backward.restype = i32
    lib.cdu_backward.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, i32, vp]
    lib.cdu_backward_inject.restype = i32
    lib.cdu_backward_inject.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, i32, vp]
    lib.cdu_backward_eq12.restype = i32
    lib.cdu_backward_eq12.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i32, vp]
    lib.cdu_get_features.restype = i32
    lib.cdu_get_features.argtypes = [vp, i32, vp, vp, vp, vp, vp, i32, vp]
    lib.cdu_rectify_rho.restype = i32
    lib.cdu_rectify_rho.argtypes = [vp, i32, vp, i32, vp]
    lib.cdu_solve.restype = i32
    lib.cdu_solve.argtypes = [vp, i32, i32, f64, f64, f64, f64, i32, f64, vp, vp, vp, vp, vp, vp, vp, vp, i32, vp]
    lib.cdu_get_stats.restype = i32
    lib.cdu_get_stats.argtypes = [vp, C.POINTER(_Stats)]
    lib.cdu_get_iterate.restype = i32
    lib.cdu_get_iterate.argtypes = [vp, i32, vp, vp, vp, i32, vp]
    lib.cdu_last_error.restype = C.c_char_p
    lib.cdu_last_error.argtypes = [vp]
    lib.cdu_destroy.restype = i32
    lib.cdu_destroy.argtypes = [vp]
    lib.cdu_version.restype = C.c_char_p
    lib.cdu_version.argtypes = []
    lib.cdu_profile.restype = i32
    lib.cdu_profile.argtypes = [vp, i32]
    lib.cdu_get_profile.restype = i32
    lib.cdu_get_profile.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
    lib.cdu_psd_project.restype = i32
    lib.cdu_psd_project.argtypes = [i32, i32, i32, vp, vp, vp, vp, i32, i32, vp]
    lib.cdu_psd_project_static.restype = i32
    lib.cdu_psd_project_static.argtypes = [i32, i32, i32, vp, vp, vp, vp, vp]
    lib.cdu_psd_vjp.restype = i32
    lib.cdu_psd_vjp.argtypes = [i32, i32, i32, vp, vp, vp, vp, i32, i32, vp]
    lib.cdu_measure_peak.restype = i32
    lib.cdu_measure_peak.argtypes = [i32, C.POINTER(C.c_double), vp]
    if path is None:
        _lib = lib
    return lib


def _torch():
    import torch
    return torch


def _ptr(t) -> Optional[int]:
    """Address of a torch tensor (device or pinned host) or numpy array; None passes NULL."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return t.ctypes.data
    assert t.is_contiguous()
    return t.data_ptr()


def _stream() -> int:
    return _torch().cuda.current_stream().cuda_stream


class Handle:
    """Owns a `cdu_handle`. `packed` is the dict of `workloads.pack_batch` (host numpy arrays)."""

    def __init__(self, packed: dict, K_max: int, ckpt_mode: int = CDU_CKPT_FULL, cg_tol: float = 0.0,
                 cg_max_iter: int = 0, cg_refine: int = -1, cg_refine_tol: float = 0.0, psd_small_max: int = 0,
                 use_tensor_cores: int = -1, team_size: int = 0, no_batch: int = 0, no_diag_path: int = 0):
        torch = _torch()
        if not torch.cuda.is_available():
            raise CduError(CDU_ECUDA, "no CUDA device (there is no CPU fallback)")
        self.lib = load_library()
        self.dtype = packed["dtype"]
        self.np_dtype = np.float32 if self.dtype == "f32" else np.float64
        self.torch_dtype = torch.float32 if self.dtype == "f32" else torch.float64
        self.B = int(packed["batch"])
        self.N = int(packed["var_off"][-1])
        self.M = int(packed["row_off"][-1])
        keep = {k: np.ascontiguousarray(packed[k]) for k in
                ("var_off", "row_off", "A_rowptr", "A_colidx", "A_val", "P_rowptr", "P_colidx", "P_val", "q", "b",
                 "cone_off", "cones")}
        assert keep["A_val"].dtype == self.np_dtype and keep["q"].dtype == self.np_dtype
        assert keep["var_off"].dtype == np.int64 and keep["A_colidx"].dtype == np.int32 and keep["cones"].dtype == np.int32
        pr = _Problem(batch=self.B, dtype=CDU_F32 if self.dtype == "f32" else CDU_F64,
                      **{k: v.ctypes.data for k, v in keep.items()})
        op = _Options(cg_tol=cg_tol, cg_max_iter=cg_max_iter, K_max=K_max, ckpt_mode=ckpt_mode, cg_refine=cg_refine,
                      cg_refine_tol=cg_refine_tol, psd_small_max=psd_small_max, use_tensor_cores=use_tensor_cores,
                      team_size=team_size, no_batch=no_batch, no_diag_path=no_diag_path)
        h = C.c_void_p()
        st = self.lib.cdu_create(C.byref(pr), C.byref(op), _stream(), C.byref(h))
        if st != CDU_OK:
            raise CduError(st, self.lib.cdu_last_error(None).decode())
        self.h = h
        self.K_max = K_max
        self.K = 0
        self.rho_mode = CDU_RHO_PER_ITER

    def _check(self, st: int):
        if st != CDU_OK:
            raise CduError(st, self.lib.cdu_last_error(self.h).decode())

    def _want(self, name, t, numel, host):
        """Marshalling check: the C ABI takes bare pointers, so a wrong dtype or a short array would be read out of bounds."""
        if t is None:
            return
        n = t.size if isinstance(t, np.ndarray) else t.numel()
        dt = str(t.dtype).replace("torch.", "")
        want = "float32" if self.dtype == "f32" else "float64"
        if dt != want:
            raise ValueError(f"{name}: dtype {dt}, the handle computes in {want}")
        if n < numel:
            raise ValueError(f"{name}: {n} elements, at least {numel} are read")
        if not isinstance(t, np.ndarray) and t.is_cuda == bool(host):
            raise ValueError(f"{name}: {'host' if host else 'device'} tensor expected (host={host})")

    def forward(self, K, rho, alpha, sigma, x0=None, s0=None, y0=None, rho_mode=CDU_RHO_PER_ITER, out=None, host=False):
        """cdu_forward. Device mode: torch CUDA tensors in, returns (xK, sK, yK) CUDA tensors.
        Host mode: pinned torch CPU tensors / numpy arrays in and out (copies are inside the call)."""
        torch = _torch()
        cnt = K * (1 if rho_mode == CDU_RHO_PER_ITER else self.B)
        for nm, t, n in (("rho", rho, K * self.M if rho_mode == CDU_RHO_PER_ROW else cnt), ("alpha", alpha, cnt), ("x0", x0, self.N), ("s0", s0, self.M), ("y0", y0, self.M)):
            self._want(nm, t, n, host)
        if out is None:
            if host:
                out = tuple(torch.empty(n, dtype=self.torch_dtype).pin_memory() for n in (self.N, self.M, self.M))
            else:
                out = tuple(torch.empty(n, dtype=self.torch_dtype, device="cuda") for n in (self.N, self.M, self.M))
        self._check(self.lib.cdu_forward(self.h, K, _ptr(rho), rho_mode, float(sigma), _ptr(alpha), _ptr(x0), _ptr(s0),
                                         _ptr(y0), _ptr(out[0]), _ptr(out[1]), _ptr(out[2]), 1 if host else 0, _stream()))
        self.K, self.rho_mode = K, rho_mode
        return out

    def backward(self, g_xK=None, g_sK=None, g_yK=None, out=None, host=False):
        """cdu_backward -> dict(g_rho, g_alpha, g_sigma, g_x0, g_s0, g_y0)."""
        torch = _torch()
        if out is None:
            out = self._grad_out(host)
        for nm, t, n in (("g_xK", g_xK, self.N), ("g_sK", g_sK, self.M), ("g_yK", g_yK, self.M)):
            self._want(nm, t, n, host)
        self._check(self.lib.cdu_backward(self.h, _ptr(g_xK), _ptr(g_sK), _ptr(g_yK), _ptr(out.get("g_rho")),
                                          _ptr(out.get("g_sigma")), _ptr(out.get("g_alpha")), _ptr(out.get("g_x0")),
                                          _ptr(out.get("g_s0")), _ptr(out.get("g_y0")), 1 if host else 0, _stream()))
        return out

    def _grad_out(self, host):
        torch = _torch()
        cnt = self.K * (1 if self.rho_mode == CDU_RHO_PER_ITER else self.B)
        scnt = 1 if self.rho_mode == CDU_RHO_PER_ITER else self.B
        sizes = dict(g_rho=self.K * self.M if self.rho_mode == CDU_RHO_PER_ROW else cnt, g_alpha=cnt, g_sigma=scnt, g_x0=self.N, g_s0=self.M, g_y0=self.M)
        if host:
            return {k: torch.empty(n, dtype=self.torch_dtype).pin_memory() for k, n in sizes.items()}
        return {k: torch.empty(n, dtype=self.torch_dtype, device="cuda") for k, n in sizes.items()}

    def backward_inject(self, g_xK=None, g_sK=None, g_yK=None, inj_x=None, inj_s=None, inj_y=None, host=False):
        """cdu_backward_inject: inj_x [K-1, N], inj_s, inj_y [K-1, M] are cotangents on z^1 .. z^(K-1)."""
        out = self._grad_out(host)
        self._check(self.lib.cdu_backward_inject(self.h, _ptr(g_xK), _ptr(g_sK), _ptr(g_yK), _ptr(inj_x), _ptr(inj_s), _ptr(inj_y),
                                                 _ptr(out["g_rho"]), _ptr(out["g_sigma"]), _ptr(out["g_alpha"]), _ptr(out["g_x0"]),
                                                 _ptr(out["g_s0"]), _ptr(out["g_y0"]), 1 if host else 0, _stream()))
        return out

    def backward_eq12(self, host=False):
        """cdu_backward_eq12 -> (loss [B], gradients dict): the Eq. 12 training loss of the last forward and its reverse sweep."""
        torch = _torch()
        out = self._grad_out(host)
        loss = torch.empty(self.B, dtype=self.torch_dtype).pin_memory() if host else torch.empty(self.B, dtype=self.torch_dtype, device="cuda")
        self._check(self.lib.cdu_backward_eq12(self.h, _ptr(loss), _ptr(out["g_rho"]), _ptr(out["g_sigma"]), _ptr(out["g_alpha"]),
                                               _ptr(out["g_x0"]), _ptr(out["g_s0"]), _ptr(out["g_y0"]), 1 if host else 0, _stream()))
        return loss, out

    def features(self, k: int):
        """cdu_get_features of iterate k -> dict(rp_bar [M], rd_bar [N], delta_p [M], delta_d [M], scal [B, 3])."""
        torch = _torch()
        mk = lambda n: torch.empty(n, dtype=self.torch_dtype, device="cuda")
        o = dict(rp_bar=mk(self.M), rd_bar=mk(self.N), delta_p=mk(self.M), delta_d=mk(self.M), scal=mk(self.B * 3))
        self._check(self.lib.cdu_get_features(self.h, k, _ptr(o["rp_bar"]), _ptr(o["rd_bar"]), _ptr(o["delta_p"]), _ptr(o["delta_d"]),
                                              _ptr(o["scal"]), 0, _stream()))
        o["scal"] = o["scal"].view(self.B, 3)
        return o

    def rectify_rho(self, K, rho):
        """cdu_rectify_rho in place on a device tensor [K, M]."""
        self._check(self.lib.cdu_rectify_rho(self.h, int(K), _ptr(rho), 0, _stream()))
        return rho

    def solve(self, max_iter, check_every, eps, rho0=0.1, alpha=1.6, sigma=1e-6, adapt_rho=True, eq_scale=1.0, x0=None, s0=None, y0=None):
        """cdu_solve (device pointers) -> (x, s, y, iters [B] numpy int32, res [B, 2] numpy)."""
        torch = _torch()
        out = tuple(torch.empty(n, dtype=self.torch_dtype, device="cuda") for n in (self.N, self.M, self.M))
        iters = np.zeros(self.B, np.int32); res = np.zeros((self.B, 2), np.float64)
        self._check(self.lib.cdu_solve(self.h, int(max_iter), int(check_every), float(eps), float(rho0), float(alpha), float(sigma),
                                       1 if adapt_rho else 0, float(eq_scale), _ptr(x0), _ptr(s0), _ptr(y0), _ptr(out[0]), _ptr(out[1]), _ptr(out[2]),
                                       iters.ctypes.data, res.ctypes.data, 0, _stream()))
        self.K, self.rho_mode = int(check_every), CDU_RHO_PER_PROBLEM
        return out[0], out[1], out[2], iters, res

    def iterate(self, k: int):
        torch = _torch()
        out = tuple(torch.empty(n, dtype=self.torch_dtype, device="cuda") for n in (self.N, self.M, self.M))
        self._check(self.lib.cdu_get_iterate(self.h, k, _ptr(out[0]), _ptr(out[1]), _ptr(out[2]), 0, _stream()))
        return out

    def stats(self) -> dict:
        """cdu_get_stats. `status` is CDU_OK or CDU_ENUMERIC (some problem raised a flag: see `flags_or`)."""
        s = _Stats()
        st = self.lib.cdu_get_stats(self.h, C.byref(s))
        if st not in (CDU_OK, CDU_ENUMERIC):
            self._check(st)
        d = {k: getattr(s, k) for k, _ in _Stats._fields_}
        d["status"] = st
        return d

    PROFILE_CLASSES = ("lin_fwd", "psd_fwd_small", "eig_large", "gemm_large", "lin_bwd", "psd_bwd_small", "large_misc", "misc")

    def profile(self, enable: bool):
        self._check(self.lib.cdu_profile(self.h, 1 if enable else 0))

    def get_profile(self) -> dict:
        n = len(self.PROFILE_CLASSES)
        ms = (C.c_double * n)(); cnt = (C.c_int64 * n)()
        self._check(self.lib.cdu_get_profile(self.h, n, ms, cnt))
        return {name: dict(ms=ms[i], launches=cnt[i]) for i, name in enumerate(self.PROFILE_CLASSES)}

    def close(self):
        if getattr(self, "h", None):
            self.lib.cdu_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- function-style aliases with the ABI's names ---------------------------------------------------------
def cdu_create(packed: dict, K_max: int, **options) -> Handle:
    return Handle(packed, K_max, **options)


def cdu_forward(h: Handle, K, rho, alpha, sigma, x0=None, s0=None, y0=None, **kw):
    return h.forward(K, rho, alpha, sigma, x0, s0, y0, **kw)


def cdu_backward(h: Handle, g_xK=None, g_sK=None, g_yK=None, **kw):
    return h.backward(g_xK, g_sK, g_yK, **kw)


def cdu_get_stats(h: Handle) -> dict:
    return h.stats()


def cdu_destroy(h: Handle) -> None:
    h.close()


CDU_PEAK_FP32_FMA, CDU_PEAK_FP64_FMA, CDU_PEAK_TF32_TENSOR, CDU_PEAK_HBM_COPY, CDU_PEAK_TF32_MMA_SYNC = range(5)


def cdu_measure_peak(kind: int) -> float:
    """In-tree micro-benchmark of a roofline denominator (TFLOP/s, or GB/s for the copy); see include/cdu.h."""
    if not _torch().cuda.is_available():
        raise CduError(CDU_ECUDA, "no CUDA device (there is no CPU fallback)")
    lib = load_library()
    v = C.c_double(0.0)
    st = lib.cdu_measure_peak(kind, C.byref(v), _stream())
    if st != CDU_OK:
        raise CduError(st, "cdu_measure_peak failed")
    return float(v.value)


def cdu_psd_project(S, path: int = 0, use_tensor_cores: int = 0, want_eig: bool = True):
    """Batched Pi(S) for a CUDA tensor S [count, p, p]; returns (PiS, U, lam)."""
    torch = _torch()
    lib = load_library()
    assert S.is_cuda and S.dim() == 3 and S.shape[1] == S.shape[2]
    S = S.contiguous()
    cnt, p = S.shape[0], S.shape[1]
    dt = CDU_F32 if S.dtype == torch.float32 else CDU_F64
    out = torch.empty_like(S)
    U = torch.empty_like(S) if want_eig else None
    lam = torch.empty(cnt, p, dtype=S.dtype, device=S.device) if want_eig else None
    st = lib.cdu_psd_project(dt, cnt, p, _ptr(S), _ptr(out), _ptr(U), _ptr(lam), path, use_tensor_cores, _stream())
    if st != CDU_OK:
        raise CduError(st, lib.cdu_last_error(None).decode())
    return out, U, lam


PSD_STATIC_BYTES = 8 << 20     # CDU_PSD_STATIC_BYTES of include/cdu.h
PSD_STATIC_MAX_P = 64          # CDU_PSD_STATIC_MAX_P


def cdu_psd_project_static(S, PiS, U=None, lam=None) -> None:
    """Batched Pi(S) with no allocation anywhere: S and every output are the caller's CUDA tensors (S, PiS, U
    [count, p, p], lam [count, p], one dtype, contiguous); the scratch is a static device array inside the library
    (include/cdu.h: limits, and why overlapping calls race). Enqueues on the current stream and does not synchronise."""
    torch = _torch()
    lib = load_library()
    if not (S.is_cuda and S.dim() == 3 and S.shape[1] == S.shape[2] and S.is_contiguous()):
        raise CduError(CDU_EINVAL, "S must be a contiguous CUDA tensor [count, p, p]")
    if S.dtype not in (torch.float32, torch.float64):
        raise CduError(CDU_EINVAL, "S must be float32 or float64")
    cnt, p = S.shape[0], S.shape[1]
    for name, t, shape in (("PiS", PiS, (cnt, p, p)), ("U", U, (cnt, p, p)), ("lam", lam, (cnt, p))):
        if t is None and name != "PiS":
            continue
        if t is None or not t.is_cuda or t.dtype != S.dtype or tuple(t.shape) != shape or not t.is_contiguous() or t.device != S.device:
            raise CduError(CDU_EINVAL, f"{name} must be a contiguous CUDA tensor of shape {shape} and S's dtype and device")
    dt = CDU_F32 if S.dtype == torch.float32 else CDU_F64
    st = lib.cdu_psd_project_static(dt, cnt, p, _ptr(S), _ptr(PiS), _ptr(U), _ptr(lam), _stream())
    if st != CDU_OK:
        raise CduError(st, lib.cdu_last_error(None).decode())


def cdu_psd_vjp(U, lam, Gbar, path: int = 0, use_tensor_cores: int = 0):
    """Batched Dalecki-Krein VJP; U [count,p,p] (eigenvectors in columns), lam [count,p], Gbar [count,p,p]."""
    torch = _torch()
    lib = load_library()
    U, lam, Gbar = U.contiguous(), lam.contiguous(), Gbar.contiguous()
    cnt, p = U.shape[0], U.shape[1]
    dt = CDU_F32 if U.dtype == torch.float32 else CDU_F64
    out = torch.empty_like(Gbar)
    st = lib.cdu_psd_vjp(dt, cnt, p, _ptr(U), _ptr(lam), _ptr(Gbar), _ptr(out), path, use_tensor_cores, _stream())
    if st != CDU_OK:
        raise CduError(st, lib.cdu_last_error(None).decode())
    return out

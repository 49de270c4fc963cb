"""cdu_psd_project_static (include/cdu.h): the PSD projection of PAPER.md Eq. 7 with its scratch in a static device
array, for callers that may not call cudaMalloc. Checked against the existing cdu_psd_project (path 1, the same
shared-memory Jacobi code) and against the oracle's projection, on two calls in a row that share the array.
Named test_zz_* so that pytest collects it last (the suite runs with pytest -x)."""
import numpy as np
import pytest

from oracle import cones as C

pytestmark = pytest.mark.gpu


def _sym(rng, cnt, p):
    S = rng.standard_normal((cnt, p, p))
    return 0.5 * (S + S.transpose(0, 2, 1))


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_static_scratch_projection_matches_existing_path_twice(dtype):
    import torch
    import paper_2606_13825_b200 as cdu
    tdt = torch.float32 if dtype == "f32" else torch.float64
    tol = 2e-5 if dtype == "f32" else 1e-12                       # the tolerances of test_psd_ops_gpu.py
    rng = np.random.default_rng(2606)
    # second call: other order, other count, so the carve-up of the shared array moves and stale contents of the first
    # call lie under every part of it
    for cnt, p in ((7, 50), (19, 33)):
        S = _sym(rng, cnt, p)
        S = S.astype(np.float32).astype(np.float64) if dtype == "f32" else S
        St = torch.as_tensor(S, dtype=tdt, device="cuda")
        Pi = torch.full_like(St, float("nan"))
        U = torch.full_like(St, float("nan"))
        lam = torch.full((cnt, p), float("nan"), dtype=tdt, device="cuda")
        before = torch.cuda.memory_allocated()
        cdu.cdu_psd_project_static(St, Pi, U, lam)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() == before            # the binding allocates nothing either
        Pi0, U0, lam0 = cdu.cdu_psd_project(St, path=1)
        torch.cuda.synchronize()
        Pn, Un, ln = (t.double().cpu().numpy() for t in (Pi, U, lam))
        P0n, l0n = Pi0.double().cpu().numpy(), lam0.double().cpu().numpy()
        for i in range(cnt):
            n2 = np.linalg.norm(S[i], 2)
            assert np.isfinite(Pn[i]).all() and np.isfinite(Un[i]).all() and np.isfinite(ln[i]).all()
            assert np.abs(Pn[i] - P0n[i]).max() <= tol * n2                         # against the existing path
            assert np.abs(np.sort(ln[i]) - np.sort(l0n[i])).max() <= tol * n2
            ref = C.smat(C.proj_psd(C.svec(S[i]))[0])                               # and against the oracle
            assert np.abs(Pn[i] - ref).max() <= tol * n2
            assert np.abs(Un[i].T @ Un[i] - np.eye(p)).max() <= (5e-6 if dtype == "f32" else 1e-13)
            assert np.abs((Un[i] * np.maximum(ln[i], 0.0)) @ Un[i].T - ref).max() <= 4 * tol * n2


def test_static_scratch_same_input_twice_and_optional_outputs():
    """The same input twice in a row gives the same bits (nothing of the first call leaks into the second); U and lam
    may be NULL; PiS may alias S."""
    import torch
    import paper_2606_13825_b200 as cdu
    rng = np.random.default_rng(7)
    St = torch.as_tensor(_sym(rng, 5, 64), dtype=torch.float64, device="cuda")
    a, b = torch.empty_like(St), torch.empty_like(St)
    cdu.cdu_psd_project_static(St, a)
    cdu.cdu_psd_project_static(St, b)
    c = St.clone()
    cdu.cdu_psd_project_static(c, c)
    torch.cuda.synchronize()
    assert torch.equal(a, b) and torch.equal(a, c)
    ref = cdu.cdu_psd_project(St, path=1, want_eig=False)[0]
    assert float((a - ref).abs().max()) <= 1e-12 * float(torch.linalg.matrix_norm(St, 2).max())


def test_static_scratch_limits_are_errors():
    import torch
    import paper_2606_13825_b200 as cdu
    for cnt, p, what in ((1, cdu.PSD_STATIC_MAX_P + 1, "maximum order"), (200, 64, "bytes of scratch")):
        St = torch.zeros(cnt, p, p, dtype=torch.float64, device="cuda")
        out = torch.full_like(St, 3.0)
        with pytest.raises(cdu.CduError) as e:
            cdu.cdu_psd_project_static(St, out)
        assert e.value.status == cdu.CDU_EINVAL and what in str(e.value)
        torch.cuda.synchronize()
        assert bool((out == 3.0).all())                            # nothing was launched
    St = torch.zeros(120, 64, 64, dtype=torch.float64, device="cuda")       # the documented size at p = 64 fits
    out = torch.full_like(St, 3.0)
    cdu.cdu_psd_project_static(St, out)
    torch.cuda.synchronize()
    assert bool((out == 0.0).all())

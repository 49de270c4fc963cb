"""GPU unit tests of the stand-alone PSD projection / Dalecki-Krein VJP entry points (both kernel paths)
against the oracle's cone functions: projected matrices are compared, never eigenvectors."""
import numpy as np
import pytest

from oracle import cones as C

pytestmark = pytest.mark.gpu

# (dtype, order, path, tensor cores): path 1 = shared-memory Jacobi, 2 = large-block path; tc = tcgen05 3xTF32 products
CASES = [("f32", 10, 1, 0), ("f32", 50, 1, 0), ("f32", 100, 1, 0), ("f32", 128, 1, 0), ("f32", 33, 2, 0), ("f32", 140, 2, 0),
         ("f32", 512, 2, 0), ("f32", 128, 2, 1), ("f32", 256, 2, 1), ("f32", 512, 2, 1),
         ("f64", 10, 1, 0), ("f64", 51, 1, 0), ("f64", 64, 2, 0), ("f64", 140, 2, 0)]


def _sym(rng, cnt, p):
    S = rng.standard_normal((cnt, p, p))
    return 0.5 * (S + S.transpose(0, 2, 1))


@pytest.mark.parametrize("dtype,p,path,tc", CASES)
def test_projection_and_vjp_match_oracle(dtype, p, path, tc):
    import torch
    import paper_2606_13825_b200 as cdu
    tdt = torch.float32 if dtype == "f32" else torch.float64
    rng = np.random.default_rng(p)
    cnt = 3
    S = _sym(rng, cnt, p)
    S = S.astype(np.float32).astype(np.float64) if dtype == "f32" else S
    Pi, U, lam = cdu.cdu_psd_project(torch.as_tensor(S, dtype=tdt, device="cuda"), path=path, use_tensor_cores=tc)
    Pi, U, lam = (t.double().cpu().numpy() for t in (Pi, U, lam))
    G = _sym(rng, cnt, p)
    G = G.astype(np.float32).astype(np.float64) if dtype == "f32" else G
    Sb = cdu.cdu_psd_vjp(torch.as_tensor(U, dtype=tdt, device="cuda"), torch.as_tensor(lam, dtype=tdt, device="cuda"),
                         torch.as_tensor(G, dtype=tdt, device="cuda"), path=path, use_tensor_cores=tc).double().cpu().numpy()
    tolp, tolv = (2e-5, 2e-4) if dtype == "f32" else (1e-12, 1e-11)
    for i in range(cnt):
        ref = C.smat(C.proj_psd(C.svec(S[i]))[0])
        n2 = np.linalg.norm(S[i], 2)
        assert np.abs(Pi[i] - ref).max() <= tolp * n2
        assert np.abs(U[i].T @ U[i] - np.eye(p)).max() <= (5e-6 if dtype == "f32" else 1e-13)
        lam_ref, U_ref = np.linalg.eigh(S[i])
        assert np.abs(np.sort(lam[i]) - lam_ref).max() <= tolp * n2
        vref = C.dk_vjp_matrix(U_ref, lam_ref, G[i])        # oracle's own eigendecomposition, not the GPU's
        assert np.abs(Sb[i] - vref).max() <= tolv * np.abs(vref).max()


@pytest.mark.parametrize("dtype,path", [("f64", 1), ("f32", 1), ("f64", 2)])
def test_repeated_and_zero_eigenvalues(dtype, path):
    """Exactly repeated eigenvalues {2,2,2,-1,-1,0.5} plus an exactly singular matrix: finite, correct."""
    import torch
    import paper_2606_13825_b200 as cdu
    tdt = torch.float32 if dtype == "f32" else torch.float64
    rng = np.random.default_rng(0)
    lam = np.array([2.0, 2.0, 2.0, -1.0, -1.0, 0.5, 0.0, 0.0])
    p = lam.size
    Q, _ = np.linalg.qr(rng.standard_normal((p, p)))
    S = (Q * lam) @ Q.T
    S = 0.5 * (S + S.T)
    if dtype == "f32":
        S = S.astype(np.float32).astype(np.float64)
    St = torch.as_tensor(np.stack([S, np.zeros_like(S), np.eye(p)]), dtype=tdt, device="cuda")
    Pi, U, l = cdu.cdu_psd_project(St, path=path)
    assert torch.isfinite(Pi).all() and torch.isfinite(U).all()
    tol = 5e-6 if dtype == "f32" else 1e-13
    ref = C.smat(C.proj_psd(C.svec(S))[0])
    assert np.abs(Pi[0].double().cpu().numpy() - ref).max() <= tol * 2
    assert torch.all(Pi[1] == 0) and torch.allclose(Pi[2], torch.eye(p, dtype=tdt, device="cuda"), atol=tol)
    G = rng.standard_normal((p, p)); G = 0.5 * (G + G.T)
    Gt = torch.as_tensor(np.stack([G, G, G]), dtype=tdt, device="cuda")
    Sb = cdu.cdu_psd_vjp(U, l, Gt, path=path)
    assert torch.isfinite(Sb).all()
    assert torch.allclose(Sb[2], Gt[2], atol=tol * 10)             # S > 0: the VJP is the identity
    assert torch.all(Sb[1] == 0)                                   # S = 0: f'(0) := 0 (reading A11)


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_dk_vjp_error_does_not_depend_on_the_eigenvalue_gap(dtype):
    """PAPER.md App. C / Fig. 4 left (L270-277): matrices of Eq. 13 at n = 40, gap delta from 1 down to 1e-10. The GPU's
    projection and DK VJP (its own eigendecomposition) against the oracle's (LAPACK eigh): the error, relative to the size
    of the matrix / of the cotangent, stays at rounding level for every delta."""
    import torch
    import paper_2606_13825_b200 as cdu
    import workloads as W
    tdt = torch.float32 if dtype == "f32" else torch.float64
    rng = np.random.default_rng(40)
    n, cnt = 40, 4
    tolp, tolv = (5e-6, 2e-4) if dtype == "f32" else (1e-13, 1e-11)
    for delta in (1.0, 1e-2, 1e-5, 1e-8, 1e-10):
        S = np.stack([W.clustered_spectrum_matrix(rng, n, delta) for _ in range(cnt)])
        G = _sym(rng, cnt, n)
        if dtype == "f32":
            S = S.astype(np.float32).astype(np.float64); G = G.astype(np.float32).astype(np.float64)
        Pi, U, lam = cdu.cdu_psd_project(torch.as_tensor(S, dtype=tdt, device="cuda"))
        Sb = cdu.cdu_psd_vjp(U, lam, torch.as_tensor(G, dtype=tdt, device="cuda")).double().cpu().numpy()
        assert np.isfinite(Sb).all()
        for i in range(cnt):
            ref = C.smat(C.proj_psd(C.svec(S[i]))[0])
            assert np.abs(Pi[i].double().cpu().numpy() - ref).max() <= tolp * delta, (delta, i)
            lam_ref, U_ref = np.linalg.eigh(S[i])
            vref = C.dk_vjp_matrix(U_ref, lam_ref, G[i])
            assert np.abs(Sb[i] - vref).max() <= tolv * np.abs(G[i]).max(), (delta, i, np.abs(Sb[i] - vref).max())

"""SURVEY.md 8(f) F2 on the GPU: cotangents on the intermediate iterates (cdu_backward_inject), the Eq. 12 training loss with
its reverse sweep (cdu_backward_eq12) and the App. E policy features (cdu_get_features, L321-339), each
against the oracle on the same seeded inputs."""
import numpy as np
import pytest

import workloads as W
from workloads.generators import Workload, _round_problem
import parity_util as PU
from oracle import cosmo_oracle as O
from test_parity_gpu import _mixed_workload

pytestmark = pytest.mark.gpu


def _run(wl, fn, ckpt=0, **opts):
    import torch
    import paper_2606_13825_b200 as cdu
    tdt = torch.float32 if wl.dtype == "f32" else torch.float64
    T = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=tdt, device="cuda")
    h = cdu.cdu_create(W.pack_batch(wl.problems, wl.dtype), K_max=wl.K, ckpt_mode=ckpt, **opts)
    B = wl.batch
    rho = np.repeat(wl.rho[:, None], B, 1).ravel(); alpha = np.repeat(wl.alpha[:, None], B, 1).ravel()
    h.forward(wl.K, T(rho), T(alpha), wl.sigma, T(np.concatenate(wl.x0)), T(np.concatenate(wl.s0)), T(np.concatenate(wl.y0)),
              rho_mode=cdu.CDU_RHO_PER_PROBLEM)
    out = fn(h, T)
    st = h.stats()
    h.close()
    return out, st


def _split(wl, v, kind):
    off = np.cumsum([0] + [pr.n if kind == "n" else pr.m for pr in wl.problems])
    return [v[off[i]:off[i + 1]] for i in range(wl.batch)]


def _grads_np(wl, g):
    npy = lambda t: t.detach().cpu().numpy().astype(np.float64)
    return dict(g_rho=npy(g["g_rho"]).reshape(wl.K, wl.batch), g_alpha=npy(g["g_alpha"]).reshape(wl.K, wl.batch), g_sigma=npy(g["g_sigma"]),
                g_x0=_split(wl, npy(g["g_x0"]), "n"), g_s0=_split(wl, npy(g["g_s0"]), "m"), g_y0=_split(wl, npy(g["g_y0"]), "m"))


def _compare(wl, refs, got, tol):
    for b, g in enumerate(refs):
        gfb = max(np.max(np.abs(v), initial=0.0) for v in (g.g_x0, g.g_s0, g.g_y0)) or 1.0
        for k, ref in (("g_x0", g.g_x0), ("g_s0", g.g_s0), ("g_y0", g.g_y0)):
            assert PU.nrm_err(got[k][b], ref, gfb) <= tol, (b, k)
        assert PU.nrm_err(got["g_rho"][:, b], g.g_rho_scalar) <= tol, (b, "g_rho")
        assert PU.nrm_err(got["g_alpha"][:, b], g.g_alpha) <= tol, (b, "g_alpha")
    assert PU.nrm_err(got["g_sigma"], [g.g_sigma for g in refs]) <= tol


@pytest.mark.parametrize("dtype,ckpt", [("f64", 0), ("f64", 1), ("f32", 0)])
def test_injected_cotangents_match_oracle(dtype, ckpt):
    wl = _mixed_workload(dtype, seed=21, B=3, K=6) if dtype == "f64" else W.make_config(2, batch=3, p=12, K=8)
    rng = np.random.default_rng(5)
    rd = lambda a: PU.round_to(a, wl.dtype)
    K, N, M = wl.K, sum(p.n for p in wl.problems), sum(p.m for p in wl.problems)
    ix, is_, iy = rd(rng.standard_normal((K - 1, N))), rd(rng.standard_normal((K - 1, M))), rd(rng.standard_normal((K - 1, M)))
    tx, ts, ty = rd(rng.standard_normal(N)), rd(rng.standard_normal(M)), rd(rng.standard_normal(M))
    refs = []
    for b, pr in enumerate(wl.problems):
        un = O.unroll(pr, K, wl.rho, wl.alpha, wl.sigma, wl.x0[b], wl.s0[b], wl.y0[b])
        inj = {k: (_split(wl, ix[k - 1], "n")[b], _split(wl, is_[k - 1], "m")[b], _split(wl, iy[k - 1], "m")[b]) for k in range(1, K)}
        refs.append(O.backward(pr, un, _split(wl, tx, "n")[b], _split(wl, ts, "m")[b], _split(wl, ty, "m")[b], inject=inj))
    g, st = _run(wl, lambda h, T: h.backward_inject(T(tx), T(ts), T(ty), T(ix), T(is_), T(iy)), ckpt=ckpt)
    _compare(wl, refs, _grads_np(wl, g), PU.TOL[wl.dtype]["grad"])
    assert st["flags_or"] == 0


@pytest.mark.parametrize("which", ["mixed-f64", "mixed-f64-lean", "maxcut-f32", "socp-f32"])
def test_eq12_loss_and_gradients_match_oracle(which):
    if which.startswith("mixed"):
        wl = _mixed_workload("f64", seed=22, B=3, K=7)
    elif which == "maxcut-f32":
        wl = W.make_config(2, batch=3, p=12, K=10)
    else:
        wl = W.make_config(3, batch=3, p=30, K=10)
    refs, losses = [], []
    for b, pr in enumerate(wl.problems):
        un = O.unroll(pr, wl.K, wl.rho, wl.alpha, wl.sigma, wl.x0[b], wl.s0[b], wl.y0[b])
        refs.append(O.backward_eq12(pr, un)); losses.append(O.eq12_loss(pr, un))
    (loss, g), st = _run(wl, lambda h, T: h.backward_eq12(), ckpt=1 if which.endswith("lean") else 0)
    tol = PU.TOL[wl.dtype]
    assert PU.nrm_err(loss.double().cpu().numpy(), losses) <= tol["iter"] * 10
    _compare(wl, refs, _grads_np(wl, g), tol["grad"])


def test_features_match_oracle():
    wl = _mixed_workload("f64", seed=23, B=3, K=5)
    uns = [O.unroll(pr, wl.K, wl.rho, wl.alpha, wl.sigma, wl.x0[b], wl.s0[b], wl.y0[b]) for b, pr in enumerate(wl.problems)]
    for k in (0, 1, wl.K):
        f, _ = _run(wl, lambda h, T: h.features(k))
        npy = lambda t: t.double().cpu().numpy()
        for b, pr in enumerate(wl.problems):
            ref = O.features(pr, uns[b], k)
            assert np.allclose(_split(wl, npy(f["rp_bar"]), "m")[b], ref["rp_bar"], atol=1e-9)
            assert np.allclose(_split(wl, npy(f["rd_bar"]), "n")[b], ref["rd_bar"], atol=1e-9)
            assert np.allclose(_split(wl, npy(f["delta_d"]), "m")[b], ref["delta_d"], atol=1e-9)
            assert np.allclose(_split(wl, npy(f["delta_p"]), "m")[b], ref["delta_p"], atol=1e-9)
            assert np.allclose(npy(f["scal"])[b], ref["scal"], atol=1e-7)

"""CDU_RHO_PER_ROW: one penalty per constraint row, D = diag(rho) in M = P + sigma I + A'DA (Eq. 4
L78), Eq. 6 (L90) row by row, rectified over SOC / PSD blocks (App. E). GPU against the oracle (which takes a vector rho)."""
import numpy as np
import pytest

import workloads as W
from workloads.generators import ZERO, NONNEG, SOC, PSD, cone_rows
import parity_util as PU
from oracle import cosmo_oracle as O
from test_parity_gpu import _mixed_workload

pytestmark = pytest.mark.gpu


def _rectify_np(pr, rho):
    out = rho.copy(); r = 0
    for kind, dim in pr.cones:
        n = cone_rows(kind, dim)
        if kind in (SOC, PSD):
            out[..., r:r + n] = out[..., r:r + n].mean(axis=-1, keepdims=True)
        r += n
    return out


def _run(wl, rho_rows, ckpt, **opts):
    """rho_rows: list over problems of [K, m_b]. Returns GPU results split per problem."""
    import torch
    import paper_2606_13825_b200 as cdu
    tdt = torch.float32 if wl.dtype == "f32" else torch.float64
    T = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=tdt, device="cuda")
    h = cdu.cdu_create(W.pack_batch(wl.problems, wl.dtype), K_max=wl.K, ckpt_mode=ckpt, **opts)
    B, K = wl.batch, wl.K
    rho = T(np.concatenate(rho_rows, axis=1))                       # [K, M]
    alpha = T(np.repeat(wl.alpha[:, None], B, 1))
    xK, sK, yK = h.forward(K, rho.reshape(-1), alpha.reshape(-1), wl.sigma, T(np.concatenate(wl.x0)), T(np.concatenate(wl.s0)),
                           T(np.concatenate(wl.y0)), rho_mode=cdu.CDU_RHO_PER_ROW)
    rng = np.random.default_rng(9)
    cots = [tuple(PU.round_to(rng.standard_normal(k), wl.dtype) for k in (p.n, p.m, p.m)) for p in wl.problems]
    g = h.backward(T(np.concatenate([c[0] for c in cots])), T(np.concatenate([c[1] for c in cots])), T(np.concatenate([c[2] for c in cots])))
    st = h.stats()
    npy = lambda t: t.double().cpu().numpy()
    on = np.cumsum([0] + [p.n for p in wl.problems]); om = np.cumsum([0] + [p.m for p in wl.problems])
    res = dict(x=[npy(xK)[on[b]:on[b + 1]] for b in range(B)], s=[npy(sK)[om[b]:om[b + 1]] for b in range(B)],
               y=[npy(yK)[om[b]:om[b + 1]] for b in range(B)], g_rho=[npy(g["g_rho"]).reshape(K, -1)[:, om[b]:om[b + 1]] for b in range(B)],
               g_alpha=npy(g["g_alpha"]).reshape(K, B), g_sigma=npy(g["g_sigma"]),
               g_x0=[npy(g["g_x0"])[on[b]:on[b + 1]] for b in range(B)], g_s0=[npy(g["g_s0"])[om[b]:om[b + 1]] for b in range(B)],
               g_y0=[npy(g["g_y0"])[om[b]:om[b + 1]] for b in range(B)])
    h.close()
    return res, cots, st


CASES = [("mixed-f64", 0, {}), ("mixed-f64", 1, {}), ("maxcut-f32", 0, {}), ("maxcut-f32-large-path", 1, dict(psd_small_max=8)),
         ("maxcut-f32-pcg", 0, dict(no_diag_path=1)), ("lovasz-f32", 0, {}), ("socp-f32", 0, {})]


@pytest.mark.parametrize("which,ckpt,opts", CASES)
def test_per_row_rho_matches_oracle(which, ckpt, opts):
    if which.startswith("mixed"):
        wl = _mixed_workload("f64", seed=31, B=3, K=6)
    elif which.startswith("maxcut"):
        wl = W.make_config(2, batch=3, p=12, K=8)
    elif which.startswith("lovasz"):
        wl = W.make_config(4, batch=2, p=10, K=8)
    else:
        wl = W.make_config(3, batch=3, p=30, K=8)
    rng = np.random.default_rng(4)
    base = wl.rho[:, None]
    rho_rows = [PU.round_to(_rectify_np(pr, base * np.exp(rng.uniform(-0.7, 0.7, (wl.K, pr.m)))), wl.dtype) for pr in wl.problems]
    rho_rows = [_rectify_np(pr, r) for pr, r in zip(wl.problems, rho_rows)]       # exactly constant inside the blocks after rounding
    res, cots, st = _run(wl, rho_rows, ckpt, **opts)
    tol = PU.TOL[wl.dtype]
    for b, pr in enumerate(wl.problems):
        un = O.unroll(pr, wl.K, rho_rows[b], wl.alpha, wl.sigma, wl.x0[b], wl.s0[b], wl.y0[b])
        g = O.backward(pr, un, *cots[b])
        fb = max(np.abs(un.xs[-1]).max(), np.abs(un.ys[-1]).max(), 1e-300)
        for k, ref in (("x", un.xs[-1]), ("s", un.ss[-1]), ("y", un.ys[-1])):
            assert PU.nrm_err(res[k][b], ref, fb) <= tol["iter"], (which, b, k)
        gfb = max(np.abs(v).max() for v in (g.g_x0, g.g_s0, g.g_y0)) or 1.0
        for k, ref in (("g_x0", g.g_x0), ("g_s0", g.g_s0), ("g_y0", g.g_y0)):
            assert PU.nrm_err(res[k][b], ref, gfb) <= tol["grad"], (which, b, k)
        assert PU.nrm_err(res["g_rho"][b], g.g_rho) <= tol["grad"], (which, b, "g_rho", PU.nrm_err(res["g_rho"][b], g.g_rho))
        assert PU.nrm_err(res["g_alpha"][:, b], g.g_alpha) <= tol["grad"], (which, b, "g_alpha")
    assert st["flags_or"] == 0


def test_rectify_is_the_block_mean_and_scalar_rows_equal_per_problem_mode():
    import torch
    import paper_2606_13825_b200 as cdu
    wl = _mixed_workload("f64", seed=32, B=2, K=4)
    h = cdu.cdu_create(W.pack_batch(wl.problems, "f64"), K_max=wl.K)
    rng = np.random.default_rng(1)
    M = sum(p.m for p in wl.problems)
    raw = np.exp(rng.uniform(-1, 1, (wl.K, M)))
    got = h.rectify_rho(wl.K, torch.as_tensor(raw, device="cuda").clone().reshape(-1)).cpu().numpy().reshape(wl.K, M)
    om = np.cumsum([0] + [p.m for p in wl.problems])
    want = np.concatenate([_rectify_np(p, raw[:, om[b]:om[b + 1]]) for b, p in enumerate(wl.problems)], axis=1)
    assert np.allclose(got, want, rtol=1e-14)
    h.close()
    # a per-row rho that is the same number on every row reproduces the per-problem mode (iterates to rounding, g_rho by row sums)
    rows = [np.repeat(wl.rho[:, None], p.m, 1) for p in wl.problems]
    res, cots, _ = _run(wl, rows, 0)
    ref = PU.gpu_run(wl, cots, per_problem=True)
    for b in range(wl.batch):
        assert PU.nrm_err(res["x"][b], ref["xK"][b]) <= 1e-12 and PU.nrm_err(res["y"][b], ref["yK"][b]) <= 1e-12
        assert PU.nrm_err(res["g_rho"][b].sum(1), ref["g_rho"][:, b]) <= 1e-12

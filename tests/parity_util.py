"""Shared helpers of the GPU parity tests: run a Workload through the C ABI and through the oracle and
compare norm-wise (reading A10). The oracle is imported here (tests only)."""
from __future__ import annotations

import numpy as np

import workloads as W
from oracle import cosmo_oracle as O

TOL = {"f64": dict(iter=1e-9, grad=1e-7), "f32": dict(iter=1e-4, grad=1e-3)}   # BASELINE.json north_star


def round_to(a, dtype):
    a = np.asarray(a, np.float64)
    return a.astype(np.float32).astype(np.float64) if dtype == "f32" else a


def nrm_err(a, ref, fallback_scale=None):
    """||a-ref||_inf / ||ref||_inf; identically-zero references are compared against `fallback_scale`."""
    a = np.asarray(a, np.float64).ravel(); ref = np.asarray(ref, np.float64).ravel()
    if ref.size == 0:
        return 0.0
    sc = np.max(np.abs(ref))
    if sc == 0.0:
        sc = fallback_scale if fallback_scale else 1.0
    return float(np.max(np.abs(a - ref)) / sc)


def oracle_reference(wl, problems=None, x_star=None):
    """Oracle forward, terminal cotangent of the A13 loss (fp64, from the oracle's z_K, rounded to the GPU dtype
    so both sides read identical numbers), oracle backward with that cotangent."""
    idx = list(range(wl.batch)) if problems is None else list(problems)
    ref = dict(idx=idx, xK=[], sK=[], yK=[], cot=[], g_x0=[], g_s0=[], g_y0=[], g_rho=[], g_alpha=[], g_sigma=[])
    for b in idx:
        pr = wl.problems[b]
        un = O.unroll(pr, wl.K, wl.rho, wl.alpha, wl.sigma, wl.x0[b], wl.s0[b], wl.y0[b])
        xK, sK, yK = un.xs[-1], un.ss[-1], un.ys[-1]
        xs = np.zeros(pr.n) if x_star is None else x_star[b]
        cot = tuple(round_to(c, wl.dtype) for c in O.terminal_loss_grad(pr, xK, sK, yK, xs))
        g = O.backward(pr, un, *cot)
        ref["xK"].append(xK); ref["sK"].append(sK); ref["yK"].append(yK); ref["cot"].append(cot)
        ref["g_x0"].append(g.g_x0); ref["g_s0"].append(g.g_s0); ref["g_y0"].append(g.g_y0)
        ref["g_rho"].append(g.g_rho_scalar); ref["g_alpha"].append(g.g_alpha); ref["g_sigma"].append(g.g_sigma)
    return ref


def gpu_run(wl, cot_full, ckpt_mode=0, per_problem=False, host=False, keep_iterates_of=None, **opts):
    """Forward + backward through the C ABI. cot_full: list over the WHOLE batch of (gx, gs, gy) or None (zeros).
    Returns numpy results split per problem."""
    import torch
    import paper_2606_13825_b200 as cdu

    packed = W.pack_batch(wl.problems, wl.dtype)
    h = cdu.cdu_create(packed, K_max=wl.K, ckpt_mode=ckpt_mode, **opts)
    tdt = torch.float32 if wl.dtype == "f32" else torch.float64
    dev = "cpu" if host else "cuda"

    def T(a):
        t = torch.as_tensor(np.ascontiguousarray(a), dtype=tdt)
        return t.pin_memory() if host else t.to(dev)

    B = wl.batch
    rho, alpha = wl.rho, wl.alpha
    mode = cdu.CDU_RHO_PER_ITER
    if per_problem:
        rho = np.repeat(wl.rho[:, None], B, 1).ravel(); alpha = np.repeat(wl.alpha[:, None], B, 1).ravel()
        mode = cdu.CDU_RHO_PER_PROBLEM
    cat = lambda xs: np.concatenate(xs) if len(xs) else np.zeros(0)
    xK, sK, yK = cdu.cdu_forward(h, wl.K, T(rho), T(alpha), wl.sigma, T(cat(wl.x0)), T(cat(wl.s0)), T(cat(wl.y0)),
                                 rho_mode=mode, host=host)
    if cot_full is None:
        g = cdu.cdu_backward(h, host=host)
    else:
        g = cdu.cdu_backward(h, T(cat([c[0] for c in cot_full])), T(cat([c[1] for c in cot_full])),
                             T(cat([c[2] for c in cot_full])), host=host)
    if not host:
        torch.cuda.synchronize()
    st = cdu.cdu_get_stats(h)
    vo, ro = packed["var_off"], packed["row_off"]
    npy = lambda t: t.detach().cpu().numpy().astype(np.float64)
    split = lambda v, off: [v[off[i]:off[i + 1]] for i in range(B)]
    res = dict(xK=split(npy(xK), vo), sK=split(npy(sK), ro), yK=split(npy(yK), ro),
               g_x0=split(npy(g["g_x0"]), vo), g_s0=split(npy(g["g_s0"]), ro), g_y0=split(npy(g["g_y0"]), ro),
               stats=st)
    if per_problem:
        res["g_rho"] = npy(g["g_rho"]).reshape(wl.K, B); res["g_alpha"] = npy(g["g_alpha"]).reshape(wl.K, B)
        res["g_sigma"] = npy(g["g_sigma"])
    else:
        res["g_rho"] = npy(g["g_rho"]); res["g_alpha"] = npy(g["g_alpha"]); res["g_sigma"] = float(npy(g["g_sigma"])[0])
    if keep_iterates_of is not None:      # callable(res) -> problems whose iterates z^0..z^K are wanted
        want = list(keep_iterates_of(res))
        its = {b: [] for b in want}
        for k in range(wl.K + 1):
            xs, ss, ys = (split(npy(t), o) for t, o in zip(h.iterate(k), (vo, ro, ro)))
            for b in want:
                its[b].append((xs[b], ss[b], ys[b]))
        res["iterates"] = its
    cdu.cdu_destroy(h)
    return res


def compare(wl, ref, res, per_problem):
    """Max norm-wise errors over the compared problems. Returns dict of errors."""
    e = dict(x=0.0, s=0.0, y=0.0, g_x0=0.0, g_s0=0.0, g_y0=0.0)
    for j, b in enumerate(ref["idx"]):
        fb = max(np.max(np.abs(ref["xK"][j]), initial=0.0), np.max(np.abs(ref["yK"][j]), initial=0.0), 1e-300)
        e["x"] = max(e["x"], nrm_err(res["xK"][b], ref["xK"][j], fb))
        e["s"] = max(e["s"], nrm_err(res["sK"][b], ref["sK"][j], fb))
        e["y"] = max(e["y"], nrm_err(res["yK"][b], ref["yK"][j], fb))
        gfb = max(np.max(np.abs(ref[k][j]), initial=0.0) for k in ("g_x0", "g_s0", "g_y0")) or 1.0
        for k in ("g_x0", "g_s0", "g_y0"):
            e[k] = max(e[k], nrm_err(res[k][b], ref[k][j], gfb))
    if per_problem:
        e["g_rho"] = max(nrm_err(res["g_rho"][:, b], ref["g_rho"][j]) for j, b in enumerate(ref["idx"]))
        e["g_alpha"] = max(nrm_err(res["g_alpha"][:, b], ref["g_alpha"][j]) for j, b in enumerate(ref["idx"]))
        # g_sigma has one entry per problem in this layout: compared norm-wise as that vector (reading A10), like
        # every other output. One entry alone is a sum of K signed terms and can cancel to a fraction of their size.
        e["g_sigma"] = nrm_err([res["g_sigma"][b] for b in ref["idx"]], ref["g_sigma"])
    else:
        assert len(ref["idx"]) == wl.batch
        e["g_rho"] = nrm_err(res["g_rho"], np.sum(ref["g_rho"], axis=0))
        e["g_alpha"] = nrm_err(res["g_alpha"], np.sum(ref["g_alpha"], axis=0))
        e["g_sigma"] = nrm_err([res["g_sigma"]], [np.sum(ref["g_sigma"])])
    return e


def compare_each(wl, ref, res, per_problem=True):
    """compare() problem by problem: list of error dicts in the order of ref['idx']."""
    out = []
    for j, b in enumerate(ref["idx"]):
        one = {k: ([v[j]] if isinstance(v, list) else v) for k, v in ref.items()}
        one["idx"] = [b]
        out.append(compare(wl, one, res, per_problem))
    return out


def teacher_forced_errors(wl, b, gpu_iterates, cot, res):
    """Gradient errors of problem b against the oracle's reverse sweep ALONG THE GPU's OWN ITERATES: the tape of step k is the
    oracle's exact step evaluated at the GPU's z^k (its outputs are discarded). This is the derivative of the trajectory the
    forward pass actually took, which is what BPTT computes; it separates the parity of the reverse sweep from branch
    decisions of the forward pass at near-zero eigenvalues. gpu_iterates: list over k = 0..K of
    (x, s, y) of problem b."""
    pr = wl.problems[b]
    tapes = []
    for k in range(wl.K):
        x, s, y = gpu_iterates[k]
        tapes.append(O.step(pr, x, s, y, wl.rho[k], wl.alpha[k], wl.sigma)[3])
    un = O.Unroll([z[0] for z in gpu_iterates], [z[1] for z in gpu_iterates], [z[2] for z in gpu_iterates], tapes)
    g = O.backward(pr, un, *cot)
    gfb = max(np.max(np.abs(v), initial=0.0) for v in (g.g_x0, g.g_s0, g.g_y0)) or 1.0
    e = dict(g_x0=nrm_err(res["g_x0"][b], g.g_x0, gfb), g_s0=nrm_err(res["g_s0"][b], g.g_s0, gfb), g_y0=nrm_err(res["g_y0"][b], g.g_y0, gfb),
             g_rho=nrm_err(res["g_rho"][:, b], g.g_rho_scalar), g_alpha=nrm_err(res["g_alpha"][:, b], g.g_alpha))
    return e


def full_cotangent(wl, ref, fill_seed=None):
    """Cotangent list for the whole batch: the oracle's for compared problems; elsewhere zeros, or (fill_seed given)
    seeded N(0,1) scaled to the compared problems' cotangents, so that the backward of EVERY problem does real work."""
    cots = [(np.zeros(pr.n), np.zeros(pr.m), np.zeros(pr.m)) for pr in wl.problems]
    if fill_seed is not None:
        rng = np.random.default_rng(fill_seed)
        sc = max([float(np.max(np.abs(c))) for cot in ref["cot"] for c in cot if c.size] + [1e-30])
        cots = [tuple(round_to(sc * rng.standard_normal(k), wl.dtype) for k in (pr.n, pr.m, pr.m)) for pr in wl.problems]
    for j, b in enumerate(ref["idx"]):
        cots[b] = ref["cot"][j]
    return cots


def assert_batch_sane(wl, res, rel_tol):
    """Every problem of the batch (not only the ones compared with the oracle): all outputs finite and s_K inside its
    cone (oracle.cones.in_cone) up to rel_tol x the scale of the iterate."""
    from oracle import cones as C
    for k in ("xK", "sK", "yK", "g_x0", "g_s0", "g_y0"):
        for b, v in enumerate(res[k]):
            assert np.all(np.isfinite(v)), f"{k} of problem {b} is not finite"
    for k in ("g_rho", "g_alpha", "g_sigma"):
        assert np.all(np.isfinite(res[k])), k
    for b, pr in enumerate(wl.problems):
        s = res["sK"][b]
        sc = max(float(np.max(np.abs(s), initial=0.0)), float(np.max(np.abs(res["xK"][b]), initial=0.0)), 1e-30)
        r = 0
        for kind, dim in pr.cones:
            rows = W.cone_rows(kind, dim)
            assert C.in_cone(kind, dim, s[r:r + rows], tol=rel_tol * sc), f"s_K of problem {b} leaves cone ({kind},{dim})"
            r += rows


def check(wl, problems=None, per_problem=None, x_star=None, ckpt_mode=0, host=False, tol_scale=1.0, fill_seed=None,
          sane_tol=None, **opts):
    """Oracle vs GPU on `problems` (default: all). Returns (errors, stats). fill_seed: random cotangents on the problems
    that are not compared (needs per-problem hyper-parameters); sane_tol: also run assert_batch_sane on the whole batch."""
    ref = oracle_reference(wl, problems, x_star)
    if per_problem is None:
        per_problem = problems is not None and len(list(problems)) != wl.batch
    assert fill_seed is None or per_problem
    res = gpu_run(wl, full_cotangent(wl, ref, fill_seed), ckpt_mode=ckpt_mode, per_problem=per_problem, host=host, **opts)
    if sane_tol is not None:
        assert_batch_sane(wl, res, sane_tol)
    e = compare(wl, ref, res, per_problem)
    return e, res["stats"]


def assert_within(e, dtype, tol_scale=1.0, skip=()):
    t = TOL[dtype]
    bad = {}
    for k, v in e.items():
        if k in skip:
            continue
        lim = (t["iter"] if k in ("x", "s", "y") else t["grad"]) * tol_scale
        if not (v <= lim):
            bad[k] = (v, lim)
    assert not bad, f"parity failures (value, limit): {bad}; all errors: {e}"

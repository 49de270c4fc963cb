"""Pins for oracle/cosmo_oracle.py: closed forms, identities, textbook special cases, finite differences."""
import os

import numpy as np
import pytest
import scipy.sparse as sp

import workloads as W
from workloads.generators import complete_graph, cycle_graph, ZERO, NONNEG, SOC, PSD, Problem
from oracle import cosmo_oracle as O
from oracle import cones as C
from oracle.fd import central_diff_grad, nrm_rel_err


def _golden_rows(golden_dir):
    with open(os.path.join(golden_dir, "closed_forms.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                prob, graph, n, val = line.split()
                yield prob, graph, int(n), float(val)


def _graph(kind, n):
    return {"complete": complete_graph(n), "cycle": cycle_graph(n), "empty": np.zeros((n, n))}[kind]


# ---- closed-form optima pin builders + the whole forward fixed point ----------------------------
def test_closed_form_optima(golden_dir):
    for prob, graph, n, val in _golden_rows(golden_dir):
        Wm = _graph(graph, n)
        pr = W.maxcut_problem(Wm) if prob == "maxcut" else W.lovasz_problem(Wm)
        x, s, y = O.solve_to_convergence(pr, iters=3000, rho=1.0, alpha=1.6)
        rp, rd = O.residuals(pr, x, s, y)
        assert abs(-pr.q @ x - val) < 1e-7, (prob, graph, n, -pr.q @ x)
        assert np.abs(rp).max() < 1e-8 and np.abs(rd).max() < 1e-8
        # s in K, y in K* (sign convention A1), complementary
        o = 0
        for kind, dim in pr.cones:
            r = C.cone_rows(kind, dim)
            assert C.in_cone(kind, dim, s[o:o + r], 1e-7) and C.in_dual_cone(kind, dim, y[o:o + r], 1e-7)
            o += r
        assert abs(s @ y) < 1e-6


def test_equality_only_qp_matches_kkt_solve():
    """K = zero cone: the fixed point is the KKT solution of min 1/2 x'Px+q'x s.t. Ax=b (textbook)."""
    rng = np.random.default_rng(1)
    n, m = 8, 3
    G = rng.standard_normal((n, n))
    P = G.T @ G + 0.1 * np.eye(n)
    A = rng.standard_normal((m, n))
    q, b = rng.standard_normal(n), rng.standard_normal(m)
    pr = Problem(P=sp.csr_matrix(P), q=q, A=sp.csr_matrix(A), b=b, cones=[(ZERO, m)])
    x, s, y = O.solve_to_convergence(pr, iters=4000, rho=1.0, alpha=1.6)
    kkt = np.linalg.solve(np.block([[P, A.T], [A, np.zeros((m, m))]]), np.concatenate([-q, b]))
    np.testing.assert_allclose(x, kkt[:n], atol=1e-8)
    np.testing.assert_allclose(y, kkt[n:], atol=1e-7)       # multiplier of Ax=b with r_d = Px+q+A'y
    assert np.abs(s).max() == 0.0


def test_nonneg_qp_kkt_conditions():
    rng = np.random.default_rng(2)
    n, m = 6, 9
    G = rng.standard_normal((n, n))
    pr = Problem(P=sp.csr_matrix(G.T @ G + np.eye(n)), q=rng.standard_normal(n),
                 A=sp.csr_matrix(rng.standard_normal((m, n))), b=rng.standard_normal(m) + 1.0, cones=[(NONNEG, m)])
    x, s, y = O.solve_to_convergence(pr, iters=4000)
    rp, rd = O.residuals(pr, x, s, y)
    assert np.abs(rp).max() < 1e-8 and np.abs(rd).max() < 1e-8
    assert s.min() >= 0 and y.min() >= -1e-9 and abs(s @ y) < 1e-8


# ---- Eq. 3a <=> Eq. 4, and the sign convention ---------------------------------------------------
def test_paper_literal_saddle_point_step_is_equivalent():
    rng = np.random.default_rng(3)
    pr = W.random_mixed_problem(rng)
    x, s, y = rng.standard_normal(pr.n), rng.standard_normal(pr.m), rng.standard_normal(pr.m)
    xl, sl, yl = x.copy(), s.copy(), -y.copy()          # paper's y = -ours
    for k in range(5):
        rho, alpha = float(np.exp(rng.uniform(-2, 2))), float(rng.uniform(0.5, 1.9))
        x, s, y, tape = O.step(pr, x, s, y, rho, alpha, 1e-6)
        xl, sl, yl, xt, nu, st = O.step_paper_literal(pr, xl, sl, yl, rho, alpha, 1e-6)
        np.testing.assert_allclose(xt, tape.xt, rtol=1e-9, atol=1e-9)      # Eq. 3a == Eq. 4
        np.testing.assert_allclose(st, tape.st, rtol=1e-9, atol=1e-9)      # Eq. 3b == b - A xt
        np.testing.assert_allclose(xl, x, rtol=1e-9, atol=1e-9)
        np.testing.assert_allclose(sl, s, rtol=1e-9, atol=1e-9)
        np.testing.assert_allclose(yl, -y, rtol=1e-9, atol=1e-9)


def test_dense_and_sparse_solvers_agree(monkeypatch):
    rng = np.random.default_rng(4)
    pr = W.lovasz_problem(W.erdos_renyi(rng, 12, 0.3))
    rho, al = [0.7, 2.0, 0.3], [1.6, 1.2, 1.8]
    a = O.unroll(pr, 3, rho, al, 1e-6)
    monkeypatch.setattr(O, "DENSE_MAX", 0)
    b = O.unroll(pr, 3, rho, al, 1e-6)
    for u, v in zip(a.xs + a.ss + a.ys, b.xs + b.ss + b.ys):
        np.testing.assert_allclose(u, v, atol=1e-11)


def test_zero_row_padding_is_inert():
    rng = np.random.default_rng(5)
    pr = W.random_mixed_problem(rng)
    pad = 3
    A2 = sp.vstack([pr.A, sp.csr_matrix((pad, pr.n))], format="csr")
    pr2 = Problem(P=pr.P, q=pr.q, A=A2, b=np.concatenate([pr.b, np.zeros(pad)]), cones=pr.cones + [(ZERO, pad)])
    rho, al = [0.5, 3.0, 1.0, 0.2], [1.6, 1.0, 1.9, 1.4]
    y0 = rng.standard_normal(pr.m)
    a = O.unroll(pr, 4, rho, al, 1e-6, y0=y0)
    b = O.unroll(pr2, 4, rho, al, 1e-6, y0=np.concatenate([y0, [0.3, -0.2, 0.1]]))
    np.testing.assert_allclose(b.xs[-1], a.xs[-1], atol=1e-12)
    np.testing.assert_allclose(b.ss[-1][:pr.m], a.ss[-1], atol=1e-12)
    np.testing.assert_allclose(b.ys[-1][:pr.m], a.ys[-1], atol=1e-12)
    np.testing.assert_allclose(b.ys[-1][pr.m:], [0.3, -0.2, 0.1], atol=1e-12)


# ---- Eq. 6 against the explicit middle expression of Eq. 5 ---------------------------------------
def test_eq6_matches_explicit_implicit_differentiation():
    rng = np.random.default_rng(6)
    n, m = 6, 9
    G = rng.standard_normal((n, n))
    P = G.T @ G / n
    A = rng.standard_normal((m, n)) * (rng.random((m, n)) < 0.7)
    rho = rng.uniform(0.1, 2.0, m)
    sigma = 1e-3
    xi, g = rng.standard_normal(n), rng.standard_normal(n)
    M = P + sigma * np.eye(n) + A.T @ (rho[:, None] * A)
    xt = np.linalg.solve(M, xi)
    explicit = np.array([-g @ np.linalg.solve(M, np.outer(A[i], A[i]) @ xt) for i in range(m)])   # Eq. 5
    lam = np.linalg.solve(M, g)
    np.testing.assert_allclose(-(A @ lam) * (A @ xt), explicit, rtol=1e-10, atol=1e-12)           # Eq. 6
    # and against central differences of L(rho) = g' M(rho)^-1 xi
    L = lambda r: g @ np.linalg.solve(P + sigma * np.eye(n) + A.T @ (r[:, None] * A), xi)
    np.testing.assert_allclose(central_diff_grad(L, rho, 1e-6), explicit, rtol=1e-6, atol=1e-8)


# ---- whole backward vs central differences ------------------------------------------------------
def _loss_setup(seed, cones, n=7, K=5, with_P=True):
    rng = np.random.default_rng(seed)
    pr = W.random_mixed_problem(rng, n=n, cones=cones, with_P=with_P)
    rho = np.exp(rng.uniform(np.log(0.2), np.log(3.0), K))
    alpha = rng.uniform(0.8, 1.8, K)
    sigma = 1e-2
    z0 = (0.3 * rng.standard_normal(pr.n), 0.3 * rng.standard_normal(pr.m), 0.3 * rng.standard_normal(pr.m))
    cx, cs, cy = rng.standard_normal(pr.n), rng.standard_normal(pr.m), rng.standard_normal(pr.m)
    xs = rng.standard_normal(pr.n)

    def loss(rho_, alpha_, sigma_, z0_):
        un = O.unroll(pr, K, rho_, alpha_, sigma_, *z0_, keep_tape=False)
        x, s, y = un.xs[-1], un.ss[-1], un.ys[-1]
        return cx @ x + cs @ s + cy @ y + O.terminal_loss(pr, x, s, y, xs)

    un = O.unroll(pr, K, rho, alpha, sigma, *z0)
    x, s, y = un.xs[-1], un.ss[-1], un.ys[-1]
    gx, gs, gy = O.terminal_loss_grad(pr, x, s, y, xs)
    g = O.backward(pr, un, gx + cx, gs + cs, gy + cy)
    return pr, rho, alpha, sigma, z0, loss, g


@pytest.mark.parametrize("seed,cones", [
    (21, ((ZERO, 2), (NONNEG, 3), (SOC, 4), (PSD, 3))),
    (22, ((PSD, 4), (SOC, 3), (NONNEG, 2))),
    (23, ((ZERO, 3), (PSD, 2), (PSD, 3))),
    (24, ((SOC, 5), (SOC, 2), (NONNEG, 4))),
])
def test_backward_matches_central_differences(seed, cones):
    pr, rho, alpha, sigma, z0, loss, g = _loss_setup(seed, cones)
    fd_lrho = central_diff_grad(lambda lr: loss(np.exp(lr), alpha, sigma, z0), np.log(rho), 1e-6, rel=False)
    assert nrm_rel_err(g.g_rho_scalar * rho, fd_lrho) < 2e-6
    fd_alpha = central_diff_grad(lambda a: loss(rho, a, sigma, z0), alpha, 1e-6, rel=False)
    assert nrm_rel_err(g.g_alpha, fd_alpha) < 2e-6
    fd_ls = central_diff_grad(lambda ls: loss(rho, alpha, float(np.exp(ls[0])), z0), np.array([np.log(sigma)]), 1e-4, rel=False)
    assert nrm_rel_err([g.g_sigma * sigma], fd_ls) < 5e-6
    for idx, name in enumerate(["g_x0", "g_s0", "g_y0"]):
        def f(v, idx=idx):
            z = list(z0); z[idx] = v
            return loss(rho, alpha, sigma, tuple(z))
        fd = central_diff_grad(f, z0[idx], 1e-6, rel=False)
        assert nrm_rel_err(getattr(g, name), fd) < 5e-6, name


def test_backward_per_row_rho_matches_central_differences():
    """Eq. 6 verbatim (vector rho in R^m, L72/L90) incl. the RHS terms the paper leaves to autograd (L82)."""
    rng = np.random.default_rng(31)
    cones = ((ZERO, 2), (NONNEG, 3))        # separable cones only: per-row rho is well defined (L343)
    pr = W.random_mixed_problem(rng, n=5, cones=cones)
    K = 3
    rho = rng.uniform(0.3, 2.0, (K, pr.m)); alpha = rng.uniform(1.0, 1.8, K); sigma = 1e-2
    c = rng.standard_normal(pr.n + 2 * pr.m)

    def loss(r):
        un = O.unroll(pr, K, r.reshape(K, pr.m), alpha, sigma, keep_tape=False)
        return c @ np.concatenate([un.xs[-1], un.ss[-1], un.ys[-1]])

    un = O.unroll(pr, K, rho, alpha, sigma)
    g = O.backward(pr, un, c[:pr.n], c[pr.n:pr.n + pr.m], c[pr.n + pr.m:])
    fd = central_diff_grad(loss, rho.ravel(), 1e-6, rel=False)
    assert nrm_rel_err(g.g_rho.ravel(), fd) < 2e-6


def test_backward_with_repeated_eigenvalues_is_finite():
    """Isotropic target S = c I makes all eigenvalues of the projected matrix coincide (L108)."""
    p = 4
    n = W.svec_dim(p)
    A = -sp.identity(n, format="csr")
    pr = Problem(P=sp.identity(n, format="csr"), q=-C.svec(2.0 * np.eye(p)), A=A, b=np.zeros(n), cones=[(PSD, p)])
    un = O.unroll(pr, 6, [1.0] * 6, [1.6] * 6, 1e-6)
    lam = un.tapes[-1].aux[0][0]
    assert np.ptp(lam) < 1e-12                                          # exactly degenerate spectrum
    g = O.backward(pr, un, np.ones(n), np.ones(n), np.ones(n))
    for v in (g.g_rho, g.g_alpha, g.g_x0, g.g_s0, g.g_y0):
        assert np.all(np.isfinite(v))
    fd = central_diff_grad(lambda a: np.sum([np.sum(v) for v in (lambda u: (u.xs[-1], u.ss[-1], u.ys[-1]))(
        O.unroll(pr, 6, [1.0] * 6, a, 1e-6, keep_tape=False))]), np.full(6, 1.6), 1e-6, rel=False)
    assert nrm_rel_err(g.g_alpha, fd) < 1e-5


def test_injected_cotangents_match_central_differences():
    rng = np.random.default_rng(41)
    pr = W.random_mixed_problem(rng)
    K = 4
    rho = rng.uniform(0.3, 2.0, K); alpha = rng.uniform(1.0, 1.8, K); sigma = 1e-2
    cs = [rng.standard_normal(pr.n + 2 * pr.m) for _ in range(K + 1)]

    def loss(a):
        un = O.unroll(pr, K, rho, a, sigma, keep_tape=False)
        return sum(cs[k] @ np.concatenate([un.xs[k], un.ss[k], un.ys[k]]) for k in range(1, K + 1))

    sp_ = lambda c: (c[:pr.n], c[pr.n:pr.n + pr.m], c[pr.n + pr.m:])
    un = O.unroll(pr, K, rho, alpha, sigma)
    g = O.backward(pr, un, *sp_(cs[K]), inject={k: sp_(cs[k]) for k in range(1, K)})
    assert nrm_rel_err(g.g_alpha, central_diff_grad(loss, alpha, 1e-6, rel=False)) < 2e-6


# ---- Eq. 12 loss and App. E features (L321-339) -----------------------------------------------------
def test_eq12_cotangents_and_total_gradient_match_central_differences():
    """(a) eq12_cotangents = dL/dz^k with L as a function of the iterates alone (denominators detached) by central
    differences on a few coordinates; (b) backward_eq12 = d eq12_loss / d(rho_k, alpha_k, x0) of the whole unroll by central
    differences, again with detached denominators (the loss is re-evaluated against the unperturbed z^0 residuals)."""
    from workloads import random_mixed_problem
    rng = np.random.default_rng(12)
    pr = random_mixed_problem(rng, n=7)
    K = 5
    rho = np.exp(rng.uniform(-1, 1, K)); alpha = rng.uniform(1.0, 1.8, K); sigma = 1e-6
    z0 = (0.3 * rng.standard_normal(pr.n), 0.3 * rng.standard_normal(pr.m), 0.3 * rng.standard_normal(pr.m))
    un = O.unroll(pr, K, rho, alpha, sigma, *z0)
    rp0, rd0 = O.residuals(pr, *z0)
    a0, b0 = rd0 @ rd0, rp0 @ rp0

    def loss_of_iterates(xs, ss, ys):            # denominators fixed at the unperturbed z^0
        L = 0.0
        for k in range(1, K + 1):
            rp, rd = O.residuals(pr, xs[k], ss[k], ys[k])
            L += np.log(rd @ rd / a0 + rp @ rp / b0)
        return L

    assert abs(loss_of_iterates(un.xs, un.ss, un.ys) - O.eq12_loss(pr, un)) < 1e-12
    cots = O.eq12_cotangents(pr, un)
    h = 1e-6
    for k in (1, 3, K):
        for part, vecs in enumerate((un.xs, un.ss, un.ys)):
            for i in (0, len(vecs[k]) - 1):
                def pert(d):
                    cp = [[v.copy() for v in un.xs], [v.copy() for v in un.ss], [v.copy() for v in un.ys]]
                    cp[part][k][i] += d
                    return loss_of_iterates(*cp)
                fd = (pert(h) - pert(-h)) / (2 * h)
                assert abs(fd - cots[k][part][i]) <= 1e-6 * max(1.0, abs(fd)), (k, part, i, fd, cots[k][part][i])
    g = O.backward_eq12(pr, un)

    def total(rho_, alpha_, x0_):
        u = O.unroll(pr, K, rho_, alpha_, sigma, x0_, z0[1], z0[2], keep_tape=False)
        return loss_of_iterates(u.xs, u.ss, u.ys)

    for k in (0, 2, K - 1):
        d = np.zeros(K); d[k] = 1e-6
        fd = (total(rho + d, alpha, z0[0]) - total(rho - d, alpha, z0[0])) / 2e-6
        assert abs(fd - g.g_rho_scalar[k]) <= 2e-5 * max(1.0, abs(fd)), (k, fd, g.g_rho_scalar[k])
        fd = (total(rho, alpha + d, z0[0]) - total(rho, alpha - d, z0[0])) / 2e-6
        assert abs(fd - g.g_alpha[k]) <= 2e-5 * max(1.0, abs(fd)), (k, fd, g.g_alpha[k])
    # x0 enters the loss only through the iterates (z^0's own residuals are detached and k starts at 1)
    d = np.zeros(pr.n); d[1] = 1e-6
    fd = (total(rho, alpha, z0[0] + d) - total(rho, alpha, z0[0] - d)) / 2e-6
    assert abs(fd - g.g_x0[1]) <= 2e-5 * max(1.0, abs(fd))


def test_features_hand_case():
    """App. E on a two-variable problem typed out by hand: A = I, P = 2 I, q = (1, -1), b = (0, 3)."""
    import scipy.sparse as sp
    from workloads.generators import Problem, NONNEG
    pr = Problem(P=sp.csr_matrix(2.0 * np.eye(2)), q=np.array([1.0, -1.0]), A=sp.csr_matrix(np.eye(2)), b=np.array([0.0, 3.0]),
                 cones=[(NONNEG, 2)], name="hand")
    un = O.unroll(pr, 2, np.array([1.0, 1.0]), np.array([1.0, 1.0]), 1e-6, np.array([1.0, 2.0]), np.array([0.5, 0.5]), np.array([0.0, 4.0]))
    f0 = O.features(pr, un, 0)
    # z^0: Ax = (1, 2), s = (.5, .5), b = (0, 3): r_p = (1.5, -0.5), scale 3; Px = (2, 4), q = (1, -1), A'y = (0, 4): r_d = (3, 7), scale 4
    assert np.allclose(f0["rp_bar"], [0.5, -1.0 / 6.0]) and np.allclose(f0["rd_bar"], [0.75, 1.75])
    f1 = O.features(pr, un, 1)
    assert np.allclose(f1["delta_d"], un.ss[1] - un.ss[0]) and np.allclose(f1["delta_p"], un.ss[1] - un.tapes[0].st)
    assert np.allclose(f1["scal"][2], np.log(np.abs(f1["delta_p"]).max() + 1e-12))


def test_lyapunov_lmi_closed_form():
    """PAPER.md App. F.2 (L422-428) with A = -a I: A'P + PA = -2aP <= -I and P >= I give P* = max(1, 1/(2a)) I, so the optimal
    value is n max(1, 1/(2a)). Pins the generator's svec map of P -> A'P + PA together with the oracle's two-PSD-block step."""
    from workloads import lyapunov_lmi_problem
    n = 4
    for a, val in ((0.25, 2.0 * n), (2.0, 1.0 * n)):
        pr = lyapunov_lmi_problem(np.random.default_rng(0), n=n, A_sys=-a * np.eye(n))
        x, s, y = O.solve_to_convergence(pr, iters=4000, rho=1.0, alpha=1.6)
        assert abs(pr.q @ x - val) <= 1e-6 * val
        Pm = C.smat(x)
        assert np.allclose(Pm, max(1.0, 1.0 / (2 * a)) * np.eye(n), atol=1e-6)
    # a generated Hurwitz A: the converged P certifies stability
    pr = lyapunov_lmi_problem(np.random.default_rng(1), n=4, kind="oscillator")
    x, s, y = O.solve_to_convergence(pr, iters=20000, rho=1.0, alpha=1.6)
    rp, rd = O.residuals(pr, x, s, y)
    assert np.linalg.norm(rp) < 1e-6 and np.linalg.norm(rd) < 1e-6
    assert np.linalg.eigvalsh(C.smat(x)).min() >= 1.0 - 1e-6


def test_robust_mpc_solution_is_a_feasible_trajectory():
    """PAPER.md App. F.6 (L470-486), N = 6: at the oracle's fixed point the trajectory obeys the double-integrator dynamics
    from x_init, the tightened boxes, |u| <= 0.5, and the epigraph variables equal the norms they bound (gamma > 0)."""
    from workloads import robust_mpc_problem
    N = 6
    pr = robust_mpc_problem(np.random.default_rng(3), N=N)
    x, s, y = O.solve_to_convergence(pr, iters=20000, rho=1.0, alpha=1.6)
    rp, rd = O.residuals(pr, x, s, y)
    assert np.linalg.norm(rp) < 1e-7 and np.linalg.norm(rd) < 1e-7
    X = x[:2 * (N + 1)].reshape(N + 1, 2); U = x[2 * (N + 1):2 * (N + 1) + N]; tau = x[2 * (N + 1) + N:-1]
    Ad = np.array([[1.0, 1.0], [0.0, 1.0]]); Bd = np.array([0.5, 0.1])
    for t in range(N):
        assert np.allclose(X[t + 1], Ad @ X[t] + Bd * U[t], atol=1e-7)
    assert np.all(np.abs(U) <= 0.5 + 1e-7) and np.all(np.abs(X[:, 0]) <= 5 + 1e-7) and np.all(np.abs(X[:, 1]) <= 1 + 1e-7)
    assert np.allclose(tau, np.abs(U), atol=1e-6) and abs(x[-1] - np.linalg.norm(X[N])) < 1e-6

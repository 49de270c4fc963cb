"""ORACLE (test infrastructure, not product code) - unrolled COSMO ADMM, forward and backward, fp64.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may
import this package. It shares no code with the CUDA path and never imports it.

The method is an iteration plus its exact reverse-mode derivative, so the oracle follows the paper's
algorithm step by step with every inner solve done *exactly* where the GPU iterates:

  forward  : PAPER.md Eq. 3a-3e (L62-70) in the indirect form Eq. 4 (L78), dense direct solve
             (numpy.linalg.solve) for n <= DENSE_MAX, else SuperLU on the sparse M; LAPACK eigh for Eq. 7.
  backward : explicit implicit differentiation of Eq. 4 - adjoint solve with the same M (Eq. 5),
             grad_rho = (A lam) o (A xt) (Eq. 6) - the cone VJPs of `cones.py` (Eq. 9-10), and the
             chain rule through the scalar/vector glue.

Sign convention (reading A1): "y in K*", i.e. the paper's Eq. 3-4 with y -> -y, so that the
residuals are exactly those printed in Eq. 12 (L146): r_p = Ax+s-b, r_d = Px+q+A'y. `step_paper_literal`
implements Eq. 3a-3e verbatim (saddle-point solve, nu-tilde, the paper's signs) and the tests assert
x, s equal and y negated.

Pins: tests/test_oracle_*.py (max-cut K_n -> n^2/4; theta(C5)=sqrt5, theta(K_n)=1, theta(empty)=n;
equality-only QP = KKT solve; Eq. 3a <=> Eq. 4; Eq. 6 = explicit -g'M^-1 a_i a_i' xt; whole backward vs
central differences). Parity status: pinned.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence

import numpy as np
import scipy.sparse as sp
import scipy.sparse.linalg as spla

from . import cones as C

DENSE_MAX = 2000


# ---------------------------------------------------------------------------------------------
# linear system  M(rho) = P + sigma I + A' D(rho) A      (Eq. 4)
# ---------------------------------------------------------------------------------------------
class MSolver:
    """Exact solver for M(rho) x = rhs; dense LAPACK for small n, sparse LU otherwise."""

    def __init__(self, P, A, rho_vec, sigma):
        n = A.shape[1]
        self.dense = n <= DENSE_MAX
        if self.dense:
            Ad = A.toarray()
            self.M = P.toarray() + sigma * np.eye(n) + Ad.T @ (rho_vec[:, None] * Ad)
        else:
            M = (P + sigma * sp.identity(n, format="csc") + (A.T @ sp.diags(rho_vec) @ A)).tocsc()
            self.lu = spla.splu(M)

    def solve(self, rhs):
        if self.dense:
            return np.linalg.solve(self.M, rhs)
        return self.lu.solve(rhs)


def _rho_vec(rho, m):
    r = np.asarray(rho, dtype=np.float64)
    return np.full(m, float(r)) if r.ndim == 0 else r.copy()


# ---------------------------------------------------------------------------------------------
# one step, "y in K*" convention
# ---------------------------------------------------------------------------------------------
@dataclass
class StepTape:
    x: np.ndarray
    s: np.ndarray
    y: np.ndarray
    rho: np.ndarray
    alpha: float
    sigma: float
    xt: np.ndarray
    st: np.ndarray
    w: np.ndarray
    s_plus: np.ndarray
    aux: list
    solver: MSolver


def step(pr, x, s, y, rho, alpha, sigma):
    """z^{k+1} = T_theta(z^k; d): Eq. 4 (L78) then Eq. 3b-3e (L64-70) with y -> -y."""
    P, q, A, b = pr.P, pr.q, pr.A, pr.b
    rv = _rho_vec(rho, A.shape[0])
    r = rv * (b - s) - y
    xi = sigma * x - q + A.T @ r                       # RHS of Eq. 4 with y -> -y
    solver = MSolver(P, A, rv, sigma)
    xt = solver.solve(xi)                              # x-tilde
    st = b - A @ xt                                    # Eq. 3b after eliminating nu-tilde
    x_plus = alpha * xt + (1.0 - alpha) * x            # Eq. 3c
    vhat = alpha * st + (1.0 - alpha) * s
    w = vhat - y / rv                                  # argument of Pi in Eq. 3d
    s_plus, aux = C.project(w, pr.cones)               # Eq. 3d
    y_plus = rv * (s_plus - w)                         # Eq. 3e
    tape = StepTape(x=x, s=s, y=y, rho=rv, alpha=float(alpha), sigma=float(sigma), xt=xt, st=st, w=w,
                    s_plus=s_plus, aux=aux, solver=solver)
    return x_plus, s_plus, y_plus, tape


def step_paper_literal(pr, x, s, y, rho, alpha, sigma):
    """Eq. 3a-3e exactly as printed (L62-70): dense saddle-point solve for (x-tilde, nu-tilde), the paper's
    signs for y (COSMO's original convention), with the garbled 'otimes' read as element-wise division
    (reading A2). Returns (x+, s+, y+, xt, nu, st)."""
    n, m = pr.n, pr.m
    rv = _rho_vec(rho, m)
    Ad = pr.A.toarray()
    Kmat = np.block([[pr.P.toarray() + sigma * np.eye(n), Ad.T], [Ad, -np.diag(1.0 / rv)]])
    rhs = np.concatenate([sigma * x - pr.q, pr.b - s + y / rv])
    sol = np.linalg.solve(Kmat, rhs)                                   # Eq. 3a
    xt, nu = sol[:n], sol[n:]
    st = s - (y + nu) / rv                                             # Eq. 3b
    x_plus = alpha * xt + (1 - alpha) * x                              # Eq. 3c
    s_plus, _ = C.project(alpha * st + (1 - alpha) * s + y / rv, pr.cones)   # Eq. 3d
    y_plus = y + rv * (alpha * st + (1 - alpha) * s - s_plus)          # Eq. 3e
    return x_plus, s_plus, y_plus, xt, nu, st


# ---------------------------------------------------------------------------------------------
# unroll and reverse sweep
# ---------------------------------------------------------------------------------------------
@dataclass
class Unroll:
    xs: List[np.ndarray]
    ss: List[np.ndarray]
    ys: List[np.ndarray]
    tapes: List[StepTape] = field(default_factory=list)


def unroll(pr, K, rho, alpha, sigma, x0=None, s0=None, y0=None, keep_tape=True) -> Unroll:
    """K applications of the fixed-point map (L50). rho: [K] scalars or [K][m]; alpha: [K]."""
    x = np.zeros(pr.n) if x0 is None else np.asarray(x0, float).copy()
    s = np.zeros(pr.m) if s0 is None else np.asarray(s0, float).copy()
    y = np.zeros(pr.m) if y0 is None else np.asarray(y0, float).copy()
    out = Unroll([x], [s], [y])
    for k in range(K):
        x, s, y, tape = step(pr, x, s, y, rho[k], alpha[k], sigma)
        out.xs.append(x); out.ss.append(s); out.ys.append(y)
        if keep_tape:
            out.tapes.append(tape)
    return out


@dataclass
class Grads:
    g_rho: np.ndarray      # [K][m] per-row (Eq. 6 verbatim + RHS terms); sum over rows for a scalar rho_k
    g_alpha: np.ndarray    # [K]
    g_sigma: float
    g_x0: np.ndarray
    g_s0: np.ndarray
    g_y0: np.ndarray

    @property
    def g_rho_scalar(self):
        return self.g_rho.sum(axis=1)


def step_backward(pr, tape: StepTape, gx_p, gs_p, gy_p):
    """Reverse of one step (re-derived and pinned by central differences).
    Returns (g_x, g_s, g_y, g_rho_rows, g_alpha, g_sigma)."""
    A = pr.A
    rv, al, sg = tape.rho, tape.alpha, tape.sigma
    # B1  y+ = rho o (s+ - w)
    G = gs_p + rv * gy_p
    g_w = -rv * gy_p
    g_rho = gy_p * (tape.s_plus - tape.w)
    # B2  s+ = Pi_K(w)
    g_w = g_w + C.project_vjp(tape.w, pr.cones, tape.aux, G)
    # B4  w = vhat - y / rho
    g_vhat = g_w
    g_y = -g_w / rv
    g_rho = g_rho + g_w * tape.y / rv ** 2
    # B5  vhat, x+
    g_st = al * g_vhat
    g_s = (1.0 - al) * g_vhat
    g_xt = al * gx_p
    g_x = (1.0 - al) * gx_p
    g_alpha = g_vhat @ (tape.st - tape.s) + gx_p @ (tape.xt - tape.x)
    # B6  st = b - A xt
    g_xt = g_xt - A.T @ g_st
    # B7  xt = M^-1 xi : adjoint solve with the same M (Eq. 5; the paper's lam-tilde = -lam)
    lam = tape.solver.solve(g_xt)
    u = A @ lam
    g_rho = g_rho - u * (A @ tape.xt)                  # Eq. 6 (L90)
    g_sigma = -(lam @ tape.xt)                         # dM/dsigma = I
    # B8  xi = sigma x - q + A' r
    g_x = g_x + sg * lam
    g_sigma = g_sigma + lam @ tape.x
    # B9  r = rho o (b - s) - y
    g_rho = g_rho + u * (pr.b - tape.s)
    g_s = g_s - rv * u
    g_y = g_y - u
    return g_x, g_s, g_y, g_rho, g_alpha, g_sigma


def backward(pr, un: Unroll, g_xK, g_sK, g_yK, inject=None) -> Grads:
    """BPTT through the unroll (L13, L52). `inject[k] = (gx, gs, gy)` adds a cotangent on z^k, k=1..K-1
    (for losses like Eq. 12 that read every iterate)."""
    K = len(un.tapes)
    gx, gs, gy = (np.asarray(v, float).copy() for v in (g_xK, g_sK, g_yK))
    g_rho = np.zeros((K, pr.m)); g_alpha = np.zeros(K); g_sigma = 0.0
    for k in range(K - 1, -1, -1):
        gx, gs, gy, gr, ga, gsg = step_backward(pr, un.tapes[k], gx, gs, gy)
        g_rho[k] = gr; g_alpha[k] = ga; g_sigma += gsg
        if inject is not None and k in inject:
            ix, is_, iy = inject[k]
            gx = gx + ix; gs = gs + is_; gy = gy + iy
    return Grads(g_rho, g_alpha, g_sigma, gx, gs, gy)


# ---------------------------------------------------------------------------------------------
# residuals and the terminal loss of BASELINE.json configs[0] (reading A13)
# ---------------------------------------------------------------------------------------------
def residuals(pr, x, s, y):
    """r_p = Ax + s - b, r_d = Px + q + A'y   as printed in Eq. 12 (L146) and App. E (L323)."""
    return pr.A @ x + s - pr.b, pr.P @ x + pr.q + pr.A.T @ y


def terminal_loss(pr, x, s, y, x_star):
    rp, rd = residuals(pr, x, s, y)
    return float((x - x_star) @ (x - x_star) + rp @ rp + rd @ rd)


def terminal_loss_grad(pr, x, s, y, x_star):
    rp, rd = residuals(pr, x, s, y)
    gx = 2.0 * (x - x_star) + 2.0 * (pr.A.T @ rp) + 2.0 * (pr.P @ rd)
    return gx, 2.0 * rp, 2.0 * (pr.A @ rd)


def solve_to_convergence(pr, iters=3000, rho=1.0, alpha=1.6, sigma=1e-6, x0=None, s0=None, y0=None):
    """Vanilla fixed-hyper-parameter COSMO (a zero-initialised policy reduces to this, L341)."""
    un = unroll(pr, iters, [rho] * iters, [alpha] * iters, sigma, x0, s0, y0, keep_tape=False)
    return un.xs[-1], un.ss[-1], un.ys[-1]


# ---------------------------------------------------------------------------------------------
# batch helpers used by tests / smoke / cpu_baseline
# ---------------------------------------------------------------------------------------------
def run_workload(wl, cot_fn=None, x_star: Optional[Sequence[np.ndarray]] = None, problems=None):
    """Forward + backward for every instance of a Workload (rho, alpha shared by the batch, so their
    gradients are summed over the batch: CDU_RHO_PER_ITER). `cot_fn(b, pr, xK, sK, yK) -> (gx, gs, gy)`
    supplies the terminal cotangent; default = gradient of `terminal_loss` with x_star (zeros if absent).
    Returns dict with lists xK, sK, yK, cot, g_x0, g_s0, g_y0 and summed g_rho[K], g_alpha[K], g_sigma."""
    idx = range(wl.batch) if problems is None else problems
    res = dict(xK=[], sK=[], yK=[], cot=[], g_x0=[], g_s0=[], g_y0=[], g_rho_pb=[], g_alpha_pb=[], g_sigma_pb=[])
    for b in idx:
        pr = wl.problems[b]
        un = unroll(pr, wl.K, wl.rho, wl.alpha, wl.sigma, wl.x0[b], wl.s0[b], wl.y0[b])
        xK, sK, yK = un.xs[-1], un.ss[-1], un.ys[-1]
        if cot_fn is not None:
            cot = cot_fn(b, pr, xK, sK, yK)
        else:
            xs = np.zeros(pr.n) if x_star is None else x_star[b]
            cot = terminal_loss_grad(pr, xK, sK, yK, xs)
        g = backward(pr, un, *cot)
        res["xK"].append(xK); res["sK"].append(sK); res["yK"].append(yK); res["cot"].append(cot)
        res["g_x0"].append(g.g_x0); res["g_s0"].append(g.g_s0); res["g_y0"].append(g.g_y0)
        res["g_rho_pb"].append(g.g_rho_scalar); res["g_alpha_pb"].append(g.g_alpha); res["g_sigma_pb"].append(g.g_sigma)
    res["g_rho"] = np.sum(res["g_rho_pb"], axis=0)
    res["g_alpha"] = np.sum(res["g_alpha_pb"], axis=0)
    res["g_sigma"] = float(np.sum(res["g_sigma_pb"]))
    return res


# ---------------------------------------------------------------------------------------------
# training loss of Eq. 12 (L146-148) and the policy features of App. E (L321-339)
# ---------------------------------------------------------------------------------------------
def eq12_loss(pr, un: Unroll) -> float:
    """L = sum_{k=1..K} log(||r_d^k||^2 / det(||r_d^0||^2) + ||r_p^k||^2 / det(||r_p^0||^2))  (Eq. 12); a term whose
    denominator is zero is dropped (paper silent; reading A12)."""
    rp0, rd0 = residuals(pr, un.xs[0], un.ss[0], un.ys[0])
    a0, b0 = rd0 @ rd0, rp0 @ rp0
    L = 0.0
    for k in range(1, len(un.xs)):
        rp, rd = residuals(pr, un.xs[k], un.ss[k], un.ys[k])
        Dk = (rd @ rd / a0 if a0 > 0 else 0.0) + (rp @ rp / b0 if b0 > 0 else 0.0)
        if Dk > 0:
            L += np.log(Dk)
    return float(L)


def eq12_cotangents(pr, un: Unroll):
    """dL/dz^k of Eq. 12 for k = 1..K with the denominators detached ("det", L148): dict k -> (gx, gs, gy).
    d/dx = (2/D_k)(P' r_d / a_0 + A' r_p / b_0), d/ds = (2/D_k) r_p / b_0, d/dy = (2/D_k) A r_d / a_0."""
    rp0, rd0 = residuals(pr, un.xs[0], un.ss[0], un.ys[0])
    a0, b0 = rd0 @ rd0, rp0 @ rp0
    out = {}
    for k in range(1, len(un.xs)):
        rp, rd = residuals(pr, un.xs[k], un.ss[k], un.ys[k])
        Dk = (rd @ rd / a0 if a0 > 0 else 0.0) + (rp @ rp / b0 if b0 > 0 else 0.0)
        if not Dk > 0:
            out[k] = (np.zeros(pr.n), np.zeros(pr.m), np.zeros(pr.m))
            continue
        c1 = 2.0 / (Dk * a0) if a0 > 0 else 0.0
        c2 = 2.0 / (Dk * b0) if b0 > 0 else 0.0
        out[k] = (c1 * (pr.P.T @ rd) + c2 * (pr.A.T @ rp), c2 * rp, c1 * (pr.A @ rd))
    return out


def backward_eq12(pr, un: Unroll) -> Grads:
    """BPTT of the Eq. 12 loss: its cotangent on z^K is the terminal one, those on z^1..z^(K-1) are injected."""
    cots = eq12_cotangents(pr, un)
    K = len(un.tapes)
    return backward(pr, un, *cots[K], inject={k: cots[k] for k in range(1, K)})


def features(pr, un: Unroll, k: int, eps: float = 1e-12):
    """App. E (L323-335): OSQP-scaled KKT residuals of z^k, the ADMM residuals delta_d = s^k - s^(k-1) and
    delta_p = s^k - s-tilde^k, and the three log-infinity-norms the alpha policy reads."""
    x, s, y = un.xs[k], un.ss[k], un.ys[k]
    Ax, Px, ATy = pr.A @ x, pr.P @ x, pr.A.T @ y
    inf = lambda v: float(np.max(np.abs(v), initial=0.0))
    dp, dd = max(inf(Ax), inf(s), inf(pr.b)), max(inf(Px), inf(pr.q), inf(ATy))
    rp_bar = (Ax + s - pr.b) / (dp if dp > 0 else 1.0)
    rd_bar = (Px + pr.q + ATy) / (dd if dd > 0 else 1.0)
    delta_d = s - un.ss[k - 1] if k >= 1 else np.zeros(pr.m)
    delta_p = s - un.tapes[k - 1].st if k >= 1 else np.zeros(pr.m)
    scal = np.log(np.array([inf(rp_bar), inf(rd_bar), inf(delta_p)]) + eps)
    return dict(rp_bar=rp_bar, rd_bar=rd_bar, delta_p=delta_p, delta_d=delta_d, scal=scal)

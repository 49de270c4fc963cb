"""Seeded synthetic workloads for the unrolled COSMO hot path (inputs only, no solver arithmetic).

Problem statement: PAPER.md Eq. 1 (L42-48)   min 1/2 x'Px + q'x  s.t.  Ax + s = b, s in K.
Workload recipes: BASELINE.json `configs[0..4]` (they re-parameterise the paper's max-cut and
Lovasz generators, App. F.3/F.4) and SURVEY.md section 8(d).

Interface conventions fixed here:
  * svec: upper triangle, column by column, off-diagonals scaled by sqrt(2)
      (X11, r2*X12, X22, r2*X13, r2*X23, X33, ...), so <svec X, svec Y> = tr(XY).
  * SOC_d = {(t,u) : ||u||_2 <= t}, t first.
  * cones tile the rows of A in order; PSD cone of order p owns p(p+1)/2 rows.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np
import scipy.sparse as sp

ZERO, NONNEG, SOC, PSD = 0, 1, 2, 3
BASE_SEED = 2606138250
CONFIG_NAMES = {
    1: "cfg1-maxcut-n10-b4-f64-K20",
    2: "cfg2-maxcut-n50-b256-f32-K50",
    3: "cfg3-socp-n200-b1024-f32-K100",
    4: "cfg4-lovasz-n100-b64-f32-K100",
    5: "cfg5-maxcut-n512-b8-f32-K200",
}
_SQRT2 = float(np.sqrt(2.0))


def svec_dim(p: int) -> int:
    return p * (p + 1) // 2


def svec_index(i: int, j: int) -> int:
    """Position of X_ij (any order of i, j) in svec(X); upper triangle, column by column."""
    if i > j:
        i, j = j, i
    return j * (j + 1) // 2 + i


def cone_rows(kind: int, dim: int) -> int:
    return svec_dim(dim) if kind == PSD else dim


@dataclass
class Problem:
    """One instance d = (P, q, A, b, K) of PAPER.md Eq. 1 (L48)."""

    P: sp.csr_matrix  # n x n, full symmetric storage (both triangles)
    q: np.ndarray  # n
    A: sp.csr_matrix  # m x n
    b: np.ndarray  # m
    cones: List[Tuple[int, int]]  # (kind, dim); dim = rows, or matrix order for PSD
    name: str = ""

    @property
    def n(self) -> int:
        return self.A.shape[1]

    @property
    def m(self) -> int:
        return self.A.shape[0]

    def check(self) -> None:
        assert self.P.shape == (self.n, self.n)
        assert self.q.shape == (self.n,) and self.b.shape == (self.m,)
        assert sum(cone_rows(k, d) for k, d in self.cones) == self.m


@dataclass
class Workload:
    """A batch of instances plus the unroll's hyper-parameters and start."""

    name: str
    dtype: str  # "f32" | "f64": dtype the GPU computes in; all values are pre-rounded to it
    problems: List[Problem]
    K: int
    rho: np.ndarray  # [K], shared by the batch (CDU_RHO_PER_ITER)
    alpha: np.ndarray  # [K]
    sigma: float
    x0: List[np.ndarray] = field(default_factory=list)
    s0: List[np.ndarray] = field(default_factory=list)
    y0: List[np.ndarray] = field(default_factory=list)

    @property
    def batch(self) -> int:
        return len(self.problems)


# ----------------------------------------------------------------------------------------------
# graphs
# ----------------------------------------------------------------------------------------------
def erdos_renyi(rng: np.random.Generator, n: int, p: float, weights: str = "unit") -> np.ndarray:
    """Symmetric weight matrix of G ~ ER(n, p); `weights` = "unit" or "uniform" (U[0,1])."""
    iu = np.triu_indices(n, 1)
    mask = rng.random(iu[0].size) < p
    w = np.ones(iu[0].size) if weights == "unit" else rng.random(iu[0].size)
    W = np.zeros((n, n))
    W[iu] = np.where(mask, w, 0.0)
    return W + W.T


def complete_graph(n: int) -> np.ndarray:
    return np.ones((n, n)) - np.eye(n)


def cycle_graph(n: int) -> np.ndarray:
    W = np.zeros((n, n))
    for i in range(n):
        W[i, (i + 1) % n] = W[(i + 1) % n, i] = 1.0
    return W


# ----------------------------------------------------------------------------------------------
# problem builders
# ----------------------------------------------------------------------------------------------
def _svec_of_symmetric(S: np.ndarray) -> np.ndarray:
    """Layout helper for building q from a data matrix (same convention as svec_index)."""
    p = S.shape[0]
    out = np.empty(svec_dim(p))
    for j in range(p):
        base = j * (j + 1) // 2
        out[base : base + j] = _SQRT2 * S[:j, j]
        out[base + j] = S[j, j]
    return out


def maxcut_problem(W: np.ndarray, name: str = "maxcut") -> Problem:
    """Max-cut SDP (App. F.3; display missing, BASELINE.json configs[0] states it):
    min -1/4 <L, X>  s.t. diag(X) = 1, X PSD;  L = D - W.
    x = svec(X); P = 0; q = -svec(L/4); rows 0..p-1: X_ii + s = 1 (ZERO); then -svec(X) + s = 0 (PSD_p).
    """
    p = W.shape[0]
    n = svec_dim(p)
    L = np.diag(W.sum(1)) - W
    q = -_svec_of_symmetric(L / 4.0)
    rows = np.arange(p)
    cols = np.array([svec_index(i, i) for i in range(p)])
    E = sp.csr_matrix((np.ones(p), (rows, cols)), shape=(p, n))
    A = sp.vstack([E, -sp.identity(n, format="csr")], format="csr")
    b = np.concatenate([np.ones(p), np.zeros(n)])
    P = sp.csr_matrix((n, n))
    return Problem(P=P, q=q, A=A, b=b, cones=[(ZERO, p), (PSD, p)], name=name)


def lovasz_problem(W: np.ndarray, name: str = "lovasz") -> Problem:
    """Lovasz theta SDP (App. F.4): max <J,X> s.t. tr X = 1, X_ij = 0 on edges, X PSD.
    q = -svec(J); row 0: sum of diagonal = 1; one row per edge: sqrt(2) X_ij = 0 written as a unit
    entry at the svec position; all ZERO; then -svec(X) + s = 0 (PSD_p).  theta = -q'x.
    """
    p = W.shape[0]
    n = svec_dim(p)
    q = -_svec_of_symmetric(np.ones((p, p)))
    edges = [(i, j) for j in range(p) for i in range(j) if W[i, j] != 0.0]
    ne = len(edges)
    r = [0] * p + list(range(1, ne + 1))
    c = [svec_index(i, i) for i in range(p)] + [svec_index(i, j) for (i, j) in edges]
    Aeq = sp.csr_matrix((np.ones(p + ne), (r, c)), shape=(1 + ne, n))
    A = sp.vstack([Aeq, -sp.identity(n, format="csr")], format="csr")
    b = np.concatenate([[1.0], np.zeros(ne), np.zeros(n)])
    return Problem(P=sp.csr_matrix((n, n)), q=q, A=A, b=b, cones=[(ZERO, 1 + ne), (PSD, p)], name=name)


def socp_problem(rng: np.random.Generator, n: int = 200, ncones: int = 100, cdim: int = 11,
                 density: float = 0.1, name: str = "socp") -> Problem:
    """BASELINE.json configs[2]: x in R^n, P = M'M/n + 0.1 I, q ~ N(0,1); cones
    ||A_i x + b_i|| <= c_i'x + d_i of dimension cdim; rows [-c_i'; -A_i], rhs [d_i; b_i]."""
    M = rng.standard_normal((n, n))
    Pd = M.T @ M / float(n) + 0.1 * np.eye(n)
    Pd = 0.5 * (Pd + Pd.T)
    q = rng.standard_normal(n)
    xfeas = rng.standard_normal(n)
    k = cdim - 1
    Ai = rng.standard_normal((ncones, k, n)) * (rng.random((ncones, k, n)) < density)
    bi = rng.standard_normal((ncones, k))
    ci = rng.standard_normal((ncones, n))
    di = np.linalg.norm(Ai @ xfeas + bi, axis=1) - ci @ xfeas + 1.0
    blocks = -np.concatenate([ci[:, None, :], Ai], axis=1).reshape(ncones * cdim, n)
    rhs = np.concatenate([di[:, None], bi], axis=1).reshape(-1)
    A = sp.csr_matrix(blocks)
    A.eliminate_zeros()
    return Problem(P=sp.csr_matrix(Pd), q=q, A=A, b=rhs,
                   cones=[(SOC, cdim)] * ncones, name=name)


def random_mixed_problem(rng: np.random.Generator, n: int = 7,
                         cones: Sequence[Tuple[int, int]] = ((ZERO, 2), (NONNEG, 3), (SOC, 4), (PSD, 3)),
                         density: float = 0.6, with_P: bool = True) -> Problem:
    """Small random instance with every cone type (test fixture; SURVEY.md 8(c)-C 'whole backward')."""
    m = sum(cone_rows(k, d) for k, d in cones)
    A = rng.standard_normal((m, n)) * (rng.random((m, n)) < density)
    for i in range(m):  # no empty rows / columns so that M is well conditioned
        if not A[i].any():
            A[i, rng.integers(n)] = rng.standard_normal()
    for j in range(n):
        if not A[:, j].any():
            A[rng.integers(m), j] = rng.standard_normal()
    if with_P:
        G = rng.standard_normal((n, n))
        Pd = G.T @ G / n
        Pd = 0.5 * (Pd + Pd.T)
    else:
        Pd = np.zeros((n, n))
    return Problem(P=sp.csr_matrix(Pd), q=rng.standard_normal(n), A=sp.csr_matrix(A),
                   b=rng.standard_normal(m), cones=list(cones), name="mixed")


def fig2_linear_problem(rng: np.random.Generator, n: int, density: float = 0.01) -> Problem:
    """PAPER.md App. B (L247): m = n/2, diagonal P ~ U(0,10), A `density` dense with N(0,1) entries,
    b ~ N(0,1). The cone is irrelevant to the linear-solve experiment; rows are declared ZERO."""
    m = n // 2
    P = sp.diags(rng.uniform(0.0, 10.0, n), format="csr")
    A = sp.random(m, n, density=density, format="csr", random_state=rng,
                  data_rvs=lambda k: rng.standard_normal(k))
    return Problem(P=P, q=rng.standard_normal(n), A=A, b=rng.standard_normal(m), cones=[(ZERO, m)],
                   name=f"fig2-n{n}")


# ----------------------------------------------------------------------------------------------
# hyper-parameter schedules and configs
# ----------------------------------------------------------------------------------------------
def ar1_rho_schedule(rng: np.random.Generator, K: int, rho_base: float, decay: float = 0.9,
                     step: float = 0.15, lo: float = 0.01, hi: float = 10.0) -> np.ndarray:
    """Smooth mean-reverting schedule of SURVEY.md 8(d): u_0 = g_0, u_k = decay u_{k-1} + g_k,
    g_k ~ N(0, step^2), rho_k = clip(rho_base e^{u_k}, lo, hi)."""
    g = rng.standard_normal(K) * step
    u = np.empty(K)
    acc = 0.0
    for k in range(K):
        acc = decay * acc + g[k] if k else g[0]
        u[k] = acc
    return np.clip(rho_base * np.exp(u), lo, hi)


def _round_to(a, dtype: str):
    a = np.asarray(a, dtype=np.float64)
    return a.astype(np.float32).astype(np.float64) if dtype == "f32" else a


def _round_problem(pr: Problem, dtype: str) -> Problem:
    if dtype != "f32":
        return pr
    P = pr.P.copy()
    P.data = _round_to(P.data, dtype)
    A = pr.A.copy()
    A.data = _round_to(A.data, dtype)
    return Problem(P=P, q=_round_to(pr.q, dtype), A=A, b=_round_to(pr.b, dtype), cones=pr.cones, name=pr.name)


def lovasz_dual_feasible_start(pr: Problem):
    """Start for cfg4: X0 = I/p, s0 = svec(X0) on the PSD rows, y0 = t on the
    trace row, 0 on edge rows, svec(t I - J) on the PSD rows with t = p (so that Px+q+A'y = 0)."""
    (k0, nz), (k1, p) = pr.cones
    assert k0 == ZERO and k1 == PSD
    x0 = _svec_of_symmetric(np.eye(p) / p)
    s0 = np.concatenate([np.zeros(nz), x0])
    t = float(p)
    y0 = np.concatenate([[t], np.zeros(nz - 1), _svec_of_symmetric(t * np.eye(p) - np.ones((p, p)))])
    return x0, s0, y0


def make_config(cfg: int, batch: Optional[int] = None, K: Optional[int] = None,
                p: Optional[int] = None, seed_offset: int = 0, dtype: Optional[str] = None) -> Workload:
    """BASELINE.json configs[cfg-1] with the recipes of SURVEY.md 8(d). `batch`, `K`, `p` (graph order /
    number of variables for cfg3) override the full sizes for down-scaled parity cases; `seed_offset` shifts the
    instance seeds (hyper-parameters stay shared) so that every rank of a weak-scaling run draws its own batch;
    `dtype` overrides the config's precision (parity cases that push the fp64 kernels through the large-block path)."""
    full = {1: (4, 20, 10), 2: (256, 50, 50), 3: (1024, 100, 200), 4: (64, 100, 100), 5: (8, 200, 512)}[cfg]
    B = batch if batch is not None else full[0]
    Kk = K if K is not None else full[1]
    pp = p if p is not None else full[2]
    dtype_cfg = "f64" if cfg == 1 else "f32"
    dtype = dtype if dtype is not None else dtype_cfg
    hrng = np.random.default_rng(BASE_SEED + 1000 * cfg + 999)
    problems = []
    for b in range(B):
        rng = np.random.default_rng(BASE_SEED + 1000 * cfg + b + seed_offset)
        if cfg == 1:
            pr = maxcut_problem(erdos_renyi(rng, pp, 0.5, "unit"))
        elif cfg == 2:
            pb = rng.uniform(0.1, 0.5)
            pr = maxcut_problem(erdos_renyi(rng, pp, pb, "uniform"))
        elif cfg == 3:
            pr = socp_problem(rng, n=pp, ncones=max(1, pp // 2), cdim=11, density=0.1)
        elif cfg == 4:
            pr = lovasz_problem(erdos_renyi(rng, pp, 0.1, "unit"))
        elif cfg == 5:
            pr = maxcut_problem(erdos_renyi(rng, pp, 0.02, "unit"))
        else:
            raise ValueError(cfg)
        pr.name = f"cfg{cfg}-b{b}"
        problems.append(_round_problem(pr, dtype))
    if cfg == 1:
        rho = np.exp(hrng.uniform(np.log(0.01), np.log(10.0), Kk))
    else:
        base = {2: 0.3, 3: 1.0, 4: 10.0, 5: 0.3}[cfg]
        rho = ar1_rho_schedule(hrng, Kk, base)
    alpha = np.full(Kk, 1.6)
    sigma = 1e-6
    x0, s0, y0 = [], [], []
    for pr in problems:
        if cfg == 4:
            a, b_, c = lovasz_dual_feasible_start(pr)
        else:
            a, b_, c = np.zeros(pr.n), np.zeros(pr.m), np.zeros(pr.m)
        x0.append(_round_to(a, dtype)); s0.append(_round_to(b_, dtype)); y0.append(_round_to(c, dtype))
    return Workload(name=CONFIG_NAMES[cfg] if (batch, K, p) == (None, None, None) and dtype == dtype_cfg else
                    f"cfg{cfg}-p{pp}-b{B}-K{Kk}-{dtype}", dtype=dtype, problems=problems, K=Kk,
                    rho=_round_to(rho, dtype), alpha=_round_to(alpha, dtype), sigma=sigma, x0=x0, s0=s0, y0=y0)


def lyapunov_lmi_problem(rng: np.random.Generator, n: int = 40, kind: str = "triangular", A_sys: Optional[np.ndarray] = None) -> Problem:
    """Minimum-trace Lyapunov LMI of PAPER.md App. F.2 (L422-434): min tr(P) s.t. A'P + PA <= -I, P >= I, for a Hurwitz A
    generated as Q T Q' (T upper triangular, T_ii ~ U(-2,-0.1), N(0,1) above the diagonal; kind "triangular") or Q R Q' (R =
    blkdiag of damped oscillators [[-z w, w], [-w, -z w]], w ~ U(0.5,5), z ~ U(0.05,0.5); kind "oscillator"; the paper prints
    +z w in the lower right entry, which is not Hurwitz - read as -z w). Conic form: x = svec(P), q = svec(I),
    rows [svec(A'PA-map); -I], b = [-svec(I); -svec(I)], two PSD_n cones."""
    if A_sys is None:
        Q, _ = np.linalg.qr(rng.standard_normal((n, n)))
        if kind == "triangular":
            Tm = np.triu(rng.standard_normal((n, n)), 1) + np.diag(rng.uniform(-2.0, -0.1, n))
            A_sys = Q @ Tm @ Q.T
        else:
            R = np.zeros((n, n))
            for i in range(n // 2):
                w, z = rng.uniform(0.5, 5.0), rng.uniform(0.05, 0.5)
                R[2 * i:2 * i + 2, 2 * i:2 * i + 2] = [[-z * w, w], [-w, -z * w]]
            if n % 2:
                R[-1, -1] = -rng.uniform(0.1, 2.0)
            A_sys = Q @ R @ Q.T
    d = svec_dim(n)
    cols = []
    for j in range(n):
        for i in range(j + 1):
            E = np.zeros((n, n))
            if i == j:
                E[i, i] = 1.0
            else:
                E[i, j] = E[j, i] = 1.0 / np.sqrt(2.0)
            cols.append(_svec_of_symmetric(A_sys.T @ E + E @ A_sys))
    L = np.stack(cols, axis=1)
    L[np.abs(L) < 1e-15] = 0.0
    eye = _svec_of_symmetric(np.eye(n))
    A = sp.vstack([sp.csr_matrix(L), -sp.identity(d, format="csr")], format="csr")
    return Problem(P=sp.csr_matrix((d, d)), q=eye.copy(), A=A, b=np.concatenate([-eye, -eye]), cones=[(PSD, n), (PSD, n)],
                   name=f"lyapunov-n{n}-{kind}")


def robust_mpc_problem(rng: np.random.Generator, N: int = 50, kappa: float = 1.0) -> Problem:
    """Robust MPC SOCP of PAPER.md App. F.6 (L470-486): 1-D double integrator A = [[1,1],[0,1]], B = (0.5, 0.1), Q = Q_N = R = I,
    box constraints |x_1| <= 5, |x_2| <= 1, |u| <= 0.5 tightened by kappa d_t with Sigma_{t+1} = A Sigma_t A' + sigma^2 I
    (sigma = 0.01, Sigma_0 = 0), ||u_t|| <= tau_t, ||x_N|| <= tau_term, x_init ~ U(-(1, 0.3), (1, 0.3)), gamma ~ U(0.01, 0.1),
    gamma_term ~ U(1, 10). kappa is not given in the paper (reading: 1). Variables (x_0..x_N, u_0..u_{N-1}, tau_0..tau_{N-1},
    tau_term); rows: dynamics and x_0 (ZERO), state and input half-spaces (NONNEG), N cones SOC_2, one SOC_3."""
    Ad = np.array([[1.0, 1.0], [0.0, 1.0]]); Bd = np.array([0.5, 0.1])
    Ax = np.array([[1.0, 0.0], [0.0, 1.0], [-1.0, 0.0], [0.0, -1.0]]); bx = np.array([5.0, 1.0, 5.0, 1.0])
    bu = 0.5
    x_init = rng.uniform(-1.0, 1.0, 2) * np.array([1.0, 0.3])
    gam, gam_t = rng.uniform(0.01, 0.1), rng.uniform(1.0, 10.0)
    nx, nu = 2 * (N + 1), N
    ix = lambda t: 2 * t
    iu = lambda t: nx + t
    it = lambda t: nx + nu + t
    itt = nx + 2 * nu
    n = itt + 1
    Pd = np.zeros(n); Pd[:nx + nu] = 2.0                      # x'Qx + u'Ru = 1/2 z'(2I)z on the x and u entries
    q = np.zeros(n); q[nx + nu:itt] = gam; q[itt] = gam_t
    rows, cols, vals, b = [], [], [], []

    def add(entries, rhs):
        r = len(b)
        for c, v in entries:
            rows.append(r); cols.append(c); vals.append(v)
        b.append(rhs)

    for t in range(N):                                        # x_{t+1} - A x_t - B u_t = 0
        for i in range(2):
            add([(ix(t + 1) + i, 1.0)] + [(ix(t) + j, -Ad[i, j]) for j in range(2) if Ad[i, j] != 0.0] + [(iu(t), -Bd[i])], 0.0)
    for i in range(2):
        add([(ix(0) + i, 1.0)], x_init[i])
    n_zero = len(b)
    Sig = np.zeros((2, 2))
    for t in range(N + 1):                                    # A_x x_t + s = b_x - kappa d_t
        d = np.sqrt(np.maximum(np.einsum("ij,jk,ik->i", Ax, Sig, Ax), 0.0))
        for i in range(4):
            add([(ix(t) + j, Ax[i, j]) for j in range(2) if Ax[i, j] != 0.0], bx[i] - kappa * d[i])
        Sig = Ad @ Sig @ Ad.T + 0.01 ** 2 * np.eye(2)
    for t in range(N):                                        # +-u_t + s = b_u
        add([(iu(t), 1.0)], bu); add([(iu(t), -1.0)], bu)
    n_nonneg = len(b) - n_zero
    for t in range(N):                                        # (tau_t, u_t) in SOC_2
        add([(it(t), -1.0)], 0.0); add([(iu(t), -1.0)], 0.0)
    add([(itt, -1.0)], 0.0)                                   # (tau_term, x_N - 0) in SOC_3
    for i in range(2):
        add([(ix(N) + i, -1.0)], 0.0)
    A = sp.csr_matrix((vals, (rows, cols)), shape=(len(b), n))
    cones = [(ZERO, n_zero), (NONNEG, n_nonneg)] + [(SOC, 2)] * N + [(SOC, 3)]
    return Problem(P=sp.diags(Pd, format="csr"), q=q, A=A, b=np.array(b), cones=cones, name=f"robust-mpc-N{N}")


def clustered_spectrum_matrix(rng: np.random.Generator, n: int, delta: float) -> np.ndarray:
    """The sampler of PAPER.md Eq. 13 (App. C): n even, eigenvalues -delta/2 + u_i (first half) and +delta/2 + u_i,
    u_i ~ U(-sigma, sigma) with sigma = 1e-3 delta, S = Q diag(lambda) Q' for a random orthogonal Q."""
    sig = 1e-3 * delta
    lam = np.concatenate([-delta / 2 + rng.uniform(-sig, sig, n // 2), delta / 2 + rng.uniform(-sig, sig, n - n // 2)])
    Q, _ = np.linalg.qr(rng.standard_normal((n, n)))
    S = (Q * lam) @ Q.T
    return 0.5 * (S + S.T)


def make_fig2(n: int, batch: int = 1, dtype: str = "f64", seed_offset: int = 0) -> Workload:
    """The linear-solve scaling workload of PAPER.md Fig. 2 / App. B (L96, L247-255): `batch` instances of
    fig2_linear_problem(n) (m = n/2, diag P ~ U(0,10), A 1 % dense N(0,1), b ~ N(0,1)), ONE step (K = 1) with
    rho ~ U(0,1) (a scalar per instance: per-row rho is SURVEY 8(f) F3), alpha = 1 (x_1 = x-tilde), sigma = 1e-6, from a
    N(0,1) iterate. The loss of the experiment, 1/2 ||x-tilde - x*||^2, lives with the caller (x* ~ N(0,1))."""
    problems, x0, s0, y0 = [], [], [], []
    for b in range(batch):
        rng = np.random.default_rng(BASE_SEED + 6000 + 97 * n + b + seed_offset)
        pr = fig2_linear_problem(rng, n)
        pr.name = f"fig2-n{n}-b{b}"
        problems.append(_round_problem(pr, dtype))
        x0.append(_round_to(rng.standard_normal(pr.n), dtype)); s0.append(_round_to(rng.standard_normal(pr.m), dtype))
        y0.append(_round_to(rng.standard_normal(pr.m), dtype))
    hrng = np.random.default_rng(BASE_SEED + 6000 + 999)
    return Workload(name=f"fig2-linsolve-n{n}-b{batch}-{dtype}-K1", dtype=dtype, problems=problems, K=1,
                    rho=_round_to(hrng.uniform(0.05, 1.0, 1), dtype), alpha=_round_to(np.ones(1), dtype), sigma=1e-6,
                    x0=x0, s0=s0, y0=y0)


# ----------------------------------------------------------------------------------------------
# batched-CSR packing (layout of include/cdu.h `cdu_problem`)
# ----------------------------------------------------------------------------------------------
def pack_batch(problems: Sequence[Problem], dtype: str) -> dict:
    """Block-diagonal batched CSR: global rowptr (int64), problem-local column indices (int32)."""
    fdt = np.float32 if dtype == "f32" else np.float64
    var_off = np.zeros(len(problems) + 1, np.int64)
    row_off = np.zeros(len(problems) + 1, np.int64)
    cone_off = np.zeros(len(problems) + 1, np.int64)
    for i, pr in enumerate(problems):
        var_off[i + 1] = var_off[i] + pr.n
        row_off[i + 1] = row_off[i] + pr.m
        cone_off[i + 1] = cone_off[i] + len(pr.cones)

    def stack(mats):
        ptr, idx, val, base = [np.zeros(1, np.int64)], [], [], 0
        for M in mats:
            M = M.tocsr()
            M.sort_indices()
            ptr.append(M.indptr[1:].astype(np.int64) + base)
            idx.append(M.indices.astype(np.int32))
            val.append(M.data.astype(fdt))
            base += M.nnz
        cat = lambda xs, dt: np.concatenate(xs).astype(dt) if xs else np.zeros(0, dt)
        return np.concatenate(ptr), cat(idx, np.int32), cat(val, fdt)

    A_rowptr, A_colidx, A_val = stack([pr.A for pr in problems])
    P_rowptr, P_colidx, P_val = stack([pr.P for pr in problems])
    cones = np.array([c for pr in problems for c in pr.cones], np.int32).reshape(-1, 2)
    return dict(batch=len(problems), dtype=dtype, var_off=var_off, row_off=row_off,
                A_rowptr=A_rowptr, A_colidx=A_colidx, A_val=A_val,
                P_rowptr=P_rowptr, P_colidx=P_colidx, P_val=P_val,
                q=np.concatenate([pr.q for pr in problems]).astype(fdt),
                b=np.concatenate([pr.b for pr in problems]).astype(fdt),
                cone_off=cone_off, cones=np.ascontiguousarray(cones))

"""ORACLE (test infrastructure, not product code) - cone projections and their VJPs, fp64, NumPy.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may
import this package. It shares no code with the CUDA path.

What each function follows:
  * projection onto K in PAPER.md Eq. 3d (L68); "zero, nonnegative-orthant, and SOCs ... smooth (or
    piecewise-smooth)" (L100) - textbook formulas, reading A4;
  * PSD projection  Pi(S) = U max(Lambda,0) U'   PAPER.md Eq. 7 (L102), with LAPACK `eigh`;
  * Dalecki-Krein VJP  Sbar = U (L o (U' Tbar U)) U'   PAPER.md Eq. 9-10 (L112-117);
  * the naive eigendecomposition VJP  Sbar = U (Lbar + F o (U' Ubar)) U'   PAPER.md Eq. 8 (L106),
    kept only as the negative control (it must blow up where Eq. 9 does not, L119).

Pins (tests/test_oracle_cones.py): idempotence, Moreau decomposition, Pi(S) - Pi(-S) = S,
Pi(S) = (S+|S|)/2 (L131), central differences incl. exactly repeated eigenvalues, Eq. 13 sweep.
Parity status: pinned.
"""
from __future__ import annotations

import numpy as np

ZERO, NONNEG, SOC, PSD = 0, 1, 2, 3
_R2 = np.sqrt(2.0)


# ---------------------------------------------------------------------------------------------
# svec / smat  (reading A3: upper triangle column by column, off-diagonals * sqrt 2)
# ---------------------------------------------------------------------------------------------
def svec(X: np.ndarray) -> np.ndarray:
    p = X.shape[0]
    out = np.empty(p * (p + 1) // 2)
    k = 0
    for j in range(p):
        for i in range(j + 1):
            out[k] = X[i, j] if i == j else _R2 * X[i, j]
            k += 1
    return out


def smat(v: np.ndarray) -> np.ndarray:
    d = v.shape[0]
    p = int(round((np.sqrt(8 * d + 1) - 1) / 2))
    assert p * (p + 1) // 2 == d
    X = np.empty((p, p))
    k = 0
    for j in range(p):
        for i in range(j + 1):
            if i == j:
                X[i, j] = v[k]
            else:
                X[i, j] = X[j, i] = v[k] / _R2
            k += 1
    return X


# ---------------------------------------------------------------------------------------------
# projections (each returns (projection, aux) with aux = what the VJP needs)
# ---------------------------------------------------------------------------------------------
def proj_zero(w):
    return np.zeros_like(w), None


def proj_nonneg(w):
    return np.maximum(w, 0.0), None


def proj_soc(w):
    """SOC_d = {(t,u): ||u|| <= t}. Branch order and `<=` per DESIGN.md reading A4."""
    t, u = w[0], w[1:]
    nu = np.linalg.norm(u)
    if nu <= t:
        return w.copy(), 0
    if nu <= -t:
        return np.zeros_like(w), 1
    c = 0.5 * (t + nu)
    out = np.empty_like(w)
    out[0] = c
    out[1:] = c * u / nu
    return out, 2


def proj_psd(w):
    """Eq. 7 (L102) on S = smat(w)."""
    S = smat(w)
    lam, U = np.linalg.eigh(S)
    T = (U * np.maximum(lam, 0.0)) @ U.T
    T = 0.5 * (T + T.T)
    return svec(T), (lam, U)


# ---------------------------------------------------------------------------------------------
# VJPs  (J_Pi is symmetric for every cone, so VJP = JVP)
# ---------------------------------------------------------------------------------------------
def vjp_zero(w, aux, G):
    return np.zeros_like(G)


def vjp_nonneg(w, aux, G):
    return G * (w > 0.0)  # reading A11: pass iff w > 0


def vjp_soc(w, aux, G):
    """Derivative of the three-branch formula; boundary branch."""
    t, u = w[0], w[1:]
    nu = np.linalg.norm(u)
    if nu <= t:
        return G.copy()
    if nu <= -t:
        return np.zeros_like(G)
    uh = u / nu
    Gt, Gu = G[0], G[1:]
    out = np.empty_like(G)
    d = uh @ Gu
    out[0] = 0.5 * (Gt + d)
    out[1:] = 0.5 * (Gt * uh + (1.0 + t / nu) * Gu - (t / nu) * d * uh)
    return out


def loewner_relu(lam: np.ndarray) -> np.ndarray:
    """Loewner matrix of first divided differences of f = max(.,0)  (Eq. 10), written so that no
    difference of close eigenvalues is formed: both > 0 -> 1; both <= 0 -> 0 (f'(0) := 0, reading A11);
    mixed signs -> max(li,lj) / (|li| + |lj|)  [= (f(lj)-f(li))/(lj-li) when the signs differ]."""
    li, lj = lam[:, None], lam[None, :]
    pos_i, pos_j = li > 0.0, lj > 0.0
    both = pos_i & pos_j
    mixed = pos_i ^ pos_j
    den = np.abs(li) + np.abs(lj)
    with np.errstate(divide="ignore", invalid="ignore"):
        mix = np.where(mixed, np.maximum(li, lj) / np.where(den > 0.0, den, 1.0), 0.0)
    return np.where(both, 1.0, mix)


def loewner_literal(lam: np.ndarray) -> np.ndarray:
    """Eq. 10 (L116) exactly as printed: (f(lj)-f(li))/(lj-li) if li != lj else f'(li)."""
    f = np.maximum(lam, 0.0)
    p = lam.size
    L = np.empty((p, p))
    for i in range(p):
        for j in range(p):
            if lam[i] != lam[j]:
                L[i, j] = (f[j] - f[i]) / (lam[j] - lam[i])
            else:
                L[i, j] = 1.0 if lam[i] > 0.0 else 0.0
    return L


def dk_vjp_matrix(U: np.ndarray, lam: np.ndarray, Tbar: np.ndarray) -> np.ndarray:
    """Eq. 9 (L112): Sbar = U (L o (U' Tbar U)) U'."""
    C = U.T @ Tbar @ U
    return U @ (loewner_relu(lam) * C) @ U.T


def vjp_psd(w, aux, G):
    lam, U = aux
    Gm = smat(G)  # svec is an isometry, so the svec-space VJP is svec(DK(smat G))
    Sbar = dk_vjp_matrix(U, lam, Gm)
    return svec(0.5 * (Sbar + Sbar.T))


def naive_eig_vjp_matrix(U: np.ndarray, lam: np.ndarray, Tbar: np.ndarray) -> np.ndarray:
    """Eq. 8 (L106), the rule autograd applies to T = U f(Lambda) U' through (U, Lambda):
    Ubar = 2 Tbar U f(Lambda), Lambda_bar = f'(lam) o diag(U' Tbar U), F_ij = 1/(lam_j - lam_i).
    Negative control only: divides by eigenvalue gaps."""
    f = np.maximum(lam, 0.0)
    fp = (lam > 0.0).astype(float)
    Tb = 0.5 * (Tbar + Tbar.T)
    Ubar = 2.0 * Tb @ U * f[None, :]
    Lbar = np.diag(fp * np.einsum("ij,ij->j", U, Tb @ U))
    with np.errstate(divide="ignore", invalid="ignore"):
        F = 1.0 / (lam[None, :] - lam[:, None])
    np.fill_diagonal(F, 0.0)
    inner = F * (U.T @ Ubar)
    Sb = U @ (Lbar + inner) @ U.T
    return 0.5 * (Sb + Sb.T)


# ---------------------------------------------------------------------------------------------
# product cone
# ---------------------------------------------------------------------------------------------
_PROJ = {ZERO: proj_zero, NONNEG: proj_nonneg, SOC: proj_soc, PSD: proj_psd}
_VJP = {ZERO: vjp_zero, NONNEG: vjp_nonneg, SOC: vjp_soc, PSD: vjp_psd}


def cone_rows(kind, dim):
    return dim * (dim + 1) // 2 if kind == PSD else dim


def project(w: np.ndarray, cones):
    """Pi_K(w) for K = product of `cones` tiling w in order. Returns (s_plus, aux list)."""
    out = np.empty_like(w)
    aux = []
    o = 0
    for kind, dim in cones:
        r = cone_rows(kind, dim)
        out[o:o + r], a = _PROJ[kind](w[o:o + r])
        aux.append(a)
        o += r
    assert o == w.size
    return out, aux


def project_vjp(w: np.ndarray, cones, aux, G: np.ndarray) -> np.ndarray:
    out = np.empty_like(G)
    o = 0
    for (kind, dim), a in zip(cones, aux):
        r = cone_rows(kind, dim)
        out[o:o + r] = _VJP[kind](w[o:o + r], a, G[o:o + r])
        o += r
    return out


def in_cone(kind, dim, v, tol=1e-9):
    if kind == ZERO:
        return np.all(np.abs(v) <= tol)
    if kind == NONNEG:
        return np.all(v >= -tol)
    if kind == SOC:
        return np.linalg.norm(v[1:]) <= v[0] + tol
    return np.linalg.eigvalsh(smat(v)).min() >= -tol


def in_dual_cone(kind, dim, v, tol=1e-9):
    if kind == ZERO:
        return True  # dual of {0} is everything
    return in_cone(kind, dim, v, tol)  # nonneg, SOC, PSD are self-dual

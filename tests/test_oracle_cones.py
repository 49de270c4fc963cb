"""Pins for oracle/cones.py against what the paper and the mathematics fix (no GPU, no CUDA path)."""
import os

import numpy as np
import pytest

from oracle import cones as C
from oracle.fd import central_diff_jvp


def _rand_sym(rng, p):
    X = rng.standard_normal((p, p))
    return 0.5 * (X + X.T)


def _rand_orth(rng, p):
    Q, R = np.linalg.qr(rng.standard_normal((p, p)))
    return Q * np.sign(np.diag(R))


# ---- svec / smat -------------------------------------------------------------------------------
def test_svec_layout_and_isometry():
    X = np.array([[1.0, 2.0, 4.0], [2.0, 3.0, 5.0], [4.0, 5.0, 6.0]])
    r2 = np.sqrt(2.0)
    # upper triangle, column by column, off-diagonals * sqrt2 (reading A3)
    np.testing.assert_allclose(C.svec(X), [1.0, 2 * r2, 3.0, 4 * r2, 5 * r2, 6.0])
    np.testing.assert_allclose(C.smat(C.svec(X)), X)
    rng = np.random.default_rng(0)
    A, B = _rand_sym(rng, 6), _rand_sym(rng, 6)
    assert abs(C.svec(A) @ C.svec(B) - np.trace(A @ B)) < 1e-12


# ---- projections: idempotence, Moreau, hand cases ------------------------------------------------
CONES = [(C.ZERO, 4), (C.NONNEG, 5), (C.SOC, 1), (C.SOC, 2), (C.SOC, 6), (C.PSD, 1), (C.PSD, 2), (C.PSD, 7)]


@pytest.mark.parametrize("kind,dim", CONES)
def test_projection_idempotent_and_moreau(kind, dim):
    rng = np.random.default_rng(10 * kind + dim)
    r = C.cone_rows(kind, dim)
    for trial in range(20):
        w = rng.standard_normal(r) * 10.0 ** rng.integers(-2, 3)
        s, _ = C.project(w, [(kind, dim)])
        s2, _ = C.project(s, [(kind, dim)])
        scale = max(1.0, np.abs(w).max())
        np.testing.assert_allclose(s2, s, atol=1e-12 * scale)                 # idempotence
        assert C.in_cone(kind, dim, s, tol=1e-10 * scale)                       # s in K
        d = w - s                                                              # = Pi_{K polar}(w)
        assert C.in_dual_cone(kind, dim, -d, tol=1e-10 * scale)                 # -(w - Pi(w)) in K*
        assert abs(s @ d) <= 1e-10 * scale ** 2                                # <Pi(w), w - Pi(w)> = 0
        # Moreau: w = Pi_K(w) + Pi_{K polar}(w), Pi_{K polar}(w) = -Pi_{K*}(-w)
        if kind != C.ZERO:
            pol, _ = C.project(-w, [(kind, dim)])
            np.testing.assert_allclose(s - pol, w, atol=1e-11 * scale)


def test_soc_hand_cases():
    np.testing.assert_allclose(C.proj_soc(np.array([2.0, 1.0, 1.0]))[0], [2.0, 1.0, 1.0])        # inside
    np.testing.assert_allclose(C.proj_soc(np.array([-2.0, 1.0, 1.0]))[0], [0.0, 0.0, 0.0])       # polar
    np.testing.assert_allclose(C.proj_soc(np.array([0.0, 3.0, 4.0]))[0], [2.5, 1.5, 2.0])        # boundary
    np.testing.assert_allclose(C.proj_soc(np.zeros(3))[0], np.zeros(3))
    # (0,0) maps to itself with J = I (reading A4: first test, with <=)
    np.testing.assert_allclose(C.vjp_soc(np.zeros(3), None, np.array([1.0, 2.0, 3.0])), [1.0, 2.0, 3.0])


def test_psd_projection_identities():
    rng = np.random.default_rng(3)
    for p in (2, 5, 12):
        S = _rand_sym(rng, p)
        T = C.smat(C.proj_psd(C.svec(S))[0])
        lam = np.linalg.eigvalsh(S)
        np.testing.assert_allclose(np.linalg.eigvalsh(T), np.sort(np.maximum(lam, 0)), atol=1e-12)
        Tm = C.smat(C.proj_psd(C.svec(-S))[0])
        np.testing.assert_allclose(T - Tm, S, atol=1e-12)                       # Pi(S) - Pi(-S) = S
        # Pi(S) = (S + |S|)/2 with |S| = sqrt(S^2) from an independent route
        lam2, Q = np.linalg.eigh(S @ S)
        absS = (Q * np.sqrt(np.maximum(lam2, 0))) @ Q.T
        np.testing.assert_allclose(T, 0.5 * (S + absS), atol=1e-8)


# ---- VJPs against central differences ---------------------------------------------------------
@pytest.mark.parametrize("kind,dim", [(C.NONNEG, 5), (C.SOC, 2), (C.SOC, 6), (C.PSD, 2), (C.PSD, 6)])
def test_vjp_matches_central_differences(kind, dim):
    rng = np.random.default_rng(100 + 10 * kind + dim)
    r = C.cone_rows(kind, dim)
    F = lambda w: C.project(w, [(kind, dim)])[0]
    hits = set()
    for trial in range(30):
        w = rng.standard_normal(r)
        if kind == C.SOC and trial % 3 == 0:
            w[0] = np.linalg.norm(w[1:]) * rng.choice([2.0, -2.0, 0.3])
        s, aux = C.project(w, [(kind, dim)])
        if kind == C.SOC:
            hits.add(aux[0])
        G, v = rng.standard_normal(r), rng.standard_normal(r)
        vjp = C.project_vjp(w, [(kind, dim)], aux, G)
        jvp = central_diff_jvp(F, w, v, h=1e-6)
        assert abs(vjp @ v - G @ jvp) <= 2e-7 * (1 + abs(G @ jvp))             # <J'G, v> = <G, Jv>
    if kind == C.SOC:
        assert hits == {0, 1, 2}


def _load_spectrum(golden_dir):
    with open(os.path.join(golden_dir, "dk_repeated_spectrum.txt")) as f:
        rows = [l for l in f if l.strip() and not l.startswith("#")]
    return np.array([float(t) for t in rows[0].split()])


def test_dk_finite_and_correct_at_exactly_repeated_eigenvalues(golden_dir):
    lam = _load_spectrum(golden_dir)
    p = lam.size
    rng = np.random.default_rng(7)
    Q = _rand_orth(rng, p)
    S = (Q * lam) @ Q.T
    S = 0.5 * (S + S.T)
    lam_e, U = np.linalg.eigh(S)
    Tbar = _rand_sym(rng, p)
    dk = C.dk_vjp_matrix(U, lam_e, Tbar)
    assert np.all(np.isfinite(dk))
    F = lambda s: C.proj_psd(s)[0]
    for trial in range(6):
        V = _rand_sym(rng, p)
        jvp = central_diff_jvp(F, C.svec(S), C.svec(V), h=1e-6)
        assert abs(np.sum(dk * V) - C.svec(Tbar) @ jvp) < 5e-8
    # same divided differences as Eq. 10 typed literally, on the EXACT spectrum (ties hit f')
    np.testing.assert_allclose(C.loewner_relu(lam), C.loewner_literal(lam), atol=1e-15)
    # negative control: Eq. 8 on the exact spectrum divides by zero gaps (L108)
    with np.errstate(all="ignore"):
        naive = C.naive_eig_vjp_matrix(Q, lam, Tbar)
    assert not np.all(np.isfinite(naive))


def test_dk_agrees_with_naive_rule_when_gaps_are_large():
    rng = np.random.default_rng(11)
    p = 6
    lam = np.array([-3.0, -1.5, -0.4, 0.7, 1.9, 3.2])
    Q = _rand_orth(rng, p)
    Tbar = _rand_sym(rng, p)
    np.testing.assert_allclose(C.dk_vjp_matrix(Q, lam, Tbar), C.naive_eig_vjp_matrix(Q, lam, Tbar), atol=1e-11)


def test_dk_special_cases():
    rng = np.random.default_rng(5)
    p = 5
    Q = _rand_orth(rng, p)
    Tbar = _rand_sym(rng, p)
    pos = np.array([0.5, 1.0, 1.0, 2.0, 3.0])
    np.testing.assert_allclose(C.dk_vjp_matrix(Q, pos, Tbar), Tbar, atol=1e-12)     # S > 0: identity
    np.testing.assert_allclose(C.dk_vjp_matrix(Q, -pos, Tbar), 0 * Tbar, atol=1e-12)  # S < 0: zero
    L = C.loewner_relu(np.array([-2.0, 0.0, 0.0, 1.0, 1.0]))
    assert np.all((L >= 0) & (L <= 1)) and np.all(np.isfinite(L))                      # f' in [0,1] (L119)
    assert L[1, 2] == 0.0 and L[3, 4] == 1.0 and abs(L[0, 3] - 1.0 / 3.0) < 1e-15


@pytest.mark.parametrize("delta", [1.0, 1e-2, 1e-4, 1e-6, 1e-8, 1e-10])
def test_dk_error_independent_of_gap_eq13(delta):
    """PAPER.md Eq. 13 (L270-277): n=40, two clusters at +-delta/2, spread delta*1e-3; the DK error vs a
    finite-difference reference 'does not depend on delta'. FD step is scaled with delta so that the
    reference itself stays valid (no eigenvalue crosses zero inside the stencil)."""
    n = 40
    rng = np.random.default_rng(13)
    lam = np.concatenate([-delta / 2 + rng.uniform(-1, 1, n // 2) * delta * 1e-3,
                          +delta / 2 + rng.uniform(-1, 1, n // 2) * delta * 1e-3])
    Q = _rand_orth(rng, n)
    S = (Q * lam) @ Q.T
    S = 0.5 * (S + S.T)
    lam_e, U = np.linalg.eigh(S)
    Tbar = _rand_sym(rng, n)
    dk = C.dk_vjp_matrix(U, lam_e, Tbar)
    V = _rand_sym(rng, n)
    V /= np.linalg.norm(V, 2)
    F = lambda s: C.proj_psd(s)[0]
    jvp = central_diff_jvp(F, C.svec(S), C.svec(V), h=delta * 1e-4)
    ref = C.svec(Tbar) @ jvp
    assert abs(np.sum(dk * V) - ref) <= 1e-6 * max(1.0, abs(ref))

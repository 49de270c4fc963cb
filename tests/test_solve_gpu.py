"""cdu_solve: vanilla COSMO to tolerance with residual-balancing rho (the baseline workload of PAPER.md Table 1;
SURVEY.md 8(f) F3, scalar-rho part). Pinned against the closed forms the oracle is pinned against (BASELINE.json north_star):
max-cut(K_n) = n^2/4, theta(C5) = sqrt 5, and against the oracle's own fixed-rho iteration."""
import numpy as np
import pytest

import workloads as W
from workloads.generators import complete_graph, cycle_graph, maxcut_problem, lovasz_problem, _round_problem
import parity_util as PU
from oracle import cosmo_oracle as O

pytestmark = pytest.mark.gpu


def _handle(problems, dtype, K_max):
    import paper_2606_13825_b200 as cdu
    return cdu.cdu_create(W.pack_batch(problems, dtype), K_max=K_max)


def test_fixed_rho_chunks_equal_the_oracle_iteration():
    """adapt_rho = 0, 4 chunks of 5 steps = 20 oracle steps at rho = 0.5 (fp64: the chunk hand-over keeps the fp64 state)."""
    rng = np.random.default_rng(3)
    probs = [W.random_mixed_problem(rng, n=7) for _ in range(3)]
    h = _handle(probs, "f64", 5)
    x, s, y, iters, res = h.solve(20, 5, 1e-30, rho0=0.5, alpha=1.6, adapt_rho=False)
    off_n = np.cumsum([0] + [p.n for p in probs]); off_m = np.cumsum([0] + [p.m for p in probs])
    for b, pr in enumerate(probs):
        un = O.unroll(pr, 20, np.full(20, 0.5), np.full(20, 1.6), 1e-6, keep_tape=False)
        assert PU.nrm_err(x.cpu().numpy()[off_n[b]:off_n[b + 1]], un.xs[-1]) <= 1e-9
        assert PU.nrm_err(y.cpu().numpy()[off_m[b]:off_m[b + 1]], un.ys[-1]) <= 1e-9
    assert np.all(iters == -20)          # eps = 1e-30 is never met
    h.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_solver_reaches_the_closed_form_values(dtype):
    probs = [_round_problem(maxcut_problem(complete_graph(n)), dtype) for n in (4, 5, 8)] + [_round_problem(lovasz_problem(cycle_graph(5)), dtype)]
    want = [4.0, 6.25, 16.0, np.sqrt(5.0)]
    h = _handle(probs, dtype, 25)
    x, s, y, iters, res = h.solve(5000, 25, 1e-5 if dtype == "f64" else 1e-4, rho0=0.1, alpha=1.6, adapt_rho=True)
    assert np.all(iters > 0), (iters, res)
    off_n = np.cumsum([0] + [p.n for p in probs])
    xs = x.double().cpu().numpy()
    for b, pr in enumerate(probs):
        val = -(pr.q @ xs[off_n[b]:off_n[b + 1]])
        assert abs(val - want[b]) <= (2e-4 if dtype == "f64" else 2e-3) * want[b], (b, val, want[b], iters[b])
    h.close()


def test_equality_rows_on_a_scaled_penalty():
    """eq_scale = 1e3 (COSMO / OSQP practice): the equality rows run on 1e3 rho_b through the per-row mode; the
    solver reaches the same closed-form values, and Lovasz theta(C5), whose edge constraints are equalities, in fewer iterations."""
    probs = [maxcut_problem(complete_graph(5)), lovasz_problem(cycle_graph(5))]
    want = [6.25, np.sqrt(5.0)]
    its = {}
    for es in (1.0, 1e3):
        h = _handle(probs, "f64", 25)
        x, s, y, iters, res = h.solve(20000, 25, 1e-6, rho0=0.1, alpha=1.6, adapt_rho=True, eq_scale=es)
        assert np.all(iters > 0), (es, iters, res)
        off_n = np.cumsum([0] + [p.n for p in probs]); xs = x.cpu().numpy()
        for b, pr in enumerate(probs):
            assert abs(-(pr.q @ xs[off_n[b]:off_n[b + 1]]) - want[b]) <= 1e-4 * want[b], (es, b)
        its[es] = iters.copy()
        h.close()
    print("iterations to 1e-6, eq_scale 1 vs 1e3:", its)

"""Host-side checks of the seeded input generators and the batched-CSR packing (no GPU)."""
import numpy as np

import workloads as W
from workloads.generators import ZERO, PSD, SOC
from oracle import cosmo_oracle as O


def test_config_shapes_match_survey_table():
    wl = W.make_config(1)
    assert wl.batch == 4 and wl.K == 20 and wl.dtype == "f64"
    pr = wl.problems[0]
    assert (pr.n, pr.m, pr.A.nnz, pr.P.nnz) == (55, 65, 65, 0) and pr.cones == [(ZERO, 10), (PSD, 10)]
    assert np.all((wl.rho >= 0.01) & (wl.rho <= 10.0)) and np.all(wl.alpha == 1.6) and wl.sigma == 1e-6
    wl2 = W.make_config(2, batch=2)
    assert (wl2.problems[0].n, wl2.problems[0].m) == (1275, 1325) and wl2.dtype == "f32"
    wl3 = W.make_config(3, batch=1)
    p3 = wl3.problems[0]
    assert (p3.n, p3.m) == (200, 1100) and p3.cones == [(SOC, 11)] * 100 and p3.P.nnz == 40000
    assert 38000 < p3.A.nnz < 42000
    wl4 = W.make_config(4, batch=2)
    p4 = wl4.problems[0]
    assert p4.n == 5050 and p4.m == 5050 + p4.cones[0][1] and 400 < p4.cones[0][1] < 600
    # cfg4 start is dual feasible: r_d(z0) = 0
    rp, rd = O.residuals(p4, wl4.x0[0], wl4.s0[0], wl4.y0[0])
    assert np.abs(rd).max() < 1e-5 and np.abs(rp).max() < 1e-6


def test_fp32_configs_are_pre_rounded():
    wl = W.make_config(3, batch=1, p=20)
    pr = wl.problems[0]
    for v in (pr.A.data, pr.P.data, pr.q, pr.b, wl.rho, wl.alpha):
        assert np.array_equal(v.astype(np.float32).astype(np.float64), v)
    assert abs(pr.P - pr.P.T).max() == 0.0


def test_seeding_is_deterministic():
    a, b = W.make_config(2, batch=2, p=8), W.make_config(2, batch=2, p=8)
    assert np.array_equal(a.problems[1].q, b.problems[1].q) and np.array_equal(a.rho, b.rho)
    assert not np.array_equal(a.problems[0].q, a.problems[1].q)


def test_pack_batch_roundtrip_ragged():
    wl = W.make_config(4, batch=3, p=9)
    pk = W.pack_batch(wl.problems, wl.dtype)
    assert pk["A_val"].dtype == np.float32 and pk["A_colidx"].dtype == np.int32 and pk["A_rowptr"].dtype == np.int64
    assert len({pr.m for pr in wl.problems}) > 1            # ragged m (|E| differs per instance)
    for i, pr in enumerate(wl.problems):
        r0, r1 = pk["row_off"][i], pk["row_off"][i + 1]
        assert r1 - r0 == pr.m and pk["var_off"][i + 1] - pk["var_off"][i] == pr.n
        ptr = pk["A_rowptr"][r0:r1 + 1]
        dense = np.zeros((pr.m, pr.n))
        for r in range(pr.m):
            for e in range(ptr[r], ptr[r + 1]):
                dense[r, pk["A_colidx"][e]] = pk["A_val"][e]
        assert np.array_equal(dense, pr.A.toarray())
        c0, c1 = pk["cone_off"][i], pk["cone_off"][i + 1]
        assert [tuple(c) for c in pk["cones"][c0:c1]] == pr.cones


def test_smooth_schedule_keeps_small_configs_well_conditioned():
    """Acceptance rule of SURVEY.md 8(d): iterates stay bounded and the PSD block is non-degenerate."""
    for cfg, kw in [(2, dict(batch=1, p=12, K=30)), (3, dict(batch=1, p=20, K=40)), (5, dict(batch=1, p=16, K=30))]:
        wl = W.make_config(cfg, **kw)
        pr = wl.problems[0]
        un = O.unroll(pr, wl.K, wl.rho, wl.alpha, wl.sigma, wl.x0[0], wl.s0[0], wl.y0[0])
        assert all(np.abs(v).max() < 1e3 for v in un.xs + un.ss + un.ys)
        if cfg != 3:
            fr = [np.mean(t.aux[-1][0] > 0) for t in un.tapes]
            assert sum(0 < f < 1 for f in fr) > len(fr) // 2

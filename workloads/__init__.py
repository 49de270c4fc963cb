"""Seeded synthetic input generators shared by the oracle tests, the GPU parity tests and bench.py.

This package holds *inputs only*: graphs, problem matrices in the conic standard form of
PAPER.md Eq. 1 (L42-48), hyper-parameter schedules, starts and the batched-CSR packing.
It contains none of the method's arithmetic (no ADMM step, no projection, no solver) and is
imported by neither `oracle/` nor the CUDA path for anything but inputs.
"""
from .generators import (  # noqa: F401
    Problem,
    Workload,
    svec_index,
    svec_dim,
    cone_rows,
    maxcut_problem,
    lovasz_problem,
    socp_problem,
    erdos_renyi,
    ar1_rho_schedule,
    make_config,
    make_fig2,
    lyapunov_lmi_problem,
    robust_mpc_problem,
    clustered_spectrum_matrix,
    pack_batch,
    CONFIG_NAMES,
    BASE_SEED,
    random_mixed_problem,
    fig2_linear_problem,
)

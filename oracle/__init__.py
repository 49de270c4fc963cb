"""fp64 CPU oracle for the unrolled COSMO hot path of arxiv/paper_2606_13825.

TEST INFRASTRUCTURE - not product code. Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s
`cpu_baseline` / `--impl reference` legs may import it. It shares no code with, and never imports,
`paper_2606_13825_b200` (the CUDA path).
"""

"""No-GPU checks of the boundary: the C-ABI library builds/loads and exports every symbol include/cdu.h declares;
calls that would compute fail loudly without a device (no CPU fallback)."""
import os
import re

import numpy as np
import pytest

import paper_2606_13825_b200 as cdu
from paper_2606_13825_b200 import build as cbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    cbuild.build()
    return cdu.load_library()


def _declared_symbols():
    txt = open(os.path.join(ROOT, "include", "cdu.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(cdu_[a-z0-9_]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol(lib):
    decl = _declared_symbols()
    assert {"cdu_create", "cdu_forward", "cdu_backward", "cdu_destroy"} <= set(decl)
    for name in decl:
        assert hasattr(lib, name), f"{name} declared in include/cdu.h but not exported"
    assert set(decl) == set(cdu.EXPORTED_SYMBOLS)
    assert b"sm_100a" in lib.cdu_version()


def test_no_torch_types_in_the_header():
    txt = open(os.path.join(ROOT, "include", "cdu.h")).read()
    assert "torch" not in txt.lower() and "at::" not in txt and 'extern "C"' in txt


def test_library_is_built_for_sm_100a_only():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", cdu.LIB_PATH], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_product_path_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import workloads as W
    wl = W.make_config(1)
    with pytest.raises(cdu.CduError):
        cdu.cdu_create(W.pack_batch(wl.problems, wl.dtype), K_max=wl.K)


def test_product_does_not_import_the_oracle():
    """The two sides share no code and neither imports the other (only `workloads` serves both)."""
    imp = re.compile(r"^\s*(from|import)\s+oracle\b|#include\s*[<\"].*oracle|[\"']oracle[/\"']", re.M)
    pkg = os.path.join(ROOT, "paper_2606_13825_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not imp.search(open(os.path.join(dirpath, f)).read()), f
    imp2 = re.compile(r"^\s*(from|import)\s+paper_2606_13825_b200\b|ctypes|libcdu", re.M)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert not imp2.search(open(os.path.join(ROOT, "oracle", f)).read()), f
    for f in os.listdir(os.path.join(ROOT, "workloads")):
        if f.endswith(".py"):
            src = open(os.path.join(ROOT, "workloads", f)).read()
            assert not imp.search(src) and not imp2.search(src), f


def test_shard_indices_cover_and_balance():
    from paper_2606_13825_b200.sharding import shard_indices
    for n, w in [(8, 2), (9, 2), (5, 4), (3, 8)]:
        parts = [shard_indices(n, r, w) for r in range(w)]
        assert sorted(sum(parts, [])) == list(range(n))
        assert max(map(len, parts)) - min(map(len, parts)) <= 1

"""-m "not gpu": the C-ABI library loads and exports every symbol include/wpccc.h declares; compute calls fail loudly
without a CUDA device (no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def wp():
    import __graft_entry__
    __graft_entry__.build()
    import paper_2403_04252_b200 as wp
    return wp


def test_header_symbols_are_exported(wp):
    text = open(wp.HEADER_PATH).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    declared = set(re.findall(r"\b(wpccc_[a-z0-9_]+)\s*\(", text))
    assert declared, "no declarations found in wpccc.h"
    lib = ctypes.CDLL(wp.LIB_PATH)
    for name in sorted(declared):
        assert hasattr(lib, name), "libwpccc.so does not export %s" % name
    assert declared == set(wp.EXPORTS)


def test_basis_bytes_and_argument_checks_run_on_host(wp):
    from wpccc_inputs.configs import bound_only_centre
    from wpccc_inputs import make_problem
    T = bound_only_centre(1.0, [(1, 0), (2, 0), (2, 1)], 200, 0.1)
    prob = make_problem([T], 1.0, 200, 0.1, 2)
    cs, quad, keep = wp._marshal(prob)
    n = wp._lib.wpccc_basis_bytes(1, cs, 200, 2, None)
    assert n > 3 * 6 // 2 * 224 * 8          # at least the pair-product matrix
    assert wp._lib.wpccc_basis_bytes(3, cs, 200, 2, None) == 0
    assert wp._lib.wpccc_basis_bytes(1, cs, 200, 99, None) == 0
    assert b"lambda_max" in wp._lib.wpccc_last_error()


def test_no_cpu_fallback(wp):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from wpccc_inputs.configs import bound_only_centre
    from wpccc_inputs import make_problem
    T = bound_only_centre(1.0, [(1, 0)], 100, 0.1)
    with pytest.raises(wp.WpcccError):
        wp.setup_basis(make_problem([T], 1.0, 100, 0.1, 0))
    with pytest.raises(wp.WpcccError):
        wp.fp64_peak(0)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2403_04252_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "oracle/" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_2403_04252_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "``paper_2403_04252_b200/``", "") or f == "__init__.py"

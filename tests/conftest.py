import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")
    config.addinivalue_line("markers", "slow: full-size configuration (still part of -m gpu)")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)


@pytest.fixture(scope="session")
def orc():
    import oracle
    oracle.lib()
    return oracle


@pytest.fixture(scope="session")
def small_tables(orc):
    """Oracle-built tables, small enough for the CPU suite (a few seconds)."""
    p = orc.TableParams(qs_chi_min=1e-3, qs_chi_max=1e3, qs_n_chi=25, qs_xi_min=1e-12, qs_n_xi=49,
                        bw_chi_min=2e-2, bw_chi_max=1e3, bw_n_chi=25, bw_n_xi=49)
    return orc.build_tables(p)


def golden(name):
    """rows of a tests/golden/*.txt fixture: '#' comments, whitespace-separated fields"""
    rows = []
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append(line.split())
    return rows

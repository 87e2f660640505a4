import os
import sys

import pytest

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def cuda_lib():
    """The C-ABI library through its Python binding; fails loudly if it cannot run."""
    import torch
    from paper_1807_08116_b200 import binding
    assert torch.cuda.is_available(), "gpu-marked test started without a CUDA device"
    binding.load()
    return binding


def pytest_terminal_summary(terminalreporter):
    """Reach of the parity-tolerance floors (tests/parity_util.py), printed whatever the capture mode."""
    import parity_util
    if not parity_util.REPORT:
        return
    tr = terminalreporter
    tr.write_sep("-", "parity report: error and reach of the tolerance floors per compared array")
    tr.write_line(f"{'array':58s} {'n':>8s} {'max err':>9s} {'median':>9s} {'bar':>7s} {'med.floor':>12s} {'gross floor':>14s}")
    for r in parity_util.REPORT:
        tr.write_line(f"{r['what'][:58]:58s} {r['n']:8d} {r['max_err']:9.2e} {r['median_err']:9.2e} {r['max_tol']:7.0e} "
                      f"{r['median_floor_touched']:5d} x{r['median_floor_loosening']:<5.1f} "
                      f"{r['gross_floor_touched']:5d} x{r['gross_floor_loosening']:<7.1f}")

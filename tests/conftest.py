import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


def mixed_err(got, ref):
    """DESIGN.md reading R12: max_j |got_j - ref_j| / max(|ref_j|, rms(ref))."""
    import numpy as np
    got = np.asarray(got, dtype=np.float64).ravel()
    ref = np.asarray(ref, dtype=np.float64).ravel()
    rms = float(np.sqrt(np.mean(ref ** 2))) if ref.size else 0.0
    den = np.maximum(np.abs(ref), rms)
    den[den == 0] = 1.0
    return float(np.max(np.abs(got - ref) / den)) if ref.size else 0.0


@pytest.fixture
def hsp_options():
    """Plan-time options of libhsp.so (hsp_set_option with state NULL) for the chains a test creates; restored after."""
    import paper_1608_04329_b200 as hsp
    hsp.reset_options()
    yield hsp.set_option
    hsp.reset_options()

import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def golden_lines(name):
    """Non-comment, non-empty lines of tests/golden/<name>, split on whitespace."""
    with open(os.path.join(GOLDEN, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


@pytest.fixture(scope="session")
def oracle_uniforms():
    """uniform_source for workloads.md_system backed by the oracle's sequential rand48."""
    import oracle

    def src(seed48, ndraws):
        out, _ = oracle.rand48_fill([seed48], ndraws, kind=2)
        return out[0]
    return src


@pytest.fixture(scope="session", autouse=True)
def torch_side_stream():
    """GPU tests run with a non-default PyTorch stream current, so that the binding's default plumbing
    (PyTorch's caching allocator and current stream, north_star: "PyTorch is used only for device memory
    and streams") is the path every parity test exercises.  No effect without a device."""
    try:
        import torch
    except ImportError:
        yield
        return
    if not torch.cuda.is_available():
        yield
        return
    with torch.cuda.stream(torch.cuda.Stream()):
        yield

import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.fixture(autouse=True)
def poison_native_fields(request, monkeypatch):
    """Every native field a GPU test allocates starts as NaN, so an output element a kernel leaves
    unwritten (or a launch that does not run) fails the parity check instead of inheriting a previous
    result from the caching allocator."""
    if request.node.get_closest_marker("gpu") is None:
        yield
        return
    import paper_2211_13719_b200 as mrhs
    plain = mrhs.empty_field

    def poisoned(*args, **kwargs):
        return plain(*args, **kwargs).fill_(float("nan"))

    plain_export = mrhs.field_export

    def poisoned_export(dims, ncomp, nrhs, parity, native, canonical=None, stream=None):
        if canonical is None:
            import torch
            nsites = int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3]) // (1 if parity == mrhs.FULL else 2)
            canonical = torch.full((nsites, ncomp, nrhs), float("nan"), dtype=torch.complex64, device=native.device)
        return plain_export(dims, ncomp, nrhs, parity, native, canonical, stream)

    monkeypatch.setattr(mrhs, "empty_field", poisoned)
    monkeypatch.setattr(mrhs, "field_export", poisoned_export)
    yield

"""The allocation-free entry point (mrhs_inner_products_noalloc, include/mrhs.h): simultaneous inner products with the
per-block partial sums in a static __device__ array of the library instead of stream-ordered scratch, for callers that
cannot call cudaMalloc (graph capture, serving loops).  Checked against the existing path (mrhs_inner_products) on two
calls in a row; the two paths run the same kernels on the same grid, so within the tolerance of the inner-product tests
(1e-10 relative) they are in fact bit-identical.  Collected last on purpose (the suite runs with pytest -x)."""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():
    pytest.skip("needs a CUDA device", allow_module_level=True)

import paper_2211_13719_b200 as mrhs   # noqa: E402
from gpu_common import dev, host       # noqa: E402

INNER_TOL = 1e-10     # tests/test_gpu_fine.py::test_inner_products_match_oracle


def _fields(dims, ncomp, nrhs, parity, seed):
    V = int(np.prod(dims)) // (1 if parity == mrhs.FULL else 2)
    shape = (ncomp,) if ncomp != 12 else (4, 3)
    rng = np.random.default_rng([seed, nrhs])
    x = (rng.standard_normal((V,) + shape + (nrhs,)) + 1j * rng.standard_normal((V,) + shape + (nrhs,))).astype(np.complex64)
    y = (rng.standard_normal((V,) + shape + (nrhs,)) + 1j * rng.standard_normal((V,) + shape + (nrhs,))).astype(np.complex64)
    return mrhs.field_import(dims, ncomp, nrhs, parity, dev(x)), mrhs.field_import(dims, ncomp, nrhs, parity, dev(y))


def test_inner_products_noalloc_matches_the_allocating_path_twice_in_a_row():
    # first call: 48 right-hand sides fill 8 x SMs x 48 partial sums of the static array; second call: a different lattice,
    # component count and N_rhs (odd: the one-RHS element kernel), which finds the first call's partial sums in the array
    cases = [([16, 4, 6, 4], 12, 48, mrhs.FULL, 7), ([6, 4, 2, 6], 40, 3, mrhs.ODD, 8)]
    inputs = [(c, _fields(*c)) for c in cases]
    want = [host(mrhs.inner_products(c[0], c[1], c[2], c[3], dx, dy)) for c, (dx, dy) in inputs]
    results = [torch.full((c[2],), float("nan"), dtype=torch.complex128, device="cuda") for c in cases]
    torch.cuda.synchronize()
    for (c, (dx, dy)), res in zip(inputs, results):      # back to back on one stream, no synchronisation in between
        mrhs.inner_products_noalloc(c[0], c[1], c[2], c[3], dx, dy, res)
    torch.cuda.synchronize()
    for res, w in zip(results, want):
        got = host(res)
        assert np.all(np.isfinite(got.real)) and np.all(np.isfinite(got.imag))
        assert np.max(np.abs(got - w) / np.abs(w)) < INNER_TOL, (got, w)
        assert np.array_equal(got, w)       # same kernels, same grid, same summation order
    # and the first case once more, after the smaller call has overwritten part of the array
    c, (dx, dy) = inputs[0]
    res = torch.full((c[2],), float("nan"), dtype=torch.complex128, device="cuda")
    mrhs.inner_products_noalloc(c[0], c[1], c[2], c[3], dx, dy, res)
    torch.cuda.synchronize()
    assert np.max(np.abs(host(res) - want[0]) / np.abs(want[0])) < INNER_TOL


def test_inner_products_noalloc_allocates_nothing():
    """Device memory in use (driver's view, cudaMemGetInfo) and torch's allocator are unchanged by the calls."""
    dims, ncomp, nrhs, parity = [8, 4, 6, 4], 12, 12, mrhs.FULL
    dx, dy = _fields(dims, ncomp, nrhs, parity, 9)
    res = torch.empty(nrhs, dtype=torch.complex128, device="cuda")
    mrhs.inner_products_noalloc(dims, ncomp, nrhs, parity, dx, dy, res)      # first call on the device: symbol address lookup
    torch.cuda.synchronize()
    rt = ctypes.CDLL("libcudart.so.12")
    free0, free1, total = ctypes.c_size_t(), ctypes.c_size_t(), ctypes.c_size_t()
    assert rt.cudaMemGetInfo(ctypes.byref(free0), ctypes.byref(total)) == 0
    reserved0 = torch.cuda.memory_reserved()
    for _ in range(5):
        mrhs.inner_products_noalloc(dims, ncomp, nrhs, parity, dx, dy, res)
    torch.cuda.synchronize()
    assert rt.cudaMemGetInfo(ctypes.byref(free1), ctypes.byref(total)) == 0
    assert free1.value == free0.value, (free0.value, free1.value)
    assert torch.cuda.memory_reserved() == reserved0


def test_inner_products_noalloc_rejects_sizes_beyond_the_static_scratch():
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    nrhs = 131072 // (8 * sms) + 1          # one right-hand side past the limit stated in include/mrhs.h
    if nrhs > 256:
        pytest.skip("this device has too few SMs for the limit to bind below the 256 right-hand sides the entry accepts")
    dims, ncomp = [2, 2, 2, 2], 24
    x = torch.zeros(mrhs.field_bytes(dims, ncomp, nrhs, False) // 4, dtype=torch.float32, device="cuda")
    res = torch.full((nrhs,), 5.0, dtype=torch.complex128, device="cuda")
    with pytest.raises(mrhs.MrhsError) as e:
        mrhs.inner_products_noalloc(dims, ncomp, nrhs, mrhs.FULL, x, x, res)
    assert e.value.status == mrhs.ERR_UNSUPPORTED
    assert "static scratch" in str(e.value)
    torch.cuda.synchronize()
    assert bool((res == 5.0).all())          # nothing was launched
    # the largest accepted N_rhs goes through and agrees with the allocating path
    nrhs -= 1
    x = torch.randn(mrhs.field_bytes(dims, ncomp, nrhs, False) // 4, dtype=torch.float32, device="cuda")
    res = torch.empty(nrhs, dtype=torch.complex128, device="cuda")
    mrhs.inner_products_noalloc(dims, ncomp, nrhs, mrhs.FULL, x, x, res)
    torch.cuda.synchronize()
    assert np.array_equal(host(res), host(mrhs.inner_products(dims, ncomp, nrhs, mrhs.FULL, x, x)))

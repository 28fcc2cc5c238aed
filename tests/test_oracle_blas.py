"""Pins for the oracle's simultaneous inner products (CPU only):
against numpy.vdot column by column (library routine), sesquilinearity, <x, x> = ||x||^2 real and positive,
and column independence."""
import numpy as np

import oracle
import synth_inputs as si


def test_inner_products_match_vdot_and_are_sesquilinear():
    V, N = 48, 5
    x = si.spinor_np(V, N, 81).astype(np.complex128)
    y = si.spinor_np(V, N, 82).astype(np.complex128)
    got = oracle.inner_products(x, y)
    for r in range(N):
        assert abs(got[r] - np.vdot(x[..., r].ravel(), y[..., r].ravel())) < 1e-12 * abs(got[r]) + 1e-12
    assert np.max(np.abs(oracle.inner_products(y, x) - np.conj(got))) < 1e-12
    a = 0.3 - 1.1j
    assert np.max(np.abs(oracle.inner_products(a * x, y) - np.conj(a) * got)) < 1e-11
    assert np.max(np.abs(oracle.inner_products(x, a * y) - a * got)) < 1e-11
    nrm = oracle.inner_products(x, x)
    assert np.max(np.abs(nrm.imag)) < 1e-12 and np.all(nrm.real > 0)
    assert np.max(np.abs(nrm.real - np.sum(np.abs(x) ** 2, axis=(0, 1, 2)))) < 1e-10
    # a column of the block result is the single-RHS result
    assert oracle.inner_products(x[..., 2:3], y[..., 2:3])[0] == got[2]

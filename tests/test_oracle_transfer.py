"""Pins for the oracle's intergrid operators (CPU only): against the dense
prolongator matrix of the Galerkin self-check (brute force), adjointness <R f, c> = <f, P c> for an arbitrary basis,
R P = 1 for a block-orthonormal basis, and RHS-column independence."""
import numpy as np
import pytest

import oracle
import synth_inputs as si
from oracle import galerkin, transfer


def _orthonormal_basis(dims, bdims, n_vec, seed):
    """Block-orthonormal basis vectors read back from the dense prolongator (whose columns are the block basis)."""
    V = si.volume(dims)
    phi = np.stack([si.spinor_np(V, 1, seed + k)[..., 0] for k in range(n_vec)]).astype(np.complex128)
    P, cd = galerkin.prolongator(dims, bdims, phi)
    blk, _ = galerkin.block_of_site(dims, bdims)
    Vc, nb = si.volume(cd), 2 * n_vec
    P5 = P.reshape(V, 4, 3, Vc, nb)
    basis = np.zeros((n_vec, V, 4, 3), dtype=np.complex128)
    for k in range(n_vec):
        basis[k][:, 0:2] = np.stack([P5[i, 0:2, :, blk[i], k] for i in range(V)])
        basis[k][:, 2:4] = np.stack([P5[i, 2:4, :, blk[i], n_vec + k] for i in range(V)])
    return basis, P, cd


@pytest.mark.parametrize("dims,bdims,n_vec", [((4, 4, 4, 4), (2, 2, 2, 2), 3), ((8, 4, 4, 4), (4, 2, 2, 2), 2)])
def test_prolong_restrict_match_dense_prolongator(dims, bdims, n_vec):
    basis, P, cd = _orthonormal_basis(dims, bdims, n_vec, 50)
    V, Vc, nb, N = si.volume(dims), si.volume(cd), 2 * n_vec, 3
    vc = si.coarse_vector_np(cd, nb, N, 51).astype(np.complex128)
    f = si.spinor_np(V, N, 52).astype(np.complex128)
    assert np.max(np.abs(transfer.prolong(dims, bdims, basis, vc) - (P @ vc.reshape(Vc * nb, N)).reshape(V, 4, 3, N))) < 1e-13
    assert np.max(np.abs(transfer.restrict(dims, bdims, basis, f) - (P.conj().T @ f.reshape(V * 12, N)).reshape(Vc, nb, N))) < 1e-12
    # R P = 1 for the block-orthonormal basis
    assert np.max(np.abs(transfer.restrict(dims, bdims, basis, transfer.prolong(dims, bdims, basis, vc)) - vc)) < 1e-12
    # a column of the block result is the single-RHS result
    assert np.array_equal(transfer.prolong(dims, bdims, basis, vc[..., 1:2])[..., 0], transfer.prolong(dims, bdims, basis, vc)[..., 1])


def test_restrict_is_the_adjoint_of_prolong_for_any_basis():
    dims, bdims, n_vec, N = (4, 2, 6, 4), (2, 2, 3, 2), 4, 2
    V = si.volume(dims)
    basis = np.stack([si.spinor_np(V, 1, 60 + k)[..., 0] for k in range(n_vec)]).astype(np.complex128)
    cd = [d // b for d, b in zip(dims, bdims)]
    vc = si.coarse_vector_np(cd, 2 * n_vec, N, 61).astype(np.complex128)
    f = si.spinor_np(V, N, 62).astype(np.complex128)
    lhs = oracle.inner_products(transfer.restrict(dims, bdims, basis, f), vc)
    rhs = oracle.inner_products(f, transfer.prolong(dims, bdims, basis, vc))
    assert np.max(np.abs(lhs - rhs)) < 1e-11 * np.max(np.abs(lhs))

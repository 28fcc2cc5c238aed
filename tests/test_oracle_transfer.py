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


# ---- coarse -> coarser intergrid operators
def _dense_coarse_prolongator(fdims, bdims, basis):
    """Brute force: P[(x, c), (B, j)] = phi_k(x)[c] if x lies in block B and c, j = chi n_vec + k have the same chirality."""
    n_vec, Vf, nf = basis.shape
    cd = [d // b for d, b in zip(fdims, bdims)]
    Vc = int(np.prod(cd))
    P = np.zeros((Vf, nf, Vc, 2 * n_vec), dtype=np.complex128)
    X, Y, Z, T = fdims
    for x in range(Vf):
        c4 = [x % X, (x // X) % Y, (x // (X * Y)) % Z, x // (X * Y * Z)]
        B = (c4[0] // bdims[0]) + cd[0] * ((c4[1] // bdims[1]) + cd[1] * ((c4[2] // bdims[2]) + cd[2] * (c4[3] // bdims[3])))
        for c in range(nf):
            chi = 0 if c < nf // 2 else 1
            for k in range(n_vec):
                P[x, c, B, chi * n_vec + k] = basis[k, x, c]
    return P.reshape(Vf * nf, Vc * 2 * n_vec), cd


@pytest.mark.parametrize("fdims,bdims,nf,n_vec", [((4, 4, 2, 4), (2, 2, 2, 2), 6, 4), ((6, 2, 4, 2), (3, 1, 2, 2), 8, 3)])
def test_coarse_level_prolong_restrict(fdims, bdims, nf, n_vec):
    Vf, N = si.volume(fdims), 3
    basis = np.stack([si.coarse_vector_np(fdims, nf, 1, 70 + k)[..., 0] for k in range(n_vec)]).astype(np.complex128)
    P, cd = _dense_coarse_prolongator(fdims, bdims, basis)
    Vc, nb = si.volume(cd), 2 * n_vec
    vc = si.coarse_vector_np(cd, nb, N, 71).astype(np.complex128)
    f = si.coarse_vector_np(fdims, nf, N, 72).astype(np.complex128)
    assert np.max(np.abs(transfer.prolong_coarse(fdims, bdims, basis, vc) - (P @ vc.reshape(Vc * nb, N)).reshape(Vf, nf, N))) < 1e-12
    assert np.max(np.abs(transfer.restrict_coarse(fdims, bdims, basis, f) - (P.conj().T @ f.reshape(Vf * nf, N)).reshape(Vc, nb, N))) < 1e-12
    # adjointness
    lhs = oracle.inner_products(transfer.restrict_coarse(fdims, bdims, basis, f), vc)
    rhs = oracle.inner_products(f, transfer.prolong_coarse(fdims, bdims, basis, vc))
    assert np.max(np.abs(lhs - rhs)) < 1e-11 * np.max(np.abs(lhs))
    # R P = 1 once the columns of P are orthonormal (QR of the dense matrix keeps the block / chirality structure)
    Q, _ = np.linalg.qr(P)
    qb = np.zeros_like(basis)
    blk, _ = galerkin.block_of_site(fdims, bdims)
    Q4 = Q.reshape(Vf, nf, Vc, nb)
    for k in range(n_vec):
        for x in range(Vf):
            qb[k, x, :nf // 2] = Q4[x, :nf // 2, blk[x], k]
            qb[k, x, nf // 2:] = Q4[x, nf // 2:, blk[x], n_vec + k]
    assert np.max(np.abs(transfer.restrict_coarse(fdims, bdims, qb, transfer.prolong_coarse(fdims, bdims, qb, vc)) - vc)) < 1e-12


def test_coarse_level_operators_reduce_to_the_fine_level_ones_for_twelve_components():
    """With n_f = 12 and component index 3 spin + colour the coarse-level definition IS the fine-level one (chirality 0 =
    spins {0,1} = components 0..5): pins the new functions against the already pinned prolong / restrict."""
    dims, bdims, n_vec, N = (4, 4, 4, 2), (2, 2, 2, 2), 3, 2
    V = si.volume(dims)
    basis = np.stack([si.spinor_np(V, 1, 80 + k)[..., 0] for k in range(n_vec)]).astype(np.complex128)
    cd = [d // b for d, b in zip(dims, bdims)]
    vc = si.coarse_vector_np(cd, 2 * n_vec, N, 81).astype(np.complex128)
    f = si.spinor_np(V, N, 82).astype(np.complex128)
    assert np.array_equal(transfer.prolong_coarse(dims, bdims, basis.reshape(n_vec, V, 12), vc).reshape(V, 4, 3, N),
                          transfer.prolong(dims, bdims, basis, vc))
    assert np.max(np.abs(transfer.restrict_coarse(dims, bdims, basis.reshape(n_vec, V, 12), f.reshape(V, 12, N)) -
                         transfer.restrict(dims, bdims, basis, f))) < 1e-13

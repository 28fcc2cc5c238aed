"""Pins for the oracle's coarse 9-point apply (readings S8, S9; CPU only).

PAPER.md:61 (nbasis convention), :75 (coarse-level operators).  Pins: per-site dense matmul with
numpy against gathered neighbours, RHS-column independence, the brute-force Galerkin product
R M P on tiny lattices, R P = 1, and the coarse Gamma5 symmetries of Galerkin links.
"""
import numpy as np
import pytest

import oracle
import synth_inputs as si
from helpers import shift_index
from oracle import galerkin


@pytest.mark.parametrize("cdims,nb,N", [((4, 2, 4, 2), 6, 3), ((2, 2, 2, 4), 4, 1)])
def test_coarse_apply_is_per_site_matmul(cdims, nb, N):
    A = si.coarse_links_np(cdims, nb, 31).astype(np.complex128)
    v = si.coarse_vector_np(cdims, nb, N, 32).astype(np.complex128)
    want = np.matmul(A[:, 0], v)
    for mu in range(4):
        want += np.matmul(A[:, 1 + mu], v[shift_index(cdims, mu, +1)])
        want += np.matmul(A[:, 5 + mu], v[shift_index(cdims, mu, -1)])
    got = oracle.coarse_apply(cdims, A, v)
    assert np.max(np.abs(got - want)) < 1e-12
    for r in range(N):
        assert np.array_equal(oracle.coarse_apply(cdims, A, v[..., r:r + 1])[..., 0], got[..., r])
    # single points
    assert np.max(np.abs(oracle.coarse_apply(cdims, A, v, pmask=1 << 7) -
                         np.matmul(A[:, 7], v[shift_index(cdims, 2, -1)]))) < 1e-13


def test_coarse_point_masks_are_the_single_point_matmuls():
    """Every single stencil point against numpy, and subsets add up: self + 8-point hop = 9-point (S12)."""
    cdims, nb, N = (2, 4, 2, 6), 5, 2
    A = si.coarse_links_np(cdims, nb, 37).astype(np.complex128)
    v = si.coarse_vector_np(cdims, nb, N, 38).astype(np.complex128)
    single = [np.matmul(A[:, 0], v)]
    single += [np.matmul(A[:, 1 + mu], v[shift_index(cdims, mu, +1)]) for mu in range(4)]
    single += [np.matmul(A[:, 5 + mu], v[shift_index(cdims, mu, -1)]) for mu in range(4)]
    for p in range(9):
        assert np.max(np.abs(oracle.coarse_apply(cdims, A, v, pmask=1 << p) - single[p])) < 1e-13
    hop = oracle.coarse_apply(cdims, A, v, pmask=0x1FE)
    assert np.max(np.abs(hop - sum(single[1:]))) < 1e-12
    assert np.max(np.abs(oracle.coarse_apply(cdims, A, v, pmask=0x001) + hop - oracle.coarse_apply(cdims, A, v))) < 1e-12


def test_coarse_sites_entry_matches_full():
    cdims, nb, N = (4, 2, 2, 4), 6, 2
    A = si.coarse_links_np(cdims, nb, 33).astype(np.complex128)
    v = si.coarse_vector_np(cdims, nb, N, 34).astype(np.complex128)
    full = oracle.coarse_apply(cdims, A, v)
    sites = np.array([0, 7, 31, 63])
    nbrs = np.empty((sites.size, 9, nb, N), dtype=np.complex128)
    nbrs[:, 0] = v[sites]
    for mu in range(4):
        nbrs[:, 1 + mu] = v[shift_index(cdims, mu, +1)[sites]]
        nbrs[:, 5 + mu] = v[shift_index(cdims, mu, -1)[sites]]
    assert np.array_equal(oracle.coarse_sites(A[sites], nbrs), full[sites])


@pytest.mark.parametrize("dims,bdims,n_vec", [((4, 4, 4, 4), (2, 2, 2, 2), 4),
                                              ((8, 4, 4, 4), (2, 2, 2, 2), 3),
                                              ((4, 4, 4, 8), (2, 2, 2, 4), 3)])
def test_coarse_apply_equals_galerkin_rmp(dims, bdims, n_vec):
    """9-point apply with Galerkin links = R M P, brute force (S9), including coarse extent 2 (S17)."""
    mass, csw = -0.1, 1.0
    V = si.volume(dims)
    U = si.gauge_np(dims, 35)
    phi = np.stack([si.spinor_np(V, 1, 40 + k)[..., 0] for k in range(n_vec)]).astype(np.complex128)
    P, cd = galerkin.prolongator(dims, bdims, phi)
    Vc, nb = si.volume(cd), 2 * n_vec
    assert np.max(np.abs(P.conj().T @ P - np.eye(Vc * nb))) < 1e-13          # R P = 1
    A, _ = galerkin.coarse_links(dims, bdims, U, mass, csw, P)
    N = 3
    vc = si.coarse_vector_np(cd, nb, N, 36).astype(np.complex128)
    fine = (P @ vc.reshape(Vc * nb, N)).reshape(V, 4, 3, N)
    want = (P.conj().T @ galerkin.wilson_clover_apply(dims, U, mass, csw, fine).reshape(V * 12, N)).reshape(Vc, nb, N)
    got = oracle.coarse_apply(cd, A, vc)
    assert np.max(np.abs(got - want)) < 1e-12
    # coarse Gamma5 = diag(+1 x n_vec, -1 x n_vec): A_{-mu}(x) = Gamma5 A_{+mu}(x-mu)^+ Gamma5, A_0 Gamma5-hermitian
    G5 = np.diag(np.concatenate([np.ones(n_vec), -np.ones(n_vec)]))
    for mu in range(4):
        xm = shift_index(cd, mu, -1)
        rhs = np.einsum("ij,xkj,kl->xil", G5, A[xm, 1 + mu].conj(), G5)
        assert np.max(np.abs(A[:, 5 + mu] - rhs)) < 1e-13
    assert np.max(np.abs(A[:, 0] - np.einsum("ij,xkj,kl->xil", G5, A[:, 0].conj(), G5))) < 1e-13


@pytest.mark.parametrize("cdims,nb,N", [((4, 2, 4, 2), 6, 3), ((2, 2, 2, 4), 4, 1), ((6, 4, 2, 2), 5, 2)])
def test_coarse_meooe_pins(cdims, nb, N):
    """Coarse M_eooe (NEXT-1).  Pins: (1) the 8-point hopping term on the full lattice equals the merge of
    the two parities' M_eooe (identity, like D_hop = M_eooe(0) + M_eooe(1)); (2) brute force: every output site from
    hand-computed integer coordinates and numpy matmuls; (3) RHS columns are independent; (4) the input is read from the
    other parity only (perturbing the same-parity sites of the full field changes nothing)."""
    A = si.coarse_links_np(cdims, nb, 41).astype(np.complex128)
    v = si.coarse_vector_np(cdims, nb, N, 42).astype(np.complex128)
    ve, vo = oracle.cb_split(cdims, v)
    got = [oracle.coarse_meooe(cdims, A, vo, 0), oracle.coarse_meooe(cdims, A, ve, 1)]
    # (1) hop8 = M_eooe(0) + M_eooe(1) after merging parities
    hop = oracle.coarse_apply(cdims, A, v, pmask=0x1FE)
    assert np.max(np.abs(oracle.cb_merge(cdims, got[0], got[1]) - hop)) < 1e-12
    # (2) brute force, one site at a time, coordinates by hand
    X, Y, Z, T = cdims
    for out_parity, src in ((0, vo), (1, ve)):
        for lex in range(X * Y * Z * T):
            c = [lex % X, (lex // X) % Y, (lex // (X * Y)) % Z, lex // (X * Y * Z)]
            if sum(c) % 2 != out_parity:
                continue
            want = np.zeros((nb, N), dtype=np.complex128)
            for mu in range(4):
                for sign, p in ((+1, 1 + mu), (-1, 5 + mu)):
                    d = list(c)
                    d[mu] = (d[mu] + sign) % cdims[mu]
                    nlex = d[0] + X * (d[1] + Y * (d[2] + Z * d[3]))
                    assert sum(d) % 2 == 1 - out_parity
                    want += A[lex, p] @ src[nlex >> 1]
            assert np.max(np.abs(got[out_parity][lex >> 1] - want)) < 1e-12
    # (3) columns
    for r in range(N):
        assert np.array_equal(oracle.coarse_meooe(cdims, A, vo[..., r:r + 1], 0)[..., 0], got[0][..., r])
    # (4) M_eooe(0) of a field does not depend on its even sites
    v2 = v.copy()
    v2[oracle.parity_mask(cdims) == 0] += 1.0
    assert np.array_equal(oracle.coarse_meooe(cdims, A, oracle.cb_split(cdims, v2)[1], 0), got[0])

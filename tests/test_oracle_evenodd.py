"""Pins for the oracle's dagger variants and even-odd preconditioned operator (oracle/evenodd.py; SURVEY.md Sec. 8(f)
NEXT-2; CPU only).  The forward operators are pinned elsewhere (plane wave, covariance, single hops);
here the daggers are pinned by adjointness on independent random fields, by the dense matrix on a 2^4 lattice, and the
Schur complement by block elimination of the full matrix M (which has its own pins)."""
import numpy as np
import pytest

import oracle
import synth_inputs as si
from oracle import evenodd


def _inner(a, b):
    return np.vdot(a.reshape(-1), b.reshape(-1))


def _fields(dims, N, seed):
    V = si.volume(dims)
    U = si.gauge_np(dims, seed).astype(np.complex128)
    psi = si.spinor_np(V, N, seed).astype(np.complex128)
    chi = si.spinor_np(V, N, seed + 100).astype(np.complex128)
    return U, psi, chi


@pytest.mark.parametrize("dims", [(4, 4, 2, 2), (2, 2, 2, 4), (6, 2, 4, 2)])
def test_dagger_variants_are_adjoints(dims):
    U, psi, chi = _fields(dims, 1, 3)
    mass, csw = -0.05, 1.5
    C, _ = oracle.clover_blocks(dims, U, mass, csw)
    # <chi, D psi> = <D^dagger chi, psi>
    assert abs(_inner(chi, oracle.dhop(dims, U, psi)) - _inner(evenodd.dhop_dag(dims, U, chi), psi)) < 1e-10
    assert abs(_inner(chi, evenodd.wilson_clover(dims, U, C, psi)) - _inner(evenodd.wilson_clover(dims, U, C, chi, dagger=True), psi)) < 1e-10
    pe, po = oracle.cb_split(dims, psi)
    ce, co = oracle.cb_split(dims, chi)
    # M_eooe(even <- odd)^dagger maps even fields to odd ones: <chi_e, H_eo psi_o> = <(H^dagger)_oe chi_e, psi_o>
    assert abs(_inner(ce, oracle.meooe(dims, U, po, 0)) - _inner(evenodd.meooe_dag(dims, U, ce, 1), po)) < 1e-10
    assert abs(_inner(co, oracle.meooe(dims, U, pe, 1)) - _inner(evenodd.meooe_dag(dims, U, co, 0), pe)) < 1e-10
    # D^dagger = M_eooe^dagger(0) + M_eooe^dagger(1)
    merged = oracle.cb_merge(dims, evenodd.meooe_dag(dims, U, po, 0), evenodd.meooe_dag(dims, U, pe, 1))
    assert np.max(np.abs(merged - evenodd.dhop_dag(dims, U, psi))) < 1e-12
    # the Schur complement and its dagger
    assert abs(_inner(ce, evenodd.schur(dims, U, C, pe)) - _inner(evenodd.schur(dims, U, C, ce, dagger=True), pe)) < 1e-10


def test_dagger_is_the_conjugate_transpose_of_the_dense_matrix():
    """Brute force on 2^4: build the dense 192 x 192 matrix of D_hop column by column and compare D^dagger with its
    conjugate transpose (independent of gamma_5)."""
    dims = (2, 2, 2, 2)
    V = si.volume(dims)
    U = si.gauge_np(dims, 5).astype(np.complex128)
    n = V * 12
    eye = np.eye(n, dtype=np.complex128).reshape(V, 4, 3, n)
    D = oracle.dhop(dims, U, eye).reshape(n, n)
    Dd = evenodd.dhop_dag(dims, U, eye).reshape(n, n)
    assert np.max(np.abs(Dd - D.conj().T)) < 1e-12


@pytest.mark.parametrize("dims,N", [((4, 2, 2, 4), 2), ((2, 4, 4, 2), 1)])
def test_schur_complement_is_block_elimination_of_the_full_matrix(dims, N):
    """If x_o = -M_oo^-1 M_oe x_e then (M x)_o = 0 and (M x)_e = S x_e: pins S against the full matrix M, which is pinned
    by its own tests (and is what mrhs_wilson_apply computes)."""
    mass, csw = -0.05, 1.5
    U, psi, _ = _fields(dims, N, 7)
    C, _ = oracle.clover_blocks(dims, U, mass, csw)
    Ce, Co = oracle.cb_split(dims, C)
    x_e, _ = oracle.cb_split(dims, psi)
    # M_oe x_e = -H_oe x_e / 2
    x_o = -oracle.mooee(oracle.clover_inverse(Co), -0.5 * oracle.meooe(dims, U, x_e, 1))
    x = oracle.cb_merge(dims, x_e, x_o)
    for dagger in (False, True):
        if dagger:
            x_o = -oracle.mooee(oracle.clover_inverse(Co), -0.5 * evenodd.meooe_dag(dims, U, x_e, 1))
            x = oracle.cb_merge(dims, x_e, x_o)
        Mx = evenodd.wilson_clover(dims, U, C, x, dagger=dagger)
        Mx_e, Mx_o = oracle.cb_split(dims, Mx)
        assert np.max(np.abs(Mx_o)) < 1e-12
        assert np.max(np.abs(Mx_e - evenodd.schur(dims, U, C, x_e, dagger=dagger))) < 1e-12
    # and the oracle's full matrix agrees with the Galerkin module's (used by the coarse-operator pins)
    from oracle import galerkin
    assert np.max(np.abs(galerkin.wilson_clover_apply(dims, U, mass, csw, psi) - evenodd.wilson_clover(dims, U, C, psi))) < 1e-12

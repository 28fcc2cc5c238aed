"""Pins for the oracle's fine-level hopping terms (SURVEY.md Sec. 8(c) "Pins"; CPU only).

Each pin checks ``oracle`` against something the mathematics fixes, never against itself:
gamma algebra and hand-written matrices (S2), the free-field plane-wave closed form (S3),
gamma5-hermiticity in its unstarred form (S13), gauge covariance, D_hop = M_eooe + M_eooe (S4,
PAPER.md:43), RHS-column independence and single directed hops against numpy.
"""
import os

import numpy as np
import pytest

import oracle
import synth_inputs as si
from helpers import coords, read_golden_gammas, shift_index

DIMS = [(4, 4, 4, 6), (4, 2, 6, 4)]


def inner(a, b):
    return np.vdot(a.reshape(-1), b.reshape(-1))


def test_gamma_matches_handwritten(golden_dir):
    gold = read_golden_gammas(os.path.join(golden_dir, "gamma_chiral.txt"))
    for mu in range(5):
        assert np.array_equal(oracle.gamma(mu), gold[mu])


def test_gamma_algebra():
    g = [oracle.gamma(mu) for mu in range(4)]
    for mu in range(4):
        assert np.allclose(g[mu], g[mu].conj().T)
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.allclose(anti, 2.0 * np.eye(4) * (mu == nu), atol=1e-15)
    assert np.allclose(oracle.gamma(4), np.diag([1, 1, -1, -1]))
    assert np.allclose(oracle.gamma(4), g[0] @ g[1] @ g[2] @ g[3])
    # sigma_xy = i gamma_x gamma_y = diag(-1, 1, -1, 1) in this basis
    assert np.allclose(oracle.sigma(0, 1), np.diag([-1, 1, -1, 1]))
    for mu in range(4):
        for nu in range(4):
            assert np.allclose(oracle.sigma(mu, nu), -oracle.sigma(nu, mu))
            assert np.allclose(oracle.sigma(mu, nu), oracle.sigma(mu, nu).conj().T)


@pytest.mark.parametrize("dims", DIMS)
def test_free_field_plane_wave(dims, golden_dir):
    """U = 1, psi = u exp(i p x): D_hop psi = sum_mu [2 cos p_mu - 2 i gamma_mu sin p_mu] psi."""
    gold = read_golden_gammas(os.path.join(golden_dir, "gamma_chiral.txt"))
    V = si.volume(dims)
    rng = np.random.default_rng(11)
    ks = [(1, 0, 2, 1), (0, 1, 1, 3), (3, 1, 0, 2)]
    N = len(ks)
    u = rng.standard_normal((N, 4, 3)) + 1j * rng.standard_normal((N, 4, 3))
    c = coords(dims)
    psi = np.zeros((V, 4, 3, N), dtype=np.complex128)
    want = np.zeros_like(psi)
    for r, k in enumerate(ks):
        p = [2 * np.pi * k[mu] / dims[mu] for mu in range(4)]
        phase = np.exp(1j * sum(p[mu] * c[mu] for mu in range(4)))
        psi[..., r] = phase[:, None, None] * u[r][None]
        S = sum(2 * np.cos(p[mu]) * np.eye(4) - 2j * np.sin(p[mu]) * gold[mu] for mu in range(4))
        want[..., r] = phase[:, None, None] * np.einsum("st,tc->sc", S, u[r])[None]
    got = oracle.dhop(dims, si.unit_gauge_np(dims), psi)
    assert np.max(np.abs(got - want)) < 1e-12


@pytest.mark.parametrize("dims", DIMS)
def test_gamma5_hermiticity(dims):
    """S13 (unstarred): <chi, D psi> = <gamma5 D gamma5 chi, psi>."""
    V = si.volume(dims)
    U = si.gauge_np(dims, 3)
    psi = si.spinor_np(V, 2, 4).astype(np.complex128)
    chi = si.spinor_np(V, 2, 5).astype(np.complex128)
    g5 = np.array([1, 1, -1, -1.0])[None, :, None, None]
    lhs = inner(chi, oracle.dhop(dims, U, psi))
    rhs = inner(g5 * oracle.dhop(dims, U, g5 * chi), psi)
    assert abs(lhs - rhs) < 1e-10 * abs(lhs)
    # the starred form printed in BASELINE.json does not hold (guards against a silent convention flip)
    assert abs(lhs - np.conj(rhs)) > 1e-3 * abs(lhs)


@pytest.mark.parametrize("dims", DIMS)
def test_gauge_covariance(dims):
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^+, psi' = g psi  =>  D[U'] psi' = g D[U] psi."""
    V = si.volume(dims)
    U = si.gauge_np(dims, 6).astype(np.complex128)
    g = si.gauge_transform_np(dims, 7)
    psi = si.spinor_np(V, 3, 8).astype(np.complex128)
    Up = np.empty_like(U)
    for mu in range(4):
        gn = g[shift_index(dims, mu, +1)]
        Up[:, mu] = np.einsum("xab,xbc,xdc->xad", g, U[:, mu], gn.conj())
    psip = np.einsum("xab,xsbr->xsar", g, psi)
    lhs = oracle.dhop(dims, Up, psip)
    rhs = np.einsum("xab,xsbr->xsar", g, oracle.dhop(dims, U, psi))
    assert np.max(np.abs(lhs - rhs)) < 1e-11


@pytest.mark.parametrize("dims", DIMS)
def test_single_directed_hops_against_numpy(dims, golden_dir):
    """Each of the 8 terms of S3 alone, written with numpy gathers and einsum; their sum is D_hop."""
    gold = read_golden_gammas(os.path.join(golden_dir, "gamma_chiral.txt"))
    V = si.volume(dims)
    U = si.gauge_np(dims, 9).astype(np.complex128)
    psi = si.spinor_np(V, 2, 10).astype(np.complex128)
    total = np.zeros_like(psi)
    for mu in range(4):
        fwd = np.einsum("st,xab,xtbr->xsar", np.eye(4) - gold[mu], U[:, mu], psi[shift_index(dims, mu, +1)])
        xm = shift_index(dims, mu, -1)
        bwd = np.einsum("st,xba,xtbr->xsar", np.eye(4) + gold[mu], U[xm, mu].conj(), psi[xm])
        assert np.max(np.abs(oracle.dhop(dims, U, psi, dirmask=1 << mu) - fwd)) < 1e-12
        assert np.max(np.abs(oracle.dhop(dims, U, psi, dirmask=1 << (4 + mu)) - bwd)) < 1e-12
        total += fwd + bwd
    assert np.max(np.abs(oracle.dhop(dims, U, psi) - total)) < 1e-12


@pytest.mark.parametrize("dims", DIMS + [(2, 2, 2, 2)])
def test_dhop_is_sum_of_meooe(dims):
    """on checkerboarded lattices one calls M_eooe twice instead of D_hop once."""
    V = si.volume(dims)
    U = si.gauge_np(dims, 12)
    psi = si.spinor_np(V, 3, 13)
    full = oracle.dhop(dims, U, psi)
    pe, po = oracle.cb_split(dims, psi)
    oe = oracle.meooe(dims, U, po, 0)
    oo = oracle.meooe(dims, U, pe, 1)
    assert np.array_equal(oracle.cb_merge(dims, oe, oo), full)


def test_checkerboard_index_is_lex_shift():
    dims = (4, 2, 6, 4)
    p = oracle.parity_mask(dims)
    c = coords(dims)
    assert np.array_equal(p, c.sum(axis=0) % 2)
    for par in (0, 1):
        lex = np.nonzero(p == par)[0]
        assert np.array_equal(lex >> 1, np.arange(lex.size))
    for lex in (0, 5, 17, 100):
        assert oracle.parity(dims, lex) == p[lex]
        for mu in range(4):
            assert oracle.neighbour(dims, lex, mu, +1) == shift_index(dims, mu, +1)[lex]
            assert oracle.neighbour(dims, lex, mu, -1) == shift_index(dims, mu, -1)[lex]


def test_rhs_columns_are_independent():
    """the RHS index is a spectator; column r equals the single-RHS result."""
    dims = (4, 4, 2, 4)
    V = si.volume(dims)
    U = si.gauge_np(dims, 14)
    psi = si.spinor_np(V, 5, 15)
    full = oracle.dhop(dims, U, psi)
    for r in range(5):
        assert np.array_equal(oracle.dhop(dims, U, psi[..., r:r + 1])[..., 0], full[..., r])


def test_site_entry_matches_full_lattice():
    """The packed per-site entry used for sampled 48^4 parity is the same arithmetic."""
    dims = (4, 4, 4, 4)
    V = si.volume(dims)
    U = si.gauge_np(dims, 16).astype(np.complex128)
    psi = si.spinor_np(V, 2, 17).astype(np.complex128)
    full = oracle.dhop(dims, U, psi)
    sites = np.array([0, 3, 63, 64, 200, 255])
    links = np.empty((sites.size, 8, 3, 3), dtype=np.complex128)
    nbrs = np.empty((sites.size, 8, 4, 3, 2), dtype=np.complex128)
    for mu in range(4):
        xp = shift_index(dims, mu, +1)[sites]
        xm = shift_index(dims, mu, -1)[sites]
        links[:, mu] = U[sites, mu]
        links[:, 4 + mu] = U[xm, mu]
        nbrs[:, mu] = psi[xp]
        nbrs[:, 4 + mu] = psi[xm]
    assert np.array_equal(oracle.dhop_sites(links, nbrs), full[sites])


def test_inputs_are_su3():
    U = si.gauge_np((4, 4, 4, 4), 0).astype(np.complex128)
    UU = np.einsum("xmab,xmcb->xmac", U, U.conj())
    assert np.max(np.abs(UU - np.eye(3))) < 1e-6          # fp32-rounded entries
    assert np.max(np.abs(np.linalg.det(U) - 1.0)) < 1e-6

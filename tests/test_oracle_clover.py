"""Pins for the oracle's clover term (SURVEY.md Sec. 8(c) "Pins", readings S5-S7; CPU only).

PAPER.md:47,:53: M_ooee applies a precomputed, site-diagonal term.  The paper prints no formula;
these pins fix sign, orientation and normalisation of the reading: Hermitian chiral blocks, zero
spin-off-diagonal blocks, block trace 6(4+m), pure-gauge field => (4+m) 1, uniform abelian flux
closed form, gauge covariance, and the apply against a numpy einsum.
"""
import numpy as np
import pytest

import oracle
import synth_inputs as si
from helpers import coords, shift_index

DIMS = [(4, 4, 4, 6), (4, 2, 6, 4)]


@pytest.mark.parametrize("dims", DIMS)
def test_blocks_hermitian_blockdiagonal_trace(dims):
    mass, csw = -0.1, 1.3
    U = si.gauge_np(dims, 21)
    C, off = oracle.clover_blocks(dims, U, mass, csw)
    assert off == 0.0                                     # spin off-diagonal 6x6 blocks vanish
    assert np.max(np.abs(C - np.conj(np.swapaxes(C, 2, 3)))) < 1e-14
    tr = np.trace(C, axis1=2, axis2=3)
    assert np.max(np.abs(tr - 6 * (4 + mass))) < 1e-12
    assert np.max(np.abs(C[0, 0] - np.diag(np.diag(C[0, 0])))) > 1e-2   # a hot field has a clover term


def test_field_strength_hermitian_antisymmetric():
    dims = (4, 4, 4, 4)
    U = si.gauge_np(dims, 22)
    for lex in (0, 77, 255):
        for mu in range(4):
            for nu in range(4):
                if mu == nu:
                    continue
                F = oracle.field_strength(dims, U, lex, mu, nu)
                assert np.max(np.abs(F - F.conj().T)) < 1e-14
                assert np.max(np.abs(F + oracle.field_strength(dims, U, lex, nu, mu))) < 1e-14


@pytest.mark.parametrize("dims", DIMS)
def test_pure_gauge_has_no_clover(dims):
    """U_mu(x) = g(x) g(x+mu)^+  =>  every plaquette is 1  =>  M_ooee = (4 + m) 1."""
    g = si.gauge_transform_np(dims, 23)
    U = np.empty((si.volume(dims), 4, 3, 3), dtype=np.complex128)
    for mu in range(4):
        U[:, mu] = np.einsum("xab,xcb->xac", g, g[shift_index(dims, mu, +1)].conj())
    C, off = oracle.clover_blocks(dims, U, 0.2, 1.7)
    assert off < 1e-14
    assert np.max(np.abs(C - (4 + 0.2) * np.eye(6))) < 1e-13


@pytest.mark.parametrize("plane", [(0, 1), (1, 2), (0, 3), (2, 3)])
def test_uniform_abelian_flux_closed_form(plane):
    """theta_mu(x) = -B x_nu, theta_nu(x) = B L_nu x_mu on the slice x_nu = L_nu - 1, B = 2 pi k/(L_mu L_nu),
    U = exp(i theta T), T = diag(1,-1,0): every mu-nu plaquette is exp(i B T), so F_munu = sin(B T), the other
    planes vanish, and M_ooee = (4+m) - (c_sw/2) sigma_munu (x) sin(B T).  Pins sign and orientation."""
    mu, nu = plane
    dims = (4, 6, 4, 2)
    mass, csw, k = -0.05, 1.5, 1
    V = si.volume(dims)
    c = coords(dims)
    B = 2 * np.pi * k / (dims[mu] * dims[nu])
    Tgen = np.array([1.0, -1.0, 0.0])
    U = si.unit_gauge_np(dims).astype(np.complex128)
    th_mu = -B * c[nu]
    th_nu = np.where(c[nu] == dims[nu] - 1, B * dims[nu] * c[mu], 0.0)
    for a in range(3):
        U[:, mu, a, a] = np.exp(1j * th_mu * Tgen[a])
        U[:, nu, a, a] = np.exp(1j * th_nu * Tgen[a])
    for lex in (0, 5, V - 1):
        assert np.max(np.abs(oracle.field_strength(dims, U, lex, mu, nu) - np.diag(np.sin(B * Tgen)))) < 1e-14
        for a in range(4):
            for b in range(a + 1, 4):
                if (a, b) != (mu, nu):
                    assert np.max(np.abs(oracle.field_strength(dims, U, lex, a, b))) < 1e-14
    want = (4 + mass) * np.eye(12) - 0.5 * csw * np.kron(oracle.sigma(mu, nu), np.diag(np.sin(B * Tgen)))
    for lex in (0, 9, V - 1):
        assert np.max(np.abs(oracle.clover_site_matrix(dims, U, mass, csw, lex) - want)) < 1e-13
    if plane == (0, 1):
        # sigma_xy = diag(-1,1,-1,1) written out by hand (S2): explicit diagonal of the site matrix
        s = np.sin(B * Tgen)
        diag = np.concatenate([(4 + mass) - 0.5 * csw * sg * s for sg in (-1, 1, -1, 1)])
        assert np.max(np.abs(np.diag(want) - diag)) < 1e-15


def test_clover_gauge_covariance():
    dims = (4, 4, 2, 4)
    U = si.gauge_np(dims, 24).astype(np.complex128)
    g = si.gauge_transform_np(dims, 25)
    Up = np.empty_like(U)
    for mu in range(4):
        Up[:, mu] = np.einsum("xab,xbc,xdc->xad", g, U[:, mu], g[shift_index(dims, mu, +1)].conj())
    C, _ = oracle.clover_blocks(dims, U, -0.1, 1.0)
    Cp, _ = oracle.clover_blocks(dims, Up, -0.1, 1.0)
    # block index 3*(spin%2)+colour: g acts as 1_2 (x) g on each 6x6 block
    G = np.einsum("st,xab->xsatb", np.eye(2), g).reshape(-1, 6, 6)
    want = np.einsum("xij,xbjk,xlk->xbil", G, C, G.conj())
    assert np.max(np.abs(Cp - want)) < 1e-12


def test_mooee_apply_against_einsum_and_site_matrix():
    dims = (4, 4, 4, 4)
    V = si.volume(dims)
    U = si.gauge_np(dims, 26)
    psi = si.spinor_np(V, 3, 27).astype(np.complex128)
    C, _ = oracle.clover_blocks(dims, U, -0.1, 1.0)
    got = oracle.mooee(C, psi)
    want = np.einsum("xbij,xbjr->xbir", C, psi.reshape(V, 2, 6, 3)).reshape(V, 4, 3, 3)
    assert np.max(np.abs(got - want)) < 1e-13
    for lex in (0, 100):
        M = oracle.clover_site_matrix(dims, U, -0.1, 1.0, lex)
        assert np.max(np.abs(got[lex].reshape(12, 3) - M @ psi[lex].reshape(12, 3))) < 1e-13


def test_full_matrix_gamma5_hermiticity():
    """M = M_ooee - (1/2) D_hop (S6) obeys <chi, M psi> = <gamma5 M gamma5 chi, psi> (S13)."""
    dims = (4, 4, 4, 4)
    V = si.volume(dims)
    U = si.gauge_np(dims, 28)
    C, _ = oracle.clover_blocks(dims, U, -0.1, 1.0)
    psi = si.spinor_np(V, 1, 29).astype(np.complex128)
    chi = si.spinor_np(V, 1, 30).astype(np.complex128)
    g5 = np.array([1, 1, -1, -1.0])[None, :, None, None]

    def M(v):
        return oracle.mooee(C, v) - 0.5 * oracle.dhop(dims, U, v)

    lhs = np.vdot(chi, M(psi))
    rhs = np.vdot(g5 * M(g5 * chi), psi)
    assert abs(lhs - rhs) < 1e-10 * abs(lhs)


def test_clover_inverse_blocks():
    """Inverse blocks: C C^-1 = 1, Hermitian, and (4 + m)^-1 on a pure-gauge field (closed form)."""
    dims, mass, csw = (4, 4, 2, 4), -0.1, 1.3
    U = si.gauge_np(dims, 61)
    C, _ = oracle.clover_blocks(dims, U, mass, csw)
    Ci = oracle.clover_inverse(C)
    eye = np.broadcast_to(np.eye(6), C.shape)
    assert np.max(np.abs(np.matmul(C, Ci) - eye)) < 1e-12
    assert np.max(np.abs(Ci - np.conj(np.swapaxes(Ci, 2, 3)))) < 1e-12
    g = si.gauge_transform_np(dims, 63)
    Upg = np.empty((si.volume(dims), 4, 3, 3), dtype=np.complex128)
    for mu in range(4):
        Upg[:, mu] = np.einsum("xab,xcb->xac", g, g[shift_index(dims, mu, +1)].conj())   # U_mu(x) = g(x) g(x+mu)^+
    Cpg, _ = oracle.clover_blocks(dims, Upg, mass, csw)
    assert np.max(np.abs(oracle.clover_inverse(Cpg) - eye / (4 + mass))) < 1e-12

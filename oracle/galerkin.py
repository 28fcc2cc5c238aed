"""Galerkin coarsening for the oracle's self-check -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Reading S9 of SURVEY.md Sec. 8(c) (nbasis = twice the number of multigrid basis
vectors = spinor elements per site on the next coarser level).  Used only on tiny lattices to
pin ``oracle.coarse_apply`` against the brute-force product R M P; slow by design.

Steps, in order:
  1. take n_vec = nb/2 fine vectors phi_k [V][4][3];
  2. split by chirality, phi_k^(+-) = (1 +- gamma_5)/2 phi_k, coarse index j = chi*n_vec + k;
  3. restrict each to each block (aggregate) and orthonormalise inside the block (Gram-Schmidt);
  4. P copies coarse coefficients onto the block basis, R = P^dagger;
  5. A_0(B) = P_B^+ [M_ooee + hops inside B] P_B, A_{+mu}(B) = P_B^+ [forward hops in mu leaving B]
     P_{B+mu}, A_{-mu}(B) likewise, hops carrying the -1/2 of M = M_ooee - (1/2) D_hop (S6).
"""
import numpy as np

import oracle


def block_of_site(dims, bdims):
    """coarse lex of the block containing each fine site, and the coarse dims."""
    X, Y, Z, T = [int(d) for d in dims]
    cd = [int(d) // int(b) for d, b in zip(dims, bdims)]
    assert all(c * b == d for c, b, d in zip(cd, bdims, dims))
    lex = np.arange(X * Y * Z * T)
    x = lex % X; y = (lex // X) % Y; z = (lex // (X * Y)) % Z; t = lex // (X * Y * Z)
    cx, cy, cz, ct = x // bdims[0], y // bdims[1], z // bdims[2], t // bdims[3]
    return cx + cd[0] * (cy + cd[1] * (cz + cd[2] * ct)), cd


def prolongator(dims, bdims, phi):
    """P as a dense matrix [V*12][Vc*nb] from phi [n_vec][V][4][3] (steps 1-4)."""
    n_vec = phi.shape[0]
    nb = 2 * n_vec
    V = oracle.volume(dims)
    blk, cd = block_of_site(dims, bdims)
    Vc = oracle.volume(cd)
    g5 = np.real(np.diag(oracle.gamma(4)))                 # diag(+1,+1,-1,-1)
    P = np.zeros((V, 4, 3, Vc, nb), dtype=np.complex128)
    for chi, sign in enumerate((+1.0, -1.0)):
        proj = (1.0 + sign * g5) / 2.0                      # (1 +- gamma_5)/2, diagonal
        for B in range(Vc):
            sites = np.nonzero(blk == B)[0]
            basis = []
            for k in range(n_vec):
                w = phi[k][sites] * proj[None, :, None]     # restrict + chirality
                for q in basis:                             # Gram-Schmidt inside the block
                    w = w - q * np.vdot(q, w)
                w = w / np.sqrt(np.vdot(w, w).real)
                basis.append(w)
                P[sites, :, :, B, chi * n_vec + k] = w
    return P.reshape(V * 12, Vc * nb), cd


def wilson_clover_apply(dims, U, mass, csw, psi, dirmask=0xFF, with_clover=True):
    """M psi = M_ooee psi - (1/2) D_hop psi (S6), psi [V][4][3][N], optionally only some hops."""
    out = -0.5 * oracle.dhop(dims, U, psi, dirmask)
    if with_clover:
        C, _ = oracle.clover_blocks(dims, U, mass, csw)
        out = out + oracle.mooee(C, psi)
    return out


def coarse_links(dims, bdims, U, mass, csw, P):
    """Step 5: A [Vc][9][nb][nb] assembled term by term from directed hops."""
    V = oracle.volume(dims)
    blk, cd = block_of_site(dims, bdims)
    Vc = oracle.volume(cd)
    nb = P.shape[1] // Vc
    assert all(c >= 2 for c in cd)
    Pf = P.reshape(V, 4, 3, Vc * nb)
    rows = np.repeat(blk, 12)                               # block of every fine row
    A = np.zeros((Vc, 9, nb, nb), dtype=np.complex128)

    def project(W, B, Bcol):
        PB = P[rows == B][:, B * nb:(B + 1) * nb]
        return PB.conj().T @ W[rows == B][:, Bcol * nb:(Bcol + 1) * nb]

    Wc = wilson_clover_apply(dims, U, mass, csw, Pf, dirmask=0).reshape(V * 12, Vc * nb)
    for B in range(Vc):
        A[B, 0] += project(Wc, B, B)
    for mu in range(4):
        for back in (0, 1):
            bit = 1 << (4 * back + mu)
            W = wilson_clover_apply(dims, U, mass, csw, Pf, dirmask=bit, with_clover=False).reshape(V * 12, Vc * nb)
            for B in range(Vc):
                Bn = oracle.neighbour(cd, B, mu, -1 if back else +1)
                A[B, 0] += project(W, B, B)                 # hops that stay inside B
                A[B, 1 + 4 * back + mu] += project(W, B, Bn)  # hops that leave B
    return A, cd

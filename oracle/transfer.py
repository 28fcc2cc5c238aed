"""Intergrid operators of the MRHS multigrid -- TEST INFRASTRUCTURE.

Reading S9 of SURVEY.md Sec. 8(c): n_vec = nb / 2 basis vectors phi_k [V][4][3] (as given: orthonormalising them is the
setup's business, galerkin.prolongator does it for the self-checks), chirality chi = 0 for spins {0, 1} and 1 for spins
{2, 3}, coarse index j = chi * n_vec + k, blocks (aggregates) of bdims fine sites.

    prolong:   fine(x)[s][c][r]  = sum_k phi_k(x)[s][c] * coarse(B(x))[chi(s) * n_vec + k][r]
    restrict:  coarse(B)[chi * n_vec + k][r] = sum_{x in B} sum_{s in chi} sum_c conj(phi_k(x)[s][c]) * fine(x)[s][c][r]

for every right-hand side r at once; restrict is the adjoint of prolong.  fp64, numpy einsum / add.at as the steps."""
import numpy as np

from . import galerkin


def prolong(dims, bdims, basis, coarse):
    """basis [n_vec][V][4][3], coarse [Vc][2 n_vec][N] -> fine [V][4][3][N]."""
    basis = np.asarray(basis, dtype=np.complex128)
    coarse = np.asarray(coarse, dtype=np.complex128)
    n_vec = basis.shape[0]
    blk, _ = galerkin.block_of_site(dims, bdims)
    V = basis.shape[1]
    out = np.zeros((V, 4, 3, coarse.shape[-1]), dtype=np.complex128)
    cb = coarse[blk]                                              # the block's coarse vector at every fine site
    for chi in (0, 1):
        out[:, 2 * chi:2 * chi + 2] = np.einsum("kxsc,xkn->xscn", basis[:, :, 2 * chi:2 * chi + 2], cb[:, chi * n_vec:(chi + 1) * n_vec])
    return out


def restrict(dims, bdims, basis, fine):
    """basis [n_vec][V][4][3], fine [V][4][3][N] -> coarse [Vc][2 n_vec][N]."""
    basis = np.asarray(basis, dtype=np.complex128)
    fine = np.asarray(fine, dtype=np.complex128)
    n_vec = basis.shape[0]
    blk, cd = galerkin.block_of_site(dims, bdims)
    Vc = int(np.prod(cd))
    out = np.zeros((Vc, 2 * n_vec, fine.shape[-1]), dtype=np.complex128)
    for chi in (0, 1):
        per_site = np.einsum("kxsc,xscn->xkn", np.conj(basis[:, :, 2 * chi:2 * chi + 2]), fine[:, 2 * chi:2 * chi + 2])
        np.add.at(out[:, chi * n_vec:(chi + 1) * n_vec], blk, per_site)
    return out


# ---- coarse -> coarser (the intergrid operators between the intermediate and the coarsest level act
# on spinors with nbasis_f components per site instead of 12).  Same definition with the "fine" field v(x)[c], c < n_f, whose
# chirality is chi(c) = 0 for c < n_f / 2 and 1 otherwise (coarse index j = chi * n + k of reading S9 one level up):
#     prolong:   out(x)[c][r] = sum_k phi_k(x)[c] * coarse(B(x))[chi(c) * n_vec + k][r]
#     restrict:  coarse(B)[chi * n_vec + k][r] = sum_{x in B} sum_{c in chi} conj(phi_k(x)[c]) * in(x)[c][r]

def prolong_coarse(fdims, bdims, basis, coarse):
    """basis [n_vec][Vf][n_f], coarse [Vc][2 n_vec][N] -> [Vf][n_f][N]."""
    basis = np.asarray(basis, dtype=np.complex128)
    coarse = np.asarray(coarse, dtype=np.complex128)
    n_vec, Vf, nf = basis.shape
    assert nf % 2 == 0
    h = nf // 2
    blk, _ = galerkin.block_of_site(fdims, bdims)
    cb = coarse[blk]
    out = np.zeros((Vf, nf, coarse.shape[-1]), dtype=np.complex128)
    for chi in (0, 1):
        out[:, chi * h:(chi + 1) * h] = np.einsum("kxc,xkn->xcn", basis[:, :, chi * h:(chi + 1) * h], cb[:, chi * n_vec:(chi + 1) * n_vec])
    return out


def restrict_coarse(fdims, bdims, basis, fine):
    """basis [n_vec][Vf][n_f], fine [Vf][n_f][N] -> [Vc][2 n_vec][N]."""
    basis = np.asarray(basis, dtype=np.complex128)
    fine = np.asarray(fine, dtype=np.complex128)
    n_vec, Vf, nf = basis.shape
    assert nf % 2 == 0
    h = nf // 2
    blk, cd = galerkin.block_of_site(fdims, bdims)
    Vc = int(np.prod(cd))
    out = np.zeros((Vc, 2 * n_vec, fine.shape[-1]), dtype=np.complex128)
    for chi in (0, 1):
        per_site = np.einsum("kxc,xcn->xkn", np.conj(basis[:, :, chi * h:(chi + 1) * h]), fine[:, chi * h:(chi + 1) * h])
        np.add.at(out[:, chi * n_vec:(chi + 1) * n_vec], blk, per_site)
    return out

"""Oracle for the dagger variants and the even-odd preconditioned (Schur complement) operator -- TEST INFRASTRUCTURE.

SURVEY.md Sec. 8(f) NEXT-2; PAPER.md:43 (hopping terms), :53 (precomputed clover term and its inverse).  The paper prints
no formula; the definitions follow readings S3-S6 of DESIGN.md.  Everything here is a composition of the plain oracle
operators of ``mrhs_oracle.c`` (dhop, meooe, mooee, clover_inverse), written out in the order of the definition:

* gamma_5 = diag(+1, +1, -1, -1) on the spin index (reading S2);
* D_hop^dagger = gamma_5 D_hop gamma_5 (gamma5-hermiticity of the hopping term, itself pinned in test_oracle_fine.py),
  likewise M_eooe^dagger, which maps parity 1 - p to parity p like M_eooe;
* M = M_ooee - D_hop / 2 (reading S6), M^dagger = M_ooee - D_hop^dagger / 2 (the clover blocks are Hermitian);
* with M split by parity, M_ee = M_ooee on even sites, M_eo = -M_eooe(even <- odd) / 2, the Schur complement on the even
  sites is  S = M_ee - M_eo M_oo^-1 M_oe = C_e - (1/4) H_eo C_o^-1 H_oe,  and S^dagger is the same with daggered hops.

Versus the paper's own code: parity unpinned.
"""
import numpy as np

import oracle


def gamma5(psi):
    """gamma_5 psi for psi [sites][4][3][N] (S2: diag(1, 1, -1, -1))."""
    out = np.array(psi, dtype=np.complex128, copy=True)
    out[:, 2:4] *= -1.0
    return out


def dhop_dag(dims, U, psi):
    return gamma5(oracle.dhop(dims, U, gamma5(psi)))


def meooe_dag(dims, U, psi_cb, out_parity):
    """(D_hop^dagger) restricted to output parity out_parity, input of parity 1 - out_parity."""
    return gamma5(oracle.meooe(dims, U, gamma5(psi_cb), out_parity))


def wilson_clover(dims, U, C, psi, dagger=False):
    """M psi or M^dagger psi on full-lattice fields, C = clover blocks [V][2][6][6] (S6)."""
    hop = dhop_dag(dims, U, psi) if dagger else oracle.dhop(dims, U, psi)
    return oracle.mooee(C, psi) - 0.5 * hop


def schur(dims, U, C, psi_e, dagger=False):
    """S psi_e (or S^dagger psi_e), S = C_e - (1/4) H_eo C_o^-1 H_oe on even-site fields [V/2][4][3][N]."""
    Ce, Co = oracle.cb_split(dims, C)
    hop = meooe_dag if dagger else oracle.meooe
    t_o = hop(dims, U, psi_e, 1)                       # H_oe psi_e, on odd sites
    t_o = oracle.mooee(oracle.clover_inverse(Co), t_o)  # C_o^-1
    return oracle.mooee(Ce, psi_e) - 0.25 * hop(dims, U, t_o, 0)

"""GPU parity of the MRHS intergrid operators against the fp64 oracle.
Through the C-ABI binding; basis vectors are Gaussian (the operators take the basis as given)."""
import numpy as np
import pytest

import synth_inputs as syn
from helpers import rel_l2_per_rhs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():
    pytest.skip("needs a CUDA device", allow_module_level=True)

import oracle                          # noqa: E402
from oracle import transfer as otr     # noqa: E402
import paper_2211_13719_b200 as mrhs   # noqa: E402
from gpu_common import TOL, dev, host  # noqa: E402

CASES = [
    ([4, 4, 4, 4], [2, 2, 2, 2], 3, 4),
    ([8, 4, 4, 4], [4, 2, 2, 2], 2, 1),
    ([8, 8, 4, 4], [4, 4, 2, 2], 12, 12),     # nbasis 24
    ([16, 4, 4, 8], [4, 2, 2, 4], 20, 12),    # nbasis 40, x-block of 8 sites split over two aggregates
    ([8, 8, 8, 8], [4, 4, 4, 4], 20, 24),     # 4^4 aggregates as in the paper, nbasis 40
    ([12, 6, 4, 4], [2, 3, 2, 2], 5, 3),      # odd N_rhs, block extent 3
    ([8, 4, 4, 4], [2, 2, 2, 2], 20, 96),
    ([16, 8, 4, 4], [4, 4, 2, 2], 20, 12),    # staged kernels: two aggregates per x-block, 5 x 3 tiles
    ([16, 4, 6, 4], [8, 2, 3, 2], 12, 12),    # staged kernels: block extent 8 = the x-block, odd number of rows, 4 x 3 tiles
    ([8, 4, 4, 4], [2, 2, 2, 2], 8, 8),       # staged kernels: four aggregates per x-block, 4 x 2 tiles
]


@pytest.mark.parametrize("dims,bdims,nvec,nrhs", CASES)
def test_prolong_restrict_match_oracle(dims, bdims, nvec, nrhs):
    cdims = [d // b for d, b in zip(dims, bdims)]
    V, Vc, nb = syn.volume(dims), syn.volume(cdims), 2 * nvec
    basis = np.stack([syn.spinor_np(V, 1, 100 + k)[..., 0] for k in range(nvec)])          # [nvec][V][4][3] complex64
    vc = syn.coarse_vector_np(cdims, nb, nrhs, 7)
    f = syn.spinor_np(V, nrhs, 8)
    tr = mrhs.Transfer(dims, bdims, nvec, nrhs, dev(basis))
    # prolongation
    d_c = mrhs.field_import(cdims, nb, nrhs, mrhs.FULL, dev(vc))
    d_f = mrhs.empty_field(dims, 12, nrhs, mrhs.FULL)
    tr.prolong(d_c, d_f)
    torch.cuda.synchronize()
    got = host(mrhs.field_export(dims, 12, nrhs, mrhs.FULL, d_f)).reshape(V, 4, 3, nrhs)
    err = rel_l2_per_rhs(got, otr.prolong(dims, bdims, basis, vc))
    assert err.max() < TOL, ("prolong", err)
    # restriction
    d_f = mrhs.field_import(dims, 12, nrhs, mrhs.FULL, dev(f))
    d_c = mrhs.empty_field(cdims, nb, nrhs, mrhs.FULL)
    d_c.fill_(float("nan"))
    torch.cuda.synchronize()
    tr.restrict(d_f, d_c)
    torch.cuda.synchronize()
    got = host(mrhs.field_export(cdims, nb, nrhs, mrhs.FULL, d_c)).reshape(Vc, nb, nrhs)
    err = rel_l2_per_rhs(got, otr.restrict(dims, bdims, basis, f))
    assert err.max() < TOL, ("restrict", err)
    tr.close()


def test_transfer_argument_errors():
    basis = dev(np.zeros((2, 256, 4, 3), dtype=np.complex64))
    with pytest.raises(mrhs.MrhsError):
        mrhs.Transfer([4, 4, 4, 4], [3, 2, 2, 2], 2, 4, basis)      # 3 does not divide 4
    with pytest.raises(mrhs.MrhsError):
        mrhs.Transfer([4, 4, 4, 4], [4, 2, 2, 2], 2, 4, basis)      # coarse extent 1


# ---- coarse -> coarser (nbasis 40 -> 60 in the paper's solve); both fields in the coarse layout
COARSE_CASES = [
    ([4, 4, 4, 4], [2, 2, 2, 2], 8, 3, 4),
    ([6, 6, 6, 8], [3, 3, 3, 2], 40, 30, 12),      # the paper's intermediate -> coarsest shape: 40 -> 60 components
    ([4, 4, 2, 6], [2, 2, 1, 3], 24, 20, 24),
    ([4, 2, 4, 4], [2, 1, 2, 2], 12, 6, 12),       # 12-component "fine" level: must NOT be packed like a fine spinor
    ([4, 4, 4, 4], [2, 2, 2, 2], 40, 5, 3),        # odd n_vec, odd N_rhs
    ([2, 4, 4, 4], [1, 2, 2, 2], 24, 12, 96),
]


@pytest.mark.parametrize("fdims,bdims,nf,nvec,nrhs", COARSE_CASES)
def test_coarse_level_prolong_restrict_match_oracle(fdims, bdims, nf, nvec, nrhs):
    cdims = [d // b for d, b in zip(fdims, bdims)]
    Vf, Vc, nb = syn.volume(fdims), syn.volume(cdims), 2 * nvec
    basis = np.stack([syn.coarse_vector_np(fdims, nf, 1, 200 + k)[..., 0] for k in range(nvec)])     # [nvec][Vf][nf] complex64
    vc = syn.coarse_vector_np(cdims, nb, nrhs, 17)
    f = syn.coarse_vector_np(fdims, nf, nrhs, 18)
    tr = mrhs.Transfer(fdims, bdims, nvec, nrhs, dev(basis), nf=nf)
    d_c = mrhs.coarse_field_import(cdims, nb, nrhs, mrhs.FULL, dev(vc))
    d_f = mrhs.empty_field(fdims, nf, nrhs, mrhs.FULL)
    tr.prolong(d_c, d_f)
    torch.cuda.synchronize()
    err = rel_l2_per_rhs(host(mrhs.coarse_field_export(fdims, nf, nrhs, mrhs.FULL, d_f)), otr.prolong_coarse(fdims, bdims, basis, vc))
    assert err.max() < TOL, ("prolong", err)
    d_f = mrhs.coarse_field_import(fdims, nf, nrhs, mrhs.FULL, dev(f))
    d_c = mrhs.empty_field(cdims, nb, nrhs, mrhs.FULL)
    tr.restrict(d_f, d_c)
    torch.cuda.synchronize()
    err = rel_l2_per_rhs(host(mrhs.coarse_field_export(cdims, nb, nrhs, mrhs.FULL, d_c)), otr.restrict_coarse(fdims, bdims, basis, f))
    assert err.max() < TOL, ("restrict", err)
    tr.close()


def test_fine_level_transfer_with_six_basis_vectors():
    """n_vec = 6 gives 12-component coarse vectors: through the explicit coarse layout entries they are site-contiguous."""
    dims, bdims, nvec, nrhs = [8, 4, 4, 4], [4, 2, 2, 2], 6, 12
    cdims = [d // b for d, b in zip(dims, bdims)]
    V = syn.volume(dims)
    basis = np.stack([syn.spinor_np(V, 1, 300 + k)[..., 0] for k in range(nvec)])
    vc = syn.coarse_vector_np(cdims, 12, nrhs, 27)
    f = syn.spinor_np(V, nrhs, 28)
    tr = mrhs.Transfer(dims, bdims, nvec, nrhs, dev(basis))
    d_f = mrhs.empty_field(dims, 12, nrhs, mrhs.FULL)
    tr.prolong(mrhs.coarse_field_import(cdims, 12, nrhs, mrhs.FULL, dev(vc)), d_f)
    torch.cuda.synchronize()
    got = host(mrhs.field_export(dims, 12, nrhs, mrhs.FULL, d_f)).reshape(V, 4, 3, nrhs)
    assert rel_l2_per_rhs(got, otr.prolong(dims, bdims, basis, vc)).max() < TOL
    d_c = mrhs.empty_field(cdims, 12, nrhs, mrhs.FULL)
    tr.restrict(mrhs.field_import(dims, 12, nrhs, mrhs.FULL, dev(f)), d_c)
    torch.cuda.synchronize()
    got = host(mrhs.coarse_field_export(cdims, 12, nrhs, mrhs.FULL, d_c))
    assert rel_l2_per_rhs(got, otr.restrict(dims, bdims, basis, f)).max() < TOL
    tr.close()


@pytest.mark.parametrize("nrhs", [12, 24])
def test_intergrid_operators_at_48_4_on_sampled_aggregates(nrhs):
    """The size bench.py --sweep times (48^4, 4^4 aggregates, n_vec = 20: the staged kernels in their default launch geometry):
    restriction and prolongation on sampled aggregates, each handed to the oracle as a 4^4 lattice of its own (one block).
    Inputs are gathered from the device inputs, never from outputs."""
    dims, bdims, nvec = [48] * 4, [4] * 4, 20
    cdims = [12] * 4
    V, Vc, nb = syn.volume(dims), syn.volume(cdims), 2 * nvec
    d = torch.device("cuda", 0)
    basis = syn.spinor_torch(V * nvec, 1, 411, d).reshape(nvec, V, 4, 3)
    f = syn.spinor_torch(V, nrhs, 412, d)
    vc = syn.spinor_torch(Vc, nrhs, 413, d, ncomp=(nb,))
    tr = mrhs.Transfer(dims, bdims, nvec, nrhs, basis)
    rng = np.random.default_rng(77)
    cc = rng.integers(0, 12, size=(24, 4))
    cc[0], cc[1], cc[2] = (0, 0, 0, 0), (11, 11, 11, 11), (11, 0, 11, 0)      # corners of the coarse lattice
    # fine sites of an aggregate in the lexicographic order of a 4^4 lattice
    i = np.arange(256)
    off = np.stack([i % 4, (i // 4) % 4, (i // 16) % 4, i // 64], axis=1)
    d_f = mrhs.field_import(dims, 12, nrhs, mrhs.FULL, f)
    d_c = mrhs.empty_field(cdims, nb, nrhs, mrhs.FULL)
    d_c.fill_(float("nan"))
    torch.cuda.synchronize()
    tr.restrict(d_f, d_c)
    torch.cuda.synchronize()
    got_c = mrhs.coarse_field_export(cdims, nb, nrhs, mrhs.FULL, d_c)
    del d_f
    d_p = mrhs.empty_field(dims, 12, nrhs, mrhs.FULL)
    d_p.fill_(float("nan"))
    torch.cuda.synchronize()
    tr.prolong(mrhs.coarse_field_import(cdims, nb, nrhs, mrhs.FULL, vc), d_p)
    torch.cuda.synchronize()
    got_p = mrhs.field_export(dims, 12, nrhs, mrhs.FULL, d_p).reshape(V, 4, 3, nrhs)
    for c in cc:
        x = 4 * c[None, :] + off
        lex = torch.from_numpy(x[:, 0] + 48 * (x[:, 1] + 48 * (x[:, 2] + 48 * x[:, 3]))).to(d)
        B = int(c[0] + 12 * (c[1] + 12 * (c[2] + 12 * c[3])))
        b_sub, f_sub = host(basis[:, lex]), host(f[lex])
        want = otr.restrict([4] * 4, [4] * 4, b_sub, f_sub)[0]
        assert rel_l2_per_rhs(host(got_c[B]), want).max() < TOL, ("restrict", c)
        want = otr.prolong([4] * 4, [4] * 4, b_sub, host(vc[B])[None])
        assert rel_l2_per_rhs(host(got_p[lex]), want).max() < TOL, ("prolong", c)
    tr.close()

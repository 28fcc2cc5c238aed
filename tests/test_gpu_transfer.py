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

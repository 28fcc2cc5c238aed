"""GPU parity of the coarse-level 9-point stencil against the fp64 oracle (SURVEY.md
Sec. 8(a) row a5; configs 3 and 4 of BASELINE.json).  Through the C-ABI binding."""
import numpy as np
import pytest

import synth_inputs as syn
from helpers import rel_l2_per_rhs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():
    pytest.skip("needs a CUDA device", allow_module_level=True)

import oracle                      # noqa: E402
import paper_2211_13719_b200 as mrhs   # noqa: E402
from gpu_common import TOL, dev, host   # noqa: E402


def gpu_coarse(c, v, point_mask=None):
    d_in = c.import_field(dev(v))
    d_out = c.empty()
    c.apply(d_in, d_out, point_mask)
    torch.cuda.synchronize()
    return host(c.export_field(d_out))


SMALL = [([2, 2, 2, 2], 24, n) for n in (1, 2, 4, 8, 12, 16, 24, 32, 48, 64, 96)] + \
        [([3, 2, 4, 2], 40, n) for n in (1, 2, 4, 8, 12, 16, 24, 32, 48, 64, 96)] + \
        [([5, 3, 2, 4], 24, 12), ([4, 4, 4, 6], 40, 12)]


@pytest.mark.parametrize("cdims,nb,nrhs", SMALL)
def test_coarse_apply_matches_oracle_small(cdims, nb, nrhs):
    A = syn.coarse_links_np(cdims, nb, 3)
    v = syn.coarse_vector_np(cdims, nb, nrhs, 3)
    c = mrhs.Coarse(cdims, nb, nrhs, dev(A))
    err = rel_l2_per_rhs(gpu_coarse(c, v), oracle.coarse_apply(cdims, A, v))
    assert err.max() < TOL, err
    c.close()


@pytest.mark.parametrize("nrhs", [1, 12, 24, 64])
def test_config3_intermediate_level(nrhs):
    cdims, nb = [8, 8, 8, 8], 24
    A = syn.coarse_links_np(cdims, nb, 3)
    v = syn.coarse_vector_np(cdims, nb, nrhs, 3)
    c = mrhs.Coarse(cdims, nb, nrhs, dev(A))
    err = rel_l2_per_rhs(gpu_coarse(c, v), oracle.coarse_apply(cdims, A, v))
    assert err.max() < TOL, err
    c.close()


@pytest.mark.parametrize("nrhs", [12, 24, 48, 96])
def test_config4_coarsest_level(nrhs):
    cdims, nb = [6, 6, 6, 32], 40
    A = syn.coarse_links_np(cdims, nb, 4)
    v = syn.coarse_vector_np(cdims, nb, nrhs, 4)
    c = mrhs.Coarse(cdims, nb, nrhs, dev(A))
    err = rel_l2_per_rhs(gpu_coarse(c, v), oracle.coarse_apply(cdims, A, v))
    assert err.max() < TOL, err
    # host-buffer entry
    h_in = torch.from_numpy(v).pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    mrhs.coarse_apply_host(c.h, h_in, h_out)
    err = rel_l2_per_rhs(h_out.numpy(), oracle.coarse_apply(cdims, A, v))
    assert err.max() < TOL, err
    # asynchronous entry: five calls in flight over the three staging slots, one wait
    outs = [torch.full_like(h_in, float("nan")).pin_memory() for _ in range(5)]
    for o in outs:
        mrhs.coarse_apply_host_async(c.h, h_in, o)
    mrhs.coarse_host_wait(c.h)
    for o in outs:
        assert np.array_equal(o.numpy(), h_out.numpy())
    c.close()


# ---- row a6: the tensor-core variants (tcgen05 kind::tf32 with hi/lo tf32 operands split in the kernel; kind::f16 with hi/lo
# fp16 operands split beforehand after a power-of-two scaling) are held to the same tolerance
TC_MODES = [mrhs.COARSE_TENSOR, mrhs.COARSE_TENSOR_F16]
TC_SMALL = [([2, 2, 2, 2], 24, n) for n in (2, 4, 8, 12, 16, 24, 32, 48, 64, 96)] + \
           [([3, 2, 4, 2], 40, n) for n in (2, 4, 8, 12, 16, 24, 32, 48, 64, 96)] + \
           [([5, 3, 2, 4], 24, 12), ([4, 4, 4, 6], 40, 12), ([7, 5, 3, 11], 40, 24)]


@pytest.mark.parametrize("mode", TC_MODES)
@pytest.mark.parametrize("cdims,nb,nrhs", TC_SMALL)
def test_coarse_tensor_core_matches_oracle_small(cdims, nb, nrhs, mode):
    A = syn.coarse_links_np(cdims, nb, 3)
    v = syn.coarse_vector_np(cdims, nb, nrhs, 3)
    c = mrhs.Coarse(cdims, nb, nrhs, dev(A), math_mode=mode)
    want = oracle.coarse_apply(cdims, A, v)
    err = rel_l2_per_rhs(gpu_coarse(c, v), want)
    assert err.max() < TOL, err
    # a second apply on the same handle (persistent barrier phases, reused TMEM) gives the same result
    err = rel_l2_per_rhs(gpu_coarse(c, v), want)
    assert err.max() < TOL, err
    c.close()


@pytest.mark.parametrize("nrhs", [12, 24, 48, 96])
def test_config4_tensor_core(nrhs):
    cdims, nb = [6, 6, 6, 32], 40
    A = syn.coarse_links_np(cdims, nb, 4)
    v = syn.coarse_vector_np(cdims, nb, nrhs, 4)
    want = oracle.coarse_apply(cdims, A, v)
    c = mrhs.Coarse(cdims, nb, nrhs, dev(A), math_mode=1)
    err_tc = rel_l2_per_rhs(gpu_coarse(c, v), want)
    assert err_tc.max() < TOL, err_tc
    c.close()
    c = mrhs.Coarse(cdims, nb, nrhs, dev(A), math_mode=2)
    err_h16 = rel_l2_per_rhs(gpu_coarse(c, v), want)
    assert err_h16.max() < TOL, err_h16
    # a second apply reuses the split-vector scratch, the column maxima and the barrier phases
    err_h16 = rel_l2_per_rhs(gpu_coarse(c, v), want)
    assert err_h16.max() < TOL, err_h16
    c.close()
    # the two math modes agree with each other far inside the tolerance
    c0 = mrhs.Coarse(cdims, nb, nrhs, dev(A), math_mode=0)
    err_fma = rel_l2_per_rhs(gpu_coarse(c0, v), want)
    c0.close()
    assert err_fma.max() < TOL, err_fma
    assert err_tc.max() < 20 * max(err_fma.max(), 1e-7), (err_tc.max(), err_fma.max())


@pytest.mark.parametrize("mode", TC_MODES)
@pytest.mark.parametrize("nrhs", [12, 64])
def test_config3_tensor_core(nrhs, mode):
    cdims, nb = [8, 8, 8, 8], 24
    A = syn.coarse_links_np(cdims, nb, 3)
    v = syn.coarse_vector_np(cdims, nb, nrhs, 3)
    c = mrhs.Coarse(cdims, nb, nrhs, dev(A), math_mode=mode)
    err = rel_l2_per_rhs(gpu_coarse(c, v), oracle.coarse_apply(cdims, A, v))
    assert err.max() < TOL, err
    c.close()


@pytest.mark.parametrize("mode", TC_MODES)
def test_coarse_tensor_core_rejects_odd_nrhs(mode):
    cdims, nb = [2, 2, 2, 2], 24
    A = dev(syn.coarse_links_np(cdims, nb, 3))
    with pytest.raises(mrhs.MrhsError) as e:
        mrhs.Coarse(cdims, nb, 1, A, math_mode=mode)
    assert e.value.status == mrhs.ERR_UNSUPPORTED


@pytest.mark.parametrize("cdims,nb,nrhs", [([4, 2, 6, 2], 24, 12), ([3, 2, 4, 2], 40, 24)])
def test_coarse_fp16_split_scales(cdims, nb, nrhs):
    """math_mode 2 represents every number as two fp16 parts after a power-of-two scaling: per site for the links, per RHS for
    the vectors.  Right-hand sides and sites of very different magnitudes (1e-12 .. 1e+12, far outside the fp16 range), a zero
    RHS and a RHS that is a point source must come out within the tolerance per RHS."""
    rng = np.random.default_rng(11)
    A = syn.coarse_links_np(cdims, nb, 3)
    nsites = int(np.prod(cdims))
    site_mag = (10.0 ** rng.uniform(-6, 6, size=nsites)).astype(np.float32)
    A = (A.reshape(nsites, -1) * site_mag[:, None]).reshape(A.shape).astype(np.complex64)
    v = syn.coarse_vector_np(cdims, nb, nrhs, 3)
    col_mag = (10.0 ** np.linspace(-12, 12, nrhs)).astype(np.float32)
    v = (v * col_mag).astype(np.complex64)
    v[..., 3] = 0                                   # a zero right-hand side
    v[..., 5] = 0
    v.reshape(nsites, nb, nrhs)[nsites // 2, 7, 5] = 3.0e-5 - 2.0e-5j     # a point source
    c = mrhs.Coarse(cdims, nb, nrhs, dev(A), math_mode=2)
    got = gpu_coarse(c, v)
    want = oracle.coarse_apply(cdims, A, v)
    assert np.all(got[..., 3] == 0)
    keep = [n for n in range(nrhs) if n != 3]
    err = rel_l2_per_rhs(got[..., keep], want[..., keep])
    assert err.max() < TOL, err
    # the column maxima of an apply do not leak into the next one on the handle: a much smaller input afterwards keeps its accuracy
    # (with stale maxima its fp16 parts would underflow to zero), and so does the first input once more
    small = (v * np.float32(1e-20)).astype(np.complex64)
    err = rel_l2_per_rhs(gpu_coarse(c, small)[..., keep], oracle.coarse_apply(cdims, A, small)[..., keep])
    assert err.max() < TOL, err
    err = rel_l2_per_rhs(gpu_coarse(c, v)[..., keep], want[..., keep])
    assert err.max() < TOL, err
    c.close()


# ---- subsets of the stencil (NEXT-1): stand-alone self term, 8-point hopping term, single points; both math modes
@pytest.mark.parametrize("mode", mrhs.COARSE_MODES)
@pytest.mark.parametrize("cdims,nb,nrhs", [([4, 2, 6, 2], 24, 12), ([3, 4, 2, 5], 40, 24), ([2, 2, 2, 2], 40, 96)])
def test_coarse_point_subsets_match_oracle(cdims, nb, nrhs, mode):
    A = syn.coarse_links_np(cdims, nb, 7)
    v = syn.coarse_vector_np(cdims, nb, nrhs, 7)
    c = mrhs.Coarse(cdims, nb, nrhs, dev(A), math_mode=mode)
    for mask in (mrhs.COARSE_SELF, mrhs.COARSE_HOP, mrhs.COARSE_ALL, 1 << 3, 1 << 8, 0x0AA, 0x155):
        want = oracle.coarse_apply(cdims, A, v, pmask=mask)
        err = rel_l2_per_rhs(gpu_coarse(c, v, mask), want)
        assert err.max() < TOL, (hex(mask), err)
    with pytest.raises(mrhs.MrhsError):
        c.apply(c.empty(), c.empty(), 0)
    c.close()


def test_coarse_errors():
    cdims, nb = [2, 2, 2, 2], 24
    A = dev(syn.coarse_links_np(cdims, nb, 3))
    with pytest.raises(mrhs.MrhsError) as e:
        mrhs.Coarse(cdims, nb, 5, A)
    assert e.value.status == mrhs.ERR_UNSUPPORTED
    c = mrhs.Coarse(cdims, nb, 4, A)
    f = c.empty()
    with pytest.raises(mrhs.MrhsError):
        c.apply(f, f)
    c.close()


# ---- NEXT-1: checkerboarded coarse fields and coarse M_eooe, both math modes, both parities
MEOOE_CASES = [([4, 2, 6, 2], 24, 12), ([2, 4, 2, 6], 40, 24), ([2, 2, 2, 2], 40, 96), ([6, 4, 2, 4], 24, 1), ([8, 4, 4, 6], 40, 12)]


@pytest.mark.parametrize("mode", mrhs.COARSE_MODES)
@pytest.mark.parametrize("cdims,nb,nrhs", MEOOE_CASES)
def test_coarse_meooe_matches_oracle(cdims, nb, nrhs, mode):
    if mode != mrhs.COARSE_FMA and nrhs % 2:
        pytest.skip("the tensor-core variants need an even N_rhs")
    A = syn.coarse_links_np(cdims, nb, 8)
    v = syn.coarse_vector_np(cdims, nb, nrhs, 8)
    src = oracle.cb_split(cdims, v)
    c = mrhs.Coarse(cdims, nb, nrhs, dev(A), math_mode=mode)
    for out_parity in (0, 1):
        want = oracle.coarse_meooe(cdims, A, src[1 - out_parity], out_parity)
        d_in = c.import_field(dev(src[1 - out_parity]), 1 - out_parity)
        d_out = c.empty(parity=out_parity)
        c.meooe(d_in, d_out, out_parity)
        torch.cuda.synchronize()
        err = rel_l2_per_rhs(host(c.export_field(d_out, out_parity)), want)
        assert err.max() < TOL, (out_parity, err)
    with pytest.raises(mrhs.MrhsError):
        c.meooe(c.empty(parity=0), c.empty(parity=1), 2)
    c.close()


def test_coarse_meooe_needs_even_extents():
    cdims, nb, nrhs = [3, 2, 2, 2], 24, 4
    c = mrhs.Coarse(cdims, nb, nrhs, dev(syn.coarse_links_np(cdims, nb, 9)))
    with pytest.raises(mrhs.MrhsError) as e:
        c.meooe(c.empty(), c.empty(), 0)
    assert e.value.status == mrhs.ERR_INVALID_ARG
    c.close()


@pytest.mark.parametrize("cdims,nb,nrhs", [([4, 2, 6, 2], 24, 12), ([2, 2, 4, 2], 12, 3), ([2, 4, 2, 2], 12, 4)])
def test_coarse_layout_round_trips_are_bit_exact(cdims, nb, nrhs):
    """Checkerboarded coarse fields: import / export and split / merge against the oracle-side canonical split; nb = 12
    (a coarse level with n_vec = 6) goes through the explicit coarse entries and is NOT packed like a fine spinor."""
    v = syn.coarse_vector_np(cdims, nb, nrhs, 10)
    d = dev(v)
    nat = mrhs.coarse_field_import(cdims, nb, nrhs, mrhs.FULL, d)
    assert torch.equal(mrhs.coarse_field_export(cdims, nb, nrhs, mrhs.FULL, nat), d)
    ev = mrhs.empty_field(cdims, nb, nrhs, mrhs.EVEN)
    od = mrhs.empty_field(cdims, nb, nrhs, mrhs.ODD)
    mrhs.coarse_cb_split(cdims, nb, nrhs, nat, ev, od)
    ve, vo = oracle.cb_split(cdims, v)
    assert np.array_equal(host(mrhs.coarse_field_export(cdims, nb, nrhs, mrhs.EVEN, ev)), ve)
    assert np.array_equal(host(mrhs.coarse_field_export(cdims, nb, nrhs, mrhs.ODD, od)), vo)
    assert torch.equal(mrhs.coarse_field_import(cdims, nb, nrhs, mrhs.ODD, dev(vo)), od)
    full2 = torch.zeros_like(nat)
    mrhs.coarse_cb_merge(cdims, nb, nrhs, ev, od, full2)
    assert torch.equal(full2, nat)
    # the coarse layout is site-contiguous: one site's nb x nrhs block is one run of the native field
    if nrhs % 2 == 0:
        site = host(nat).reshape(-1, nb, nrhs // 2, 4)[1]
        assert np.array_equal(site[:, :, 0] + 1j * site[:, :, 2], v[1][:, 0::2])

"""GPU parity of the fine-level kernels against the fp64 oracle (SURVEY.md Sec. 8(a) rows
a0-a4, a7; configs 1, 2 and 5 of BASELINE.json).  Everything goes through the C-ABI binding."""
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
from gpu_common import TOL, dev, gpu_dhop, gpu_meooe, gpu_mooee, host, make_wilson   # noqa: E402


def _fine_case(dims, nrhs, seed, mass, csw):
    U = syn.gauge_np(dims, seed)
    psi = syn.spinor_np(syn.volume(dims), nrhs, seed)
    return U, psi


# config 1 first; then shapes that exercise x-blocks with several blocks per line, ragged thread
# blocks (threads not a multiple of 32), extent-2 directions, odd N (scalar path) and N = 1.
FINE_CASES = [
    ([4, 4, 4, 4], 4, 0, -0.1, 1.0),
    ([4, 4, 4, 4], 1, 1, -0.1, 1.0),
    ([8, 4, 6, 2], 3, 2, 0.2, 1.3),
    ([2, 2, 2, 2], 2, 3, 0.0, 1.0),
    ([12, 6, 4, 10], 12, 4, -0.05, 1.5),
    ([48, 4, 2, 4], 12, 5, -0.05, 1.5),
    ([16, 8, 2, 4], 24, 6, -0.05, 1.5),
    ([8, 4, 4, 4], 96, 7, -0.05, 1.5),
    ([32, 2, 4, 6], 1, 8, -0.05, 1.5),
]


@pytest.mark.parametrize("dims,nrhs,seed,mass,csw", FINE_CASES)
def test_dhop_meooe_mooee_match_oracle(dims, nrhs, seed, mass, csw):
    U, psi = _fine_case(dims, nrhs, seed, mass, csw)
    w = make_wilson(dims, nrhs, mass, csw, U)
    # D_hop, full lattice (row a2)
    want = oracle.dhop(dims, U, psi)
    got = gpu_dhop(w, psi)
    err = rel_l2_per_rhs(got, want)
    assert err.max() < TOL, ("dhop", err)
    # M_eooe, both parities (row a3)
    pe, po = oracle.cb_split(dims, psi)
    for out_parity, src in ((0, po), (1, pe)):
        want = oracle.meooe(dims, U, src, out_parity)
        got = gpu_meooe(w, src, out_parity)
        err = rel_l2_per_rhs(got, want)
        assert err.max() < TOL, ("meooe", out_parity, err)
    # clover construction on the device (row a0) and M_ooee on full / even / odd fields (row a4)
    C, _ = oracle.clover_blocks(dims, U, mass, csw)
    Cg = torch.full((syn.volume(dims), 2, 6, 6), float("nan"), dtype=torch.complex64, device="cuda")
    mrhs.wilson_export_clover(w.h, Cg)
    cerr = np.linalg.norm(host(Cg) - C) / np.linalg.norm(C)
    assert cerr < 1e-6, cerr
    want = oracle.mooee(C, psi)
    err = rel_l2_per_rhs(gpu_mooee(w, psi, mrhs.FULL), want)
    assert err.max() < TOL, ("mooee full", err)
    Ce, Co = oracle.cb_split(dims, C)
    for parity, Cp, src in ((0, Ce, pe), (1, Co, po)):
        err = rel_l2_per_rhs(gpu_mooee(w, src, parity), oracle.mooee(Cp, src))
        assert err.max() < TOL, ("mooee", parity, err)
    w.close()


def test_user_supplied_clover_is_used():
    dims, nrhs = [4, 4, 4, 4], 4
    U, psi = _fine_case(dims, nrhs, 11, 0.0, 1.0)
    rng = np.random.default_rng(5)
    A = rng.standard_normal((256, 2, 6, 6)) + 1j * rng.standard_normal((256, 2, 6, 6))
    C = (A + np.conj(np.swapaxes(A, 2, 3))).astype(np.complex64)     # Hermitian blocks
    w = make_wilson(dims, nrhs, 0.0, 1.0, U, clover=C)
    err = rel_l2_per_rhs(gpu_mooee(w, psi, mrhs.FULL), oracle.mooee(C, psi))
    assert err.max() < TOL, err
    w.close()


def test_layout_round_trips_are_bit_exact():
    dims, nrhs = [12, 4, 6, 2], 12
    psi = syn.spinor_np(syn.volume(dims), nrhs, 21)
    d = dev(psi)
    nat = mrhs.field_import(dims, 12, nrhs, mrhs.FULL, d)
    back = mrhs.field_export(dims, 12, nrhs, mrhs.FULL, nat)
    assert torch.equal(back.reshape(d.shape), d)
    # full native -> even/odd native -> canonical equals the oracle-side canonical split
    ev = mrhs.empty_field(dims, 12, nrhs, mrhs.EVEN)
    od = mrhs.empty_field(dims, 12, nrhs, mrhs.ODD)
    mrhs.cb_split(dims, 12, nrhs, nat, ev, od)
    pe, po = oracle.cb_split(dims, psi)
    assert np.array_equal(host(mrhs.field_export(dims, 12, nrhs, mrhs.EVEN, ev)).reshape(pe.shape), pe)
    assert np.array_equal(host(mrhs.field_export(dims, 12, nrhs, mrhs.ODD, od)).reshape(po.shape), po)
    full2 = torch.zeros_like(nat)
    mrhs.cb_merge(dims, 12, nrhs, ev, od, full2)
    assert torch.equal(full2, nat)


def test_tilings_give_identical_results():
    dims, nrhs = [16, 8, 8, 8], 12
    U, psi = _fine_case(dims, nrhs, 31, -0.05, 1.5)
    w = make_wilson(dims, nrhs, -0.05, 1.5, U)
    ref = gpu_dhop(w, psi)
    pe, po = oracle.cb_split(dims, psi)
    ref_e = gpu_meooe(w, po, 0)
    for tile, chunk in (([1, 1, 1], [1, 1]), ([2, 2, 2], [2, 1]), ([4, 2, 1], [1, 2]), ([2, 4, 1], [2, 2])):
        mrhs.wilson_set_tiling(w.h, 0, tile, chunk)
        mrhs.wilson_set_tiling(w.h, 1, tile, chunk)
        assert mrhs.wilson_get_tiling(w.h, 0) == (tile, chunk)
        assert np.array_equal(gpu_dhop(w, psi), ref)
        assert np.array_equal(gpu_meooe(w, po, 0), ref_e)
    with pytest.raises(mrhs.MrhsError):
        mrhs.wilson_set_tiling(w.h, 0, [3, 2, 2], [1, 1])       # 3 does not divide 8
    with pytest.raises(mrhs.MrhsError):
        mrhs.wilson_set_tiling(w.h, 0, [8, 8, 8], [1, 1])       # too many threads
    w.close()


# ---- the two hop kernels (gather, slice sweep) compute the same map: both against the oracle, and the sweep
# kernel under several segment lengths / chunk shapes (prologue slice, wrap in t, partly filled warps, x-blocks
# of 2..16 sites, checkerboarded half lines of 6 sites, extent-2 directions)
KERNEL_CASES = [
    ([4, 4, 4, 4], 4, 40),
    ([2, 2, 2, 2], 2, 41),
    ([12, 6, 4, 10], 12, 42),
    ([48, 4, 2, 4], 12, 43),
    ([24, 4, 4, 6], 12, 44),
    ([16, 8, 2, 4], 24, 45),
    ([8, 4, 4, 4], 96, 46),
    ([16, 4, 6, 8], 48, 47),
    ([32, 2, 4, 6], 4, 48),
    ([16, 4, 4, 4], 12, 49),      # checkerboarded half line of 8 sites at N_rhs = 12: the instantiation config 5 runs
    ([32, 4, 2, 6], 12, 50),
]


@pytest.mark.parametrize("dims,nrhs,seed", KERNEL_CASES)
def test_gather_and_sweep_kernels_match_oracle(dims, nrhs, seed):
    U, psi = _fine_case(dims, nrhs, seed, -0.05, 1.5)
    w = make_wilson(dims, nrhs, -0.05, 1.5, U)
    assert mrhs.wilson_get_hop_kernel(w.h, 0) == mrhs.HOP_GATHER     # the default on small lattices (sweep from 32^4, N_rhs >= 12)
    want = oracle.dhop(dims, U, psi)
    pe, po = oracle.cb_split(dims, psi)
    want_cb = [oracle.meooe(dims, U, po, 0), oracle.meooe(dims, U, pe, 1)]
    T = dims[3]
    settings = [(mrhs.HOP_GATHER, None), (mrhs.HOP_SWEEP, None), (mrhs.HOP_SWEEP, (T, [1, 1])),
                (mrhs.HOP_SWEEP, (2, [dims[1] // 2, 1])), (mrhs.HOP_SWEEP, (1, [1, dims[2] // 2]))]
    results = []
    for kern, sweep in settings:
        for which in (0, 1):
            mrhs.wilson_set_hop_kernel(w.h, which, kern)
            if sweep is not None:
                mrhs.wilson_set_sweep(w.h, which, sweep[0], sweep[1])
                assert mrhs.wilson_get_sweep(w.h, which) == (sweep[0], sweep[1])
        got = gpu_dhop(w, psi)
        assert rel_l2_per_rhs(got, want).max() < TOL, ("dhop", kern, sweep)
        for out_parity, src in ((0, po), (1, pe)):
            g = gpu_meooe(w, src, out_parity)
            assert rel_l2_per_rhs(g, want_cb[out_parity]).max() < TOL, ("meooe", out_parity, kern, sweep)
        results.append(got)
    # every sweep setting adds the eight hops in the same order: bit-identical results
    for r in results[2:]:
        assert np.array_equal(r, results[1])
    with pytest.raises(mrhs.MrhsError):
        mrhs.wilson_set_sweep(w.h, 0, 3 if T % 3 else T + 1, [1, 1])     # does not divide T
    w.close()


def test_sweep_kernel_needs_even_nrhs():
    dims = [4, 4, 4, 4]
    U, psi = _fine_case(dims, 3, 50, 0.0, 1.0)
    w = make_wilson(dims, 3, 0.0, 1.0, U)
    assert mrhs.wilson_get_hop_kernel(w.h, 0) == mrhs.HOP_GATHER
    with pytest.raises(mrhs.MrhsError) as e:
        mrhs.wilson_set_hop_kernel(w.h, 0, mrhs.HOP_SWEEP)
    assert e.value.status == mrhs.ERR_UNSUPPORTED
    w.close()


def test_argument_errors():
    dims, nrhs = [4, 4, 4, 4], 4
    U, psi = _fine_case(dims, nrhs, 41, 0.0, 1.0)
    w = make_wilson(dims, nrhs, 0.0, 1.0, U)
    f = w.empty(mrhs.FULL)
    with pytest.raises(mrhs.MrhsError) as e:
        w.dhop(f, f)
    assert e.value.status == mrhs.ERR_INVALID_ARG
    with pytest.raises(mrhs.MrhsError):
        w.meooe(f, w.empty(mrhs.EVEN), 2)
    with pytest.raises(mrhs.MrhsError):
        w.mooee(f, w.empty(mrhs.FULL), 3)
    with pytest.raises(mrhs.MrhsError):
        w.dhop(f[1:], w.empty(mrhs.FULL))       # misaligned
    # overlapping (not just identical) buffers are rejected: out starts inside in
    big = torch.empty(2 * f.numel(), dtype=torch.float32, device=f.device)
    with pytest.raises(mrhs.MrhsError) as e:
        w.dhop(big[:f.numel()], big[f.numel() // 2: f.numel() // 2 + f.numel()])
    assert e.value.status == mrhs.ERR_INVALID_ARG
    half = w.empty(mrhs.EVEN).numel()
    with pytest.raises(mrhs.MrhsError):
        w.meooe(big[:half], big[half - 4: 2 * half - 4], mrhs.ODD)
    w.dhop(big[:f.numel()], big[f.numel():])    # adjacent halves are fine
    torch.cuda.synchronize()
    w.close()


def test_schur_sequence_and_host_entry():
    dims, nrhs, mass, csw = [8, 8, 4, 4], 12, -0.05, 1.5
    U, psi = _fine_case(dims, nrhs, 51, mass, csw)
    w = make_wilson(dims, nrhs, mass, csw, U)
    C, _ = oracle.clover_blocks(dims, U, mass, csw)
    Ce, Co = oracle.cb_split(dims, C)
    pe, po = oracle.cb_split(dims, psi)
    want = oracle.meooe(dims, U, oracle.mooee(Co, oracle.meooe(dims, U, pe, 1)), 0)
    d_in = w.import_field(dev(pe), mrhs.EVEN)
    t0, t1, d_out = w.empty(mrhs.ODD), w.empty(mrhs.ODD), w.empty(mrhs.EVEN)
    w.schur_sequence(d_in, t0, t1, d_out)
    torch.cuda.synchronize()
    err = rel_l2_per_rhs(host(w.export_field(d_out, mrhs.EVEN)), want)
    assert err.max() < TOL, err
    # host-buffer entry: canonical host in -> canonical host out
    h_in = torch.from_numpy(psi).pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    mrhs.wilson_apply_host(w.h, mrhs.OP_DHOP, 0, h_in, h_out)
    err = rel_l2_per_rhs(h_out.numpy(), oracle.dhop(dims, U, psi))
    assert err.max() < TOL, err
    h_in = torch.from_numpy(po).pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    mrhs.wilson_apply_host(w.h, mrhs.OP_MEOOE, 0, h_in, h_out)
    err = rel_l2_per_rhs(h_out.numpy(), oracle.meooe(dims, U, po, 0))
    assert err.max() < TOL, err
    # the asynchronous entries: five calls of four operators in flight over the three staging slots, one wait
    h_psi, h_pe, h_po = (torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (psi, pe, po))
    outs = [torch.full_like(h_psi, float("nan")).pin_memory(), torch.full_like(h_pe, float("nan")).pin_memory(),
            torch.full_like(h_po, float("nan")).pin_memory(), torch.full_like(h_psi, float("nan")).pin_memory(),
            torch.full_like(h_pe, float("nan")).pin_memory()]
    mrhs.wilson_apply_host_async(w.h, mrhs.OP_DHOP, 0, h_psi, outs[0])
    mrhs.wilson_apply_host_async(w.h, mrhs.OP_MEOOE, mrhs.EVEN, h_po, outs[1])
    mrhs.wilson_apply_host_async(w.h, mrhs.OP_MEOOE, mrhs.ODD, h_pe, outs[2])
    mrhs.wilson_apply_host_async(w.h, mrhs.OP_MOOEE, mrhs.FULL, h_psi, outs[3])
    mrhs.wilson_apply_host_async(w.h, mrhs.OP_SCHUR, 0, h_pe, outs[4])
    mrhs.wilson_host_wait(w.h)
    wants = [oracle.dhop(dims, U, psi), oracle.meooe(dims, U, po, 0), oracle.meooe(dims, U, pe, 1), oracle.mooee(C, psi), want]
    for i, (o, wnt) in enumerate(zip(outs, wants)):
        assert rel_l2_per_rhs(o.numpy(), wnt).max() < TOL, ("async host entry", i)
    w.close()


# [16, 4, 4, 4] and [32, 2, 4, 4] at N_rhs = 12 have checkerboarded half lines cut in x-blocks of 8 sites: the
# hop_sweep_kernel<8, 6, .., ..> instantiations that config 5 (48^4) and bench.py run
FUSED_CASES = [([8, 8, 4, 4], 12, 60), ([4, 4, 4, 4], 4, 61), ([24, 4, 2, 6], 12, 62), ([16, 2, 4, 4], 24, 63),
               ([8, 4, 6, 2], 3, 64), ([4, 4, 4, 4], 1, 65), ([16, 4, 4, 4], 12, 66), ([32, 2, 4, 4], 12, 67),
               ([48, 2, 2, 4], 12, 68)]


@pytest.mark.parametrize("dims,nrhs,seed", FUSED_CASES)
def test_fused_meooe_mooee_and_schur_sequence(dims, nrhs, seed):
    """out = M_ooee M_eooe in (one launch with the sweep kernel, two with the gather kernel; odd N_rhs takes
    the gather path) and the Schur sequence built on it, both parities, both kernels, against the oracle."""
    mass, csw = -0.05, 1.5
    U, psi = _fine_case(dims, nrhs, seed, mass, csw)
    w = make_wilson(dims, nrhs, mass, csw, U)
    C, _ = oracle.clover_blocks(dims, U, mass, csw)
    Cp = oracle.cb_split(dims, C)
    src = oracle.cb_split(dims, psi)
    kernels = [mrhs.HOP_GATHER] + ([mrhs.HOP_SWEEP] if nrhs % 2 == 0 else [])
    for kern in kernels:
        mrhs.wilson_set_hop_kernel(w.h, 1, kern)
        for out_parity in (0, 1):
            want = oracle.mooee(Cp[out_parity], oracle.meooe(dims, U, src[1 - out_parity], out_parity))
            d_in = w.import_field(dev(src[1 - out_parity]), 1 - out_parity)
            d_out = w.empty(out_parity)
            w.meooe_mooee(d_in, d_out, out_parity)
            torch.cuda.synchronize()
            err = rel_l2_per_rhs(host(w.export_field(d_out, out_parity)), want)
            assert err.max() < TOL, ("fused", kern, out_parity, err)
        want = oracle.meooe(dims, U, oracle.mooee(Cp[1], oracle.meooe(dims, U, src[0], 1)), 0)
        d_in = w.import_field(dev(src[0]), mrhs.EVEN)
        t0, t1, d_out = w.empty(mrhs.ODD), w.empty(mrhs.ODD), w.empty(mrhs.EVEN)
        w.schur_sequence(d_in, t0, t1, d_out)
        torch.cuda.synchronize()
        err = rel_l2_per_rhs(host(w.export_field(d_out, mrhs.EVEN)), want)
        assert err.max() < TOL, ("schur", kern, err)
    w.close()


@pytest.mark.parametrize("dims,nrhs,seed", [([8, 4, 4, 6], 12, 70), ([4, 4, 4, 4], 3, 71), ([24, 2, 4, 2], 24, 72), ([16, 4, 2, 4], 12, 73)])
def test_inverse_clover_blocks(dims, nrhs, seed):
    """M_ooee^-1 (inverse blocks built on the device at create) on full / even / odd fields, M_ooee^-1 M_ooee = 1,
    and the fused M_ooee^-1 M_eooe with both hop kernels, against the oracle (inverse by numpy.linalg.inv)."""
    mass, csw = -0.05, 1.5
    U, psi = _fine_case(dims, nrhs, seed, mass, csw)
    w = make_wilson(dims, nrhs, mass, csw, U)
    C, _ = oracle.clover_blocks(dims, U, mass, csw)
    Ci = oracle.clover_inverse(C)
    Cip = oracle.cb_split(dims, Ci)
    src = oracle.cb_split(dims, psi)

    def apply_inv(field, parity):
        d_in = w.import_field(dev(field), parity)
        d_out = w.empty(parity)
        w.mooee_inv(d_in, d_out, parity)
        torch.cuda.synchronize()
        return host(w.export_field(d_out, parity))

    assert rel_l2_per_rhs(apply_inv(psi, mrhs.FULL), oracle.mooee(Ci, psi)).max() < TOL
    for parity in (0, 1):
        assert rel_l2_per_rhs(apply_inv(src[parity], parity), oracle.mooee(Cip[parity], src[parity])).max() < TOL
    back = apply_inv(gpu_mooee(w, psi, mrhs.FULL), mrhs.FULL)
    assert rel_l2_per_rhs(back, psi.astype(np.complex128)).max() < TOL
    kernels = [mrhs.HOP_GATHER] + ([mrhs.HOP_SWEEP] if nrhs % 2 == 0 else [])
    for kern in kernels:
        mrhs.wilson_set_hop_kernel(w.h, 1, kern)
        for out_parity in (0, 1):
            want = oracle.mooee(Cip[out_parity], oracle.meooe(dims, U, src[1 - out_parity], out_parity))
            d_in = w.import_field(dev(src[1 - out_parity]), 1 - out_parity)
            d_out = w.empty(out_parity)
            w.meooe_mooee_inv(d_in, d_out, out_parity)
            torch.cuda.synchronize()
            err = rel_l2_per_rhs(host(w.export_field(d_out, out_parity)), want)
            assert err.max() < TOL, ("fused inverse", kern, out_parity, err)
    w.close()


@pytest.mark.parametrize("dims,ncomp,nrhs,parity", [([8, 4, 6, 4], 12, 12, mrhs.FULL), ([8, 4, 6, 4], 12, 12, mrhs.ODD),
                                                    ([4, 4, 4, 4], 12, 3, mrhs.FULL), ([16, 2, 4, 6], 12, 48, mrhs.EVEN),
                                                    ([3, 5, 2, 7], 40, 24, mrhs.FULL), ([2, 2, 2, 2], 24, 1, mrhs.FULL)])
def test_inner_products_match_oracle(dims, ncomp, nrhs, parity):
    """<x_r, y_r> for all RHS at once on native fields (fine full / checkerboarded, coarse), fp64 sums, reproducible."""
    V = syn.volume(dims) // (1 if parity == mrhs.FULL else 2)
    shape = (ncomp,) if ncomp != 12 else (4, 3)
    rng = np.random.default_rng([91, nrhs])
    x = (rng.standard_normal((V,) + shape + (nrhs,)) + 1j * rng.standard_normal((V,) + shape + (nrhs,))).astype(np.complex64)
    y = (rng.standard_normal((V,) + shape + (nrhs,)) + 1j * rng.standard_normal((V,) + shape + (nrhs,))).astype(np.complex64)
    dx = mrhs.field_import(dims, ncomp, nrhs, parity, dev(x))
    dy = mrhs.field_import(dims, ncomp, nrhs, parity, dev(y))
    got = host(mrhs.inner_products(dims, ncomp, nrhs, parity, dx, dy))
    want = oracle.inner_products(x, y)
    assert np.max(np.abs(got - want) / np.abs(want)) < 1e-10, (got, want)
    assert np.array_equal(host(mrhs.inner_products(dims, ncomp, nrhs, parity, dx, dy)), got)
    nrm = host(mrhs.inner_products(dims, ncomp, nrhs, parity, dx, dx))
    assert np.max(np.abs(nrm.imag)) == 0.0 and np.all(nrm.real > 0)


def test_inner_products_leave_the_default_mempool_alone():
    """The per-call scratch comes from a pool of the library's own: the release threshold of the device's default
    stream-ordered pool (a process-wide setting that belongs to the caller) is what it was before the call."""
    import ctypes
    rt = ctypes.CDLL("libcudart.so.12")
    pool, thr0, thr1 = ctypes.c_void_p(), ctypes.c_uint64(), ctypes.c_uint64()
    torch.zeros(1).cuda()
    assert rt.cudaDeviceGetDefaultMemPool(ctypes.byref(pool), 0) == 0
    kReleaseThreshold = 4     # cudaMemPoolAttrReleaseThreshold
    assert rt.cudaMemPoolGetAttribute(pool, kReleaseThreshold, ctypes.byref(thr0)) == 0
    dims, nrhs = [4, 4, 4, 4], 4
    x = (np.random.default_rng(5).standard_normal((256, 4, 3, nrhs)) + 0j).astype(np.complex64)
    dx = mrhs.field_import(dims, 12, nrhs, mrhs.FULL, dev(x))
    for _ in range(3):
        mrhs.inner_products(dims, 12, nrhs, mrhs.FULL, dx, dx)
    torch.cuda.synchronize()
    assert rt.cudaMemPoolGetAttribute(pool, kReleaseThreshold, ctypes.byref(thr1)) == 0
    assert thr1.value == thr0.value, (thr0.value, thr1.value)


def test_site_data_copies_are_made_on_first_use_in_any_order():
    """A handle packs gauge and clover per layout on first use (checkerboarded links, backward links of the sweep kernel, clover
    and inverse clover per parity): a fresh handle whose FIRST call is the last operator of the list matches the oracle."""
    dims, nrhs = [16, 4, 4, 4], 12
    U = syn.gauge_np(dims, 81)
    psi = syn.spinor_np(syn.volume(dims), nrhs, 81)
    C, _ = oracle.clover_blocks(dims, U, -0.05, 1.5)
    Ci = oracle.clover_inverse(C)
    src = oracle.cb_split(dims, psi)
    Cp, Cip = oracle.cb_split(dims, C), oracle.cb_split(dims, Ci)
    for kern in (mrhs.HOP_GATHER, mrhs.HOP_SWEEP):
        w = make_wilson(dims, nrhs, -0.05, 1.5, U)
        mrhs.wilson_set_hop_kernel(w.h, 1, kern)
        # first call: the fused inverse launch (needs checkerboarded links + inverse blocks of one parity)
        d_in = w.import_field(dev(src[0]), mrhs.EVEN)
        d_out = w.empty(mrhs.ODD)
        d_out.fill_(float("nan"))
        torch.cuda.synchronize()
        w.meooe_mooee_inv(d_in, d_out, mrhs.ODD)
        torch.cuda.synchronize()
        want = oracle.mooee(Cip[1], oracle.meooe(dims, U, src[0], 1))
        assert rel_l2_per_rhs(host(w.export_field(d_out, mrhs.ODD)), want).max() < TOL, kern
        # then the full-lattice inverse and a checkerboarded clover apply
        d_f = w.import_field(dev(psi), mrhs.FULL)
        d_o = w.empty(mrhs.FULL)
        d_o.fill_(float("nan"))
        torch.cuda.synchronize()
        w.mooee_inv(d_f, d_o, mrhs.FULL)
        torch.cuda.synchronize()
        assert rel_l2_per_rhs(host(w.export_field(d_o, mrhs.FULL)), oracle.mooee(Ci, psi)).max() < TOL, kern
        assert rel_l2_per_rhs(gpu_mooee(w, src[0], mrhs.EVEN), oracle.mooee(Cp[0], src[0])).max() < TOL, kern
        w.close()


@pytest.mark.parametrize("dims,nrhs,seed", [([8, 4, 4, 6], 12, 75), ([4, 4, 4, 4], 3, 76), ([16, 2, 4, 4], 24, 77), ([2, 2, 2, 2], 4, 78),
                                            ([16, 4, 4, 4], 12, 79), ([48, 2, 4, 2], 12, 80)])
def test_full_wilson_clover_matrix(dims, nrhs, seed):
    """out = M in = M_ooee in - D_hop in / 2 (reading S6): one fused launch with the sweep kernel, two with the gather kernel."""
    from oracle import galerkin
    mass, csw = -0.05, 1.5
    U, psi = _fine_case(dims, nrhs, seed, mass, csw)
    w = make_wilson(dims, nrhs, mass, csw, U)
    want = galerkin.wilson_clover_apply(dims, U.astype(np.complex128), mass, csw, psi.astype(np.complex128))
    kernels = [mrhs.HOP_GATHER] + ([mrhs.HOP_SWEEP] if nrhs % 2 == 0 else [])
    for kern in kernels:
        mrhs.wilson_set_hop_kernel(w.h, 0, kern)
        d_in = w.import_field(dev(psi), mrhs.FULL)
        d_out = w.empty(mrhs.FULL)
        w.apply(d_in, d_out)
        torch.cuda.synchronize()
        err = rel_l2_per_rhs(host(w.export_field(d_out, mrhs.FULL)), want)
        assert err.max() < TOL, (kern, err)
    w.close()


@pytest.mark.parametrize("nrhs", [1, 4, 12, 24, 48])
def test_config2_24x24_full_field(nrhs):
    """Config 2 (24^4, mass -0.05, c_sw 1.5, every N_rhs of the config): full-field parity for D_hop, M_eooe (both
    parities) and M_ooee with the library's default kernels, and for the sweep kernel where N_rhs allows it."""
    dims, mass, csw = [24, 24, 24, 24], -0.05, 1.5
    U, psi = _fine_case(dims, nrhs, 2, mass, csw)
    w = make_wilson(dims, nrhs, mass, csw, U)
    want = oracle.dhop(dims, U, psi)
    pe, po = oracle.cb_split(dims, psi)
    want_cb = [oracle.meooe(dims, U, po, 0), oracle.meooe(dims, U, pe, 1)]
    kernels = [None] + ([mrhs.HOP_SWEEP] if nrhs % 2 == 0 else [])
    for kern in kernels:
        if kern is not None:
            mrhs.wilson_set_hop_kernel(w.h, 0, kern)
            mrhs.wilson_set_hop_kernel(w.h, 1, kern)
        err = rel_l2_per_rhs(gpu_dhop(w, psi), want)
        assert err.max() < TOL, (kern, err)
        for out_parity, src in ((0, po), (1, pe)):
            err = rel_l2_per_rhs(gpu_meooe(w, src, out_parity), want_cb[out_parity])
            assert err.max() < TOL, (kern, out_parity, err)
    C, _ = oracle.clover_blocks(dims, U, mass, csw)
    err = rel_l2_per_rhs(gpu_mooee(w, psi, mrhs.FULL), oracle.mooee(C, psi))
    assert err.max() < TOL, err
    w.close()


# ---- NEXT-2: adjoint operators and the even-odd preconditioned (Schur complement) operator, both hop kernels
DAG_CASES = [([8, 4, 4, 6], 12, 81), ([4, 4, 4, 4], 3, 82), ([16, 4, 4, 4], 12, 83), ([16, 2, 4, 4], 24, 84), ([2, 2, 2, 2], 4, 85),
             ([48, 2, 2, 4], 12, 86)]


@pytest.mark.parametrize("dims,nrhs,seed", DAG_CASES)
def test_dagger_variants_and_schur_operator(dims, nrhs, seed):
    from oracle import evenodd
    mass, csw = -0.05, 1.5
    U, psi = _fine_case(dims, nrhs, seed, mass, csw)
    w = make_wilson(dims, nrhs, mass, csw, U)
    C, _ = oracle.clover_blocks(dims, U, mass, csw)
    src = oracle.cb_split(dims, psi)
    want_dd = evenodd.dhop_dag(dims, U, psi)
    want_md = evenodd.wilson_clover(dims, U, C, psi, dagger=True)
    kernels = [mrhs.HOP_GATHER] + ([mrhs.HOP_SWEEP] if nrhs % 2 == 0 else [])
    for kern in kernels:
        mrhs.wilson_set_hop_kernel(w.h, 0, kern)
        mrhs.wilson_set_hop_kernel(w.h, 1, kern)
        d_in = w.import_field(dev(psi), mrhs.FULL)
        d_out = w.empty(mrhs.FULL)
        w.dhop_dag(d_in, d_out)
        torch.cuda.synchronize()
        assert rel_l2_per_rhs(host(w.export_field(d_out, mrhs.FULL)), want_dd).max() < TOL, ("dhop_dag", kern)
        d_out = w.empty(mrhs.FULL)
        w.apply(d_in, d_out, dagger=True)
        torch.cuda.synchronize()
        assert rel_l2_per_rhs(host(w.export_field(d_out, mrhs.FULL)), want_md).max() < TOL, ("M^+", kern)
        for out_parity in (0, 1):
            c_in = w.import_field(dev(src[1 - out_parity]), 1 - out_parity)
            c_out = w.empty(out_parity)
            w.meooe_dag(c_in, c_out, out_parity)
            torch.cuda.synchronize()
            want = evenodd.meooe_dag(dims, U, src[1 - out_parity], out_parity)
            assert rel_l2_per_rhs(host(w.export_field(c_out, out_parity)), want).max() < TOL, ("meooe_dag", kern, out_parity)
        for dagger in (False, True):
            e_in = w.import_field(dev(src[0]), mrhs.EVEN)
            tmp, e_out = w.empty(mrhs.ODD), w.empty(mrhs.EVEN)
            w.schur_apply(e_in, tmp, e_out, dagger)
            torch.cuda.synchronize()
            want = evenodd.schur(dims, U, C, src[0], dagger=dagger)
            assert rel_l2_per_rhs(host(w.export_field(e_out, mrhs.EVEN)), want).max() < TOL, ("schur", kern, dagger)
    with pytest.raises(mrhs.MrhsError):
        f = w.empty(mrhs.EVEN)
        w.schur_apply(f, w.empty(mrhs.ODD), f)
    w.close()

"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (library
default tiling), on sampled output sites the oracle computes one by one (SURVEY.md Sec. 8(d)
"Parity at 48^4"): config 5 (48^4, N_rhs in {1, 12, 24}) for D_hop, M_eooe, M_ooee, the fused
M_ooee M_eooe launch, the Schur-style sequence (row a7) and the full matrix; config 4 (6^3x32,
nb = 40) full-field is in test_gpu_coarse.py.  N_rhs = 24 is the one shape whose fields pass 2^31
floats (64-bit indexing); N_rhs = 1 runs the scalar gather kernel at full size.  The stencils are
local, so the oracle needs only the sampled sites' neighbours and links, gathered from the device
inputs (never from outputs)."""
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
from gpu_common import TOL   # noqa: E402

DIMS, MASS, CSW, SEED = [48, 48, 48, 48], -0.05, 1.5, 5
NSAMPLE = 4096


def _sample_sites(dims, n, seed):
    """Seeded sample of lex indices that includes every corner and sites on every face."""
    X, Y, Z, T = dims
    rng = np.random.default_rng([seed, 0x9E])
    c = rng.integers(0, [X, Y, Z, T], size=(n, 4))
    k = 0
    for cx in (0, X - 1):                       # 16 corners
        for cy in (0, Y - 1):
            for cz in (0, Z - 1):
                for ct in (0, T - 1):
                    c[k] = (cx, cy, cz, ct); k += 1
    for mu in range(4):                         # 64 sites on each of the 8 faces
        for edge in (0, dims[mu] - 1):
            c[k:k + 64, mu] = edge; k += 64
    lex = c[:, 0] + X * (c[:, 1] + Y * (c[:, 2] + Z * c[:, 3]))
    return np.unique(lex)


def _nbr_lex(dims, lex, mu, sign):
    X, Y, Z, T = dims
    c = [lex % X, (lex // X) % Y, (lex // (X * Y)) % Z, lex // (X * Y * Z)]
    c[mu] = (c[mu] + sign) % dims[mu]
    return c[0] + X * (c[1] + Y * (c[2] + Z * c[3]))


def _gather_hop_inputs(dims, U_dev, psi_dev, lex, cb):
    """links [n][8][3][3] (U_mu(x), then U_mu(x-mu)) and nbrs [n][8][4][3][N] (psi(x+mu), then psi(x-mu))
    for oracle.dhop_sites; psi_dev is the canonical full field, or (cb) the field of the other parity."""
    n = lex.size
    links = np.empty((n, 8, 3, 3), dtype=np.complex64)
    nbrs = np.empty((n, 8, 4, 3, psi_dev.shape[-1]), dtype=np.complex64)
    t_lex = torch.from_numpy(lex).cuda()
    links[:, 0:4] = U_dev[t_lex].cpu().numpy()
    for mu in range(4):
        fw = torch.from_numpy(_nbr_lex(dims, lex, mu, +1)).cuda()
        bw = torch.from_numpy(_nbr_lex(dims, lex, mu, -1)).cuda()
        links[:, 4 + mu] = U_dev[bw, mu].cpu().numpy()
        nbrs[:, mu] = psi_dev[(fw >> 1) if cb else fw].cpu().numpy()
        nbrs[:, 4 + mu] = psi_dev[(bw >> 1) if cb else bw].cpu().numpy()
    return links, nbrs


@pytest.fixture(scope="module", params=[12, 1, 24], ids=lambda n: "N%d" % n)
def config5(request):
    nrhs = request.param
    dev = torch.device("cuda", 0)
    U = syn.gauge_torch(DIMS, SEED, dev)
    psi = syn.spinor_torch(syn.volume(DIMS), nrhs, SEED, dev)
    w = mrhs.Wilson(DIMS, nrhs, MASS, CSW, U)
    # the library default is what bench.py times: the sweep kernel from N_rhs = 12, the gather kernel for N_rhs = 1
    want = mrhs.HOP_SWEEP if nrhs >= 12 else mrhs.HOP_GATHER
    assert mrhs.wilson_get_hop_kernel(w.h, 0) == want and mrhs.wilson_get_hop_kernel(w.h, 1) == want
    yield U, psi, w
    w.close()
    del U, psi, w
    torch.cuda.empty_cache()


KERNELS = [mrhs.HOP_SWEEP, mrhs.HOP_GATHER]   # the library default (bench.py's configuration) first


def _set_kernel(w, which, kernel):
    if kernel == mrhs.HOP_SWEEP and w.nrhs % 2:
        pytest.skip("the sweep kernel needs an even N_rhs")
    mrhs.wilson_set_hop_kernel(w.h, which, kernel)


def _parity_of(lex):
    X, Y, Z, T = DIMS
    return (lex % X + (lex // X) % Y + (lex // (X * Y)) % Z + lex // (X * Y * Z)) % 2


def _cb_input(psi, parity):
    """canonical checkerboarded field (index lex >> 1) of the sites of one parity"""
    lex_all = torch.arange(syn.volume(DIMS), device="cuda")
    return psi[_parity_of(lex_all) == parity].contiguous()


def _clover_at(U_host, lex):
    C = np.empty((lex.size, 2, 6, 6), dtype=np.complex128)
    for i, x in enumerate(lex):
        M = oracle.clover_site_matrix(DIMS, U_host, MASS, CSW, int(x))     # 12x12, index 3*spin + colour
        C[i, 0], C[i, 1] = M[0:6, 0:6], M[6:12, 6:12]
    return C


@pytest.mark.parametrize("kernel", KERNELS)
def test_config5_dhop_sampled_sites(config5, kernel):
    U, psi, w = config5
    _set_kernel(w, 0, kernel)
    lex = _sample_sites(DIMS, NSAMPLE, 1)
    d_in = w.import_field(psi, mrhs.FULL)
    d_out = w.empty(mrhs.FULL)
    w.dhop(d_in, d_out)
    torch.cuda.synchronize()
    got = w.export_field(d_out, mrhs.FULL)[torch.from_numpy(lex).cuda()].cpu().numpy()
    del d_in, d_out
    links, nbrs = _gather_hop_inputs(DIMS, U, psi, lex, cb=False)
    want = oracle.dhop_sites(links, nbrs)
    err = rel_l2_per_rhs(got, want)
    assert err.max() < TOL, err


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("out_parity", [0, 1])
def test_config5_meooe_sampled_sites(config5, out_parity, kernel):
    U, psi, w = config5
    _set_kernel(w, 1, kernel)
    psi_in = _cb_input(psi, 1 - out_parity)
    lex = _sample_sites(DIMS, NSAMPLE, 2 + out_parity)
    lex = lex[_parity_of(lex) == out_parity]
    d_in = w.import_field(psi_in, 1 - out_parity)
    d_out = w.empty(out_parity)
    w.meooe(d_in, d_out, out_parity)
    torch.cuda.synchronize()
    got = w.export_field(d_out, out_parity)[torch.from_numpy(lex >> 1).cuda()].cpu().numpy()
    del d_in, d_out
    links, nbrs = _gather_hop_inputs(DIMS, U, psi_in, lex, cb=True)
    want = oracle.dhop_sites(links, nbrs)
    err = rel_l2_per_rhs(got, want)
    assert err.max() < TOL, err


def test_config5_mooee_sampled_sites(config5):
    U, psi, w = config5
    lex = _sample_sites(DIMS, 256, 4)
    d_in = w.import_field(psi, mrhs.FULL)
    d_out = w.empty(mrhs.FULL)
    w.mooee(d_in, d_out, mrhs.FULL)
    torch.cuda.synchronize()
    t_lex = torch.from_numpy(lex).cuda()
    got = w.export_field(d_out, mrhs.FULL)[t_lex].cpu().numpy()
    del d_in, d_out
    C = _clover_at(U.cpu().numpy().astype(np.complex128), lex)
    want = oracle.mooee(C, psi[t_lex].cpu().numpy())
    err = rel_l2_per_rhs(got, want)
    assert err.max() < TOL, err


@pytest.mark.parametrize("kernel", KERNELS)
def test_config5_fused_meooe_mooee_sampled_sites(config5, kernel):
    """The fused M_ooee M_eooe launch (first launch of the Schur-style sequence, the sweep kernel's clover
    epilogue) at full size: out(y) = C(y) H(y) on sampled odd sites, H from the oracle's site-wise hop."""
    U, psi, w = config5
    _set_kernel(w, 1, kernel)
    out_parity = 1
    psi_in = _cb_input(psi, 1 - out_parity)
    lex = _sample_sites(DIMS, 512, 6)
    lex = lex[_parity_of(lex) == out_parity]
    d_in = w.import_field(psi_in, 1 - out_parity)
    d_out = w.empty(out_parity)
    w.meooe_mooee(d_in, d_out, out_parity)
    torch.cuda.synchronize()
    got = w.export_field(d_out, out_parity)[torch.from_numpy(lex >> 1).cuda()].cpu().numpy()
    del d_in, d_out
    links, nbrs = _gather_hop_inputs(DIMS, U, psi_in, lex, cb=True)
    C = _clover_at(U.cpu().numpy().astype(np.complex128), lex)
    want = oracle.mooee(C, oracle.dhop_sites(links, nbrs))
    err = rel_l2_per_rhs(got, want)
    assert err.max() < TOL, err


@pytest.mark.parametrize("kernel", KERNELS)
def test_config5_schur_sequence_sampled_sites(config5, kernel):
    """Row a7 at full size: chi_e = M_eooe M_ooee M_eooe psi_e on sampled even sites.  The oracle evaluates the
    inner two operators on the eight odd neighbours of every sample site (each from its own eight neighbours)."""
    U, psi, w = config5
    _set_kernel(w, 1, kernel)
    psi_e = _cb_input(psi, 0)
    lex = _sample_sites(DIMS, 64, 7)
    lex = lex[_parity_of(lex) == 0][:48]
    d_in = w.import_field(psi_e, mrhs.EVEN)
    t0, t1, d_out = w.empty(mrhs.ODD), w.empty(mrhs.ODD), w.empty(mrhs.EVEN)
    w.schur_sequence(d_in, t0, t1, d_out)
    torch.cuda.synchronize()
    got = w.export_field(d_out, mrhs.EVEN)[torch.from_numpy(lex >> 1).cuda()].cpu().numpy()
    del d_in, t0, t1, d_out
    # the odd neighbours y of the sample sites, psi(x+mu) first, then psi(x-mu): t(y) = C(y) (M_eooe psi_e)(y)
    nb_lex = np.stack([_nbr_lex(DIMS, lex, mu, sgn) for sgn in (+1, -1) for mu in range(4)], axis=1)      # [n][8]
    flat = nb_lex.reshape(-1)
    links_y, nbrs_y = _gather_hop_inputs(DIMS, U, psi_e, flat, cb=True)
    Uh = U.cpu().numpy().astype(np.complex128)
    t_y = oracle.mooee(_clover_at(Uh, flat), oracle.dhop_sites(links_y, nbrs_y))
    links = np.empty((lex.size, 8, 3, 3), dtype=np.complex64)
    t_lex = torch.from_numpy(lex).cuda()
    links[:, 0:4] = U[t_lex].cpu().numpy()
    for mu in range(4):
        links[:, 4 + mu] = U[torch.from_numpy(nb_lex[:, 4 + mu]).cuda(), mu].cpu().numpy()
    want = oracle.dhop_sites(links, t_y.reshape(lex.size, 8, 4, 3, -1))
    err = rel_l2_per_rhs(got, want)
    assert err.max() < TOL, err


@pytest.mark.parametrize("kernel", KERNELS)
def test_config5_full_matrix_sampled_sites(config5, kernel):
    """mrhs_wilson_apply at full size: out = M_ooee in - D_hop in / 2 (reading S6) on sampled sites."""
    U, psi, w = config5
    _set_kernel(w, 0, kernel)
    lex = _sample_sites(DIMS, 512, 8)
    d_in = w.import_field(psi, mrhs.FULL)
    d_out = w.empty(mrhs.FULL)
    w.apply(d_in, d_out)
    torch.cuda.synchronize()
    t_lex = torch.from_numpy(lex).cuda()
    got = w.export_field(d_out, mrhs.FULL)[t_lex].cpu().numpy()
    del d_in, d_out
    links, nbrs = _gather_hop_inputs(DIMS, U, psi, lex, cb=False)
    C = _clover_at(U.cpu().numpy().astype(np.complex128), lex)
    want = oracle.mooee(C, psi[t_lex].cpu().numpy()) - 0.5 * oracle.dhop_sites(links, nbrs)
    err = rel_l2_per_rhs(got, want)
    assert err.max() < TOL, err


def test_config5_sweep_kernels_repeat_bitwise_and_match_gather_on_the_whole_field(config5):
    """Sampled sites cannot see a race that spoils a few tile rows per launch (one did: the sweep kernel's `C aux - H / 4`
    epilogue at 48^4, N_rhs = 12, 0.05 % of the elements, different ones in every call).  Every operator of the sweep path is
    therefore run twice on NaN-filled outputs and must repeat bit for bit, and must agree on the WHOLE field with the gather
    kernels (an independent kernel family, itself checked against the oracle above) to fp32 rounding."""
    U, psi, w = config5
    if w.nrhs % 2:
        pytest.skip("the sweep kernel needs an even N_rhs")
    with_gather = w.nrhs <= 12       # N_rhs = 24: repeatability only (keeps the device memory of the test below 120 GB)
    d_in = w.import_field(psi, mrhs.FULL)
    ie, io = w.empty(mrhs.EVEN), w.empty(mrhs.ODD)
    mrhs.cb_split(DIMS, 12, w.nrhs, d_in, ie, io)
    full, t0, t1 = w.empty(mrhs.FULL), w.empty(mrhs.ODD), w.empty(mrhs.ODD)
    oe, oo = w.empty(mrhs.EVEN), w.empty(mrhs.ODD)
    ops = [
        ("dhop", 0, lambda: w.dhop(d_in, full), full),
        ("dhop_dag", 0, lambda: w.dhop_dag(d_in, full), full),
        ("meooe_dag odd", 1, lambda: w.meooe_dag(ie, oo, mrhs.ODD), oo),
        ("wilson_apply", 0, lambda: w.apply(d_in, full), full),
        ("meooe odd", 1, lambda: w.meooe(ie, oo, mrhs.ODD), oo),
        ("meooe even", 1, lambda: w.meooe(io, oe, mrhs.EVEN), oe),
        ("meooe_mooee odd", 1, lambda: w.meooe_mooee(ie, oo, mrhs.ODD), oo),
        ("meooe_mooee even", 1, lambda: w.meooe_mooee(io, oe, mrhs.EVEN), oe),
        ("meooe_mooee_inv odd", 1, lambda: w.meooe_mooee_inv(ie, oo, mrhs.ODD), oo),
        ("schur_sequence", 1, lambda: w.schur_sequence(ie, t0, t1, oe), oe),
        ("schur_apply", 1, lambda: w.schur_apply(ie, t0, oe), oe),
        ("schur_apply dagger", 1, lambda: w.schur_apply(ie, t0, oe, True), oe),
    ]
    for name, which, run, buf in ops:
        res = []
        for kernel in (mrhs.HOP_SWEEP, mrhs.HOP_SWEEP, mrhs.HOP_SWEEP) + ((mrhs.HOP_GATHER,) if with_gather else ()):
            mrhs.wilson_set_hop_kernel(w.h, which, kernel)
            buf.fill_(float("nan"))
            run()
            torch.cuda.synchronize()
            res.append(buf.clone())
        assert not bool(torch.isnan(res[0]).any()), name
        assert torch.equal(res[0], res[1]) and torch.equal(res[0], res[2]), "%s: the sweep kernel does not repeat bit for bit" % name
        if with_gather:
            scale = float(res[3].abs().max())
            diff = float((res[0] - res[3]).abs().max())
            assert diff < 2e-5 * scale, "%s: sweep and gather kernels differ on the whole field: %g of %g" % (name, diff, scale)
        del res
    mrhs.wilson_set_hop_kernel(w.h, 0, mrhs.HOP_SWEEP)
    mrhs.wilson_set_hop_kernel(w.h, 1, mrhs.HOP_SWEEP)

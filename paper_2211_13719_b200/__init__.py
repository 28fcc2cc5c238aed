"""Python binding of the B200-native MRHS Wilson-clover stencil library (include/mrhs.h).

Argument marshalling only: every operator step runs in the CUDA kernels of ``libmrhs.so``
(built in-tree by ``python -m paper_2211_13719_b200.build``).  PyTorch supplies device memory
and streams.  There is no CPU fallback: loading fails loudly if the library is missing.

The functions carry the names of the C entry points without the ``mrhs_`` prefix
(``wilson_create``, ``dhop``, ``meooe``, ``mooee``, ``coarse_create``, ``coarse_apply``, ...);
``Wilson`` and ``Coarse`` are thin handle owners around them.

Canonical layouts (complex64 torch tensors): spinor [sites][4][3][N], gauge [V][4][3][3],
clover [V][2][6][6], coarse links [V][9][nb][nb], coarse vector [V][nb][N]; the timed applies
work on NATIVE fields (opaque float32 tensors made by ``field_import``).  PAPER.md:25, :43-53, :75.
"""
import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libmrhs.so")
_lib = None

OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_ALLOC, ERR_CUDA = 0, 1, 2, 3, 4
EVEN, ODD, FULL = 0, 1, 2
OP_DHOP, OP_MEOOE, OP_MOOEE, OP_SCHUR = 0, 1, 2, 3
COARSE_FMA, COARSE_TENSOR, COARSE_TENSOR_F16 = 0, 1, 2
HOP_GATHER, HOP_SWEEP = 0, 1
COARSE_SELF, COARSE_HOP, COARSE_ALL = 0x001, 0x1FE, 0x1FF
COARSE_MODES = (COARSE_FMA, COARSE_TENSOR, COARSE_TENSOR_F16)

_vp = ctypes.c_void_p
_int4 = ctypes.c_int * 4
_int3 = ctypes.c_int * 3
_int2 = ctypes.c_int * 2

_SIGNATURES = {
    "mrhs_wilson_create": (ctypes.c_int, [ctypes.POINTER(_vp), _int4, ctypes.c_int, ctypes.c_float, ctypes.c_float, _vp, _vp, _vp]),
    "mrhs_dhop": (ctypes.c_int, [_vp, _vp, _vp]),
    "mrhs_meooe": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int]),
    "mrhs_mooee": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int]),
    "mrhs_schur_sequence": (ctypes.c_int, [_vp, _vp, _vp, _vp, _vp]),
    "mrhs_wilson_apply": (ctypes.c_int, [_vp, _vp, _vp]),
    "mrhs_dhop_dag": (ctypes.c_int, [_vp, _vp, _vp]),
    "mrhs_meooe_dag": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int]),
    "mrhs_wilson_apply_dag": (ctypes.c_int, [_vp, _vp, _vp]),
    "mrhs_schur_apply": (ctypes.c_int, [_vp, _vp, _vp, _vp, ctypes.c_int]),
    "mrhs_meooe_mooee": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int]),
    "mrhs_meooe_mooee_inv": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int]),
    "mrhs_mooee_inv": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int]),
    "mrhs_wilson_export_clover": (ctypes.c_int, [_vp, _vp]),
    "mrhs_wilson_set_tiling": (ctypes.c_int, [_vp, ctypes.c_int, _int3, _int2]),
    "mrhs_wilson_get_tiling": (ctypes.c_int, [_vp, ctypes.c_int, _int3, _int2]),
    "mrhs_wilson_set_prefetch": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int]),
    "mrhs_wilson_set_hop_kernel": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int]),
    "mrhs_wilson_get_hop_kernel": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.POINTER(ctypes.c_int)]),
    "mrhs_wilson_set_sweep": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, _int2]),
    "mrhs_wilson_get_sweep": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.POINTER(ctypes.c_int), _int2]),
    "mrhs_wilson_destroy": (ctypes.c_int, [_vp]),
    "mrhs_sweep_plan": (ctypes.c_int, [_int4, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int * 9]),
    "mrhs_sweep_blocks": (ctypes.c_int, [_int4, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_int)]),
    "mrhs_coarse_create": (ctypes.c_int, [ctypes.POINTER(_vp), _int4, ctypes.c_int, ctypes.c_int, _vp, ctypes.c_int, _vp]),
    "mrhs_coarse_apply": (ctypes.c_int, [_vp, _vp, _vp]),
    "mrhs_coarse_apply_points": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int]),
    "mrhs_coarse_meooe": (ctypes.c_int, [_vp, _vp, _vp, ctypes.c_int]),
    "mrhs_coarse_destroy": (ctypes.c_int, [_vp]),
    "mrhs_transfer_create": (ctypes.c_int, [ctypes.POINTER(_vp), _int4, _int4, ctypes.c_int, ctypes.c_int, _vp, _vp]),
    "mrhs_transfer_create_coarse": (ctypes.c_int, [ctypes.POINTER(_vp), _int4, _int4, ctypes.c_int, ctypes.c_int, ctypes.c_int, _vp, _vp]),
    "mrhs_prolong": (ctypes.c_int, [_vp, _vp, _vp]),
    "mrhs_restrict": (ctypes.c_int, [_vp, _vp, _vp]),
    "mrhs_transfer_destroy": (ctypes.c_int, [_vp]),
    "mrhs_inner_products": (ctypes.c_int, [_int4, ctypes.c_int, ctypes.c_int, ctypes.c_int, _vp, _vp, _vp, _vp]),
    "mrhs_inner_products_noalloc": (ctypes.c_int, [_int4, ctypes.c_int, ctypes.c_int, ctypes.c_int, _vp, _vp, _vp, _vp]),
    "mrhs_xblock": (ctypes.c_int, [ctypes.c_int, ctypes.c_int]),
    "mrhs_field_bytes": (ctypes.c_size_t, [_int4, ctypes.c_int, ctypes.c_int, ctypes.c_int]),
    "mrhs_field_import": (ctypes.c_int, [_int4, ctypes.c_int, ctypes.c_int, ctypes.c_int, _vp, _vp, _vp]),
    "mrhs_field_export": (ctypes.c_int, [_int4, ctypes.c_int, ctypes.c_int, ctypes.c_int, _vp, _vp, _vp]),
    "mrhs_cb_split": (ctypes.c_int, [_int4, ctypes.c_int, ctypes.c_int, _vp, _vp, _vp, _vp]),
    "mrhs_cb_merge": (ctypes.c_int, [_int4, ctypes.c_int, ctypes.c_int, _vp, _vp, _vp, _vp]),
    "mrhs_coarse_field_import": (ctypes.c_int, [_int4, ctypes.c_int, ctypes.c_int, ctypes.c_int, _vp, _vp, _vp]),
    "mrhs_coarse_field_export": (ctypes.c_int, [_int4, ctypes.c_int, ctypes.c_int, ctypes.c_int, _vp, _vp, _vp]),
    "mrhs_coarse_cb_split": (ctypes.c_int, [_int4, ctypes.c_int, ctypes.c_int, _vp, _vp, _vp, _vp]),
    "mrhs_coarse_cb_merge": (ctypes.c_int, [_int4, ctypes.c_int, ctypes.c_int, _vp, _vp, _vp, _vp]),
    "mrhs_wilson_apply_host": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, _vp, _vp]),
    "mrhs_coarse_apply_host": (ctypes.c_int, [_vp, _vp, _vp]),
    "mrhs_wilson_apply_host_async": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_int, _vp, _vp]),
    "mrhs_wilson_host_wait": (ctypes.c_int, [_vp]),
    "mrhs_coarse_apply_host_async": (ctypes.c_int, [_vp, _vp, _vp]),
    "mrhs_coarse_host_wait": (ctypes.c_int, [_vp]),
    "mrhs_last_error": (ctypes.c_char_p, []),
    "mrhs_version": (ctypes.c_char_p, []),
}
EXPORTED_SYMBOLS = tuple(_SIGNATURES)


class MrhsError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("mrhs status %d: %s" % (status, message))
        self.status = status


def lib():
    """The loaded C-ABI library.  Raises if it has not been built (no fallback exists)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError("libmrhs.so is missing: run `python -m paper_2211_13719_b200.build` "
                              "(nvcc, sm_100a); there is no CPU fallback")
        l = ctypes.CDLL(_LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            f = getattr(l, name)
            f.restype = res
            f.argtypes = args
        _lib = l
    return _lib


def last_error():
    return lib().mrhs_last_error().decode()


def version():
    return lib().mrhs_version().decode()


def _check(status):
    if status != OK:
        raise MrhsError(status, last_error())


def _ptr(t):
    if t is None:
        return None
    return _vp(t.data_ptr())


def _stream_ptr(stream):
    if stream is None:
        return None
    return _vp(stream.cuda_stream)


def _dims(dims):
    return _int4(*[int(d) for d in dims])


# ------------------------------------------------------------------ layout helpers

def xblock(x_eff, nrhs):
    return lib().mrhs_xblock(int(x_eff), int(nrhs))


def field_bytes(dims, ncomp, nrhs, checkerboarded):
    return lib().mrhs_field_bytes(_dims(dims), int(ncomp), int(nrhs), int(bool(checkerboarded)))


def empty_field(dims, ncomp, nrhs, parity, device="cuda"):
    """Uninitialised native field (float32 tensor of field_bytes/4 elements)."""
    import torch
    nbytes = field_bytes(dims, ncomp, nrhs, parity != FULL)
    if nbytes == 0:
        raise MrhsError(ERR_INVALID_ARG, "invalid field shape")
    return torch.empty(nbytes // 4, dtype=torch.float32, device=device)


def field_import(dims, ncomp, nrhs, parity, canonical, native=None, stream=None):
    """canonical complex64 tensor -> native field (allocated if not given)."""
    if native is None:
        native = empty_field(dims, ncomp, nrhs, parity, canonical.device)
    _check(lib().mrhs_field_import(_dims(dims), ncomp, nrhs, parity, _ptr(canonical), _ptr(native), _stream_ptr(stream)))
    return native


class Transfer:
    """MRHS prolongation / restriction (handle owner): between the fine level and its first coarse level, or, with
    nf = the finer level's nbasis, between two coarse levels (fields of both levels in the coarse layout)."""

    def __init__(self, dims, bdims, nvec, nrhs, basis, stream=None, nf=None):
        self.dims, self.bdims, self.nvec, self.nrhs = [int(d) for d in dims], [int(b) for b in bdims], int(nvec), int(nrhs)
        self.cdims = [d // b for d, b in zip(self.dims, self.bdims)]
        self.nf = nf
        h = _vp()
        if nf is None:
            _check(lib().mrhs_transfer_create(ctypes.byref(h), _dims(self.dims), _dims(self.bdims), self.nvec, self.nrhs,
                                              _ptr(basis), _stream_ptr(stream)))
        else:
            _check(lib().mrhs_transfer_create_coarse(ctypes.byref(h), _dims(self.dims), _dims(self.bdims), int(nf), self.nvec,
                                                     self.nrhs, _ptr(basis), _stream_ptr(stream)))
        self.h = h

    def prolong(self, d_coarse, d_fine):
        _check(lib().mrhs_prolong(self.h, _ptr(d_coarse), _ptr(d_fine)))

    def restrict(self, d_fine, d_coarse):
        _check(lib().mrhs_restrict(self.h, _ptr(d_fine), _ptr(d_coarse)))

    def close(self):
        if self.h:
            _check(lib().mrhs_transfer_destroy(self.h))
            self.h = None


def inner_products(dims, ncomp, nrhs, parity, x, y, result=None, stream=None):
    """result[r] = <x_r, y_r> for two native fields of the same geometry; complex128 device tensor [nrhs]."""
    import torch
    if result is None:
        result = torch.empty(nrhs, dtype=torch.complex128, device=x.device)
    _check(lib().mrhs_inner_products(_dims(dims), ncomp, nrhs, parity, _ptr(x), _ptr(y), _ptr(result), _stream_ptr(stream)))
    return result


def inner_products_noalloc(dims, ncomp, nrhs, parity, x, y, result, stream=None):
    """inner_products through the entry that allocates nothing (static device scratch, (8 x SMs) x nrhs <= 131072);
    result: caller-provided complex128 device tensor [nrhs].  Calls that overlap on the GPU race on the shared scratch."""
    _check(lib().mrhs_inner_products_noalloc(_dims(dims), ncomp, nrhs, parity, _ptr(x), _ptr(y), _ptr(result), _stream_ptr(stream)))
    return result


def field_export(dims, ncomp, nrhs, parity, native, canonical=None, stream=None):
    """native field -> canonical complex64 tensor [sites][ncomp][nrhs] (allocated if not given)."""
    import torch
    if canonical is None:
        nsites = int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])
        if parity != FULL:
            nsites //= 2
        canonical = torch.empty((nsites, ncomp, nrhs), dtype=torch.complex64, device=native.device)
    _check(lib().mrhs_field_export(_dims(dims), ncomp, nrhs, parity, _ptr(native), _ptr(canonical), _stream_ptr(stream)))
    return canonical


def coarse_field_import(cdims, nbasis, nrhs, parity, canonical, native=None, stream=None):
    """canonical coarse vector [sites][nbasis][nrhs] -> native (coarse layout whatever nbasis is; parity 0/1 = one parity)."""
    if native is None:
        native = empty_field(cdims, nbasis, nrhs, parity, canonical.device)
    _check(lib().mrhs_coarse_field_import(_dims(cdims), nbasis, nrhs, parity, _ptr(canonical), _ptr(native), _stream_ptr(stream)))
    return native


def coarse_field_export(cdims, nbasis, nrhs, parity, native, canonical=None, stream=None):
    import torch
    if canonical is None:
        nsites = int(cdims[0]) * int(cdims[1]) * int(cdims[2]) * int(cdims[3]) // (1 if parity == FULL else 2)
        canonical = torch.empty((nsites, nbasis, nrhs), dtype=torch.complex64, device=native.device)
    _check(lib().mrhs_coarse_field_export(_dims(cdims), nbasis, nrhs, parity, _ptr(native), _ptr(canonical), _stream_ptr(stream)))
    return canonical


def coarse_cb_split(cdims, nbasis, nrhs, full, even, odd, stream=None):
    _check(lib().mrhs_coarse_cb_split(_dims(cdims), nbasis, nrhs, _ptr(full), _ptr(even), _ptr(odd), _stream_ptr(stream)))


def coarse_cb_merge(cdims, nbasis, nrhs, even, odd, full, stream=None):
    _check(lib().mrhs_coarse_cb_merge(_dims(cdims), nbasis, nrhs, _ptr(even), _ptr(odd), _ptr(full), _stream_ptr(stream)))


def cb_split(dims, ncomp, nrhs, full, even, odd, stream=None):
    _check(lib().mrhs_cb_split(_dims(dims), ncomp, nrhs, _ptr(full), _ptr(even), _ptr(odd), _stream_ptr(stream)))


def cb_merge(dims, ncomp, nrhs, even, odd, full, stream=None):
    _check(lib().mrhs_cb_merge(_dims(dims), ncomp, nrhs, _ptr(even), _ptr(odd), _ptr(full), _stream_ptr(stream)))


# ------------------------------------------------------------------ fine level

def wilson_create(dims, nrhs, mass, csw, gauge, clover=None, stream=None):
    h = _vp()
    _check(lib().mrhs_wilson_create(ctypes.byref(h), _dims(dims), int(nrhs), float(mass), float(csw),
                                    _ptr(gauge), _ptr(clover), _stream_ptr(stream)))
    return h


def dhop(h, d_in, d_out):
    _check(lib().mrhs_dhop(h, _ptr(d_in), _ptr(d_out)))


def meooe(h, d_in, d_out, out_parity):
    _check(lib().mrhs_meooe(h, _ptr(d_in), _ptr(d_out), int(out_parity)))


def mooee(h, d_in, d_out, parity):
    _check(lib().mrhs_mooee(h, _ptr(d_in), _ptr(d_out), int(parity)))


def wilson_apply(h, d_in, d_out):
    _check(lib().mrhs_wilson_apply(h, _ptr(d_in), _ptr(d_out)))


def dhop_dag(h, d_in, d_out):
    _check(lib().mrhs_dhop_dag(h, _ptr(d_in), _ptr(d_out)))


def meooe_dag(h, d_in, d_out, out_parity):
    _check(lib().mrhs_meooe_dag(h, _ptr(d_in), _ptr(d_out), int(out_parity)))


def wilson_apply_dag(h, d_in, d_out):
    _check(lib().mrhs_wilson_apply_dag(h, _ptr(d_in), _ptr(d_out)))


def schur_apply(h, d_in, d_tmp, d_out, dagger=False):
    _check(lib().mrhs_schur_apply(h, _ptr(d_in), _ptr(d_tmp), _ptr(d_out), int(bool(dagger))))


def meooe_mooee(h, d_in, d_out, out_parity):
    _check(lib().mrhs_meooe_mooee(h, _ptr(d_in), _ptr(d_out), int(out_parity)))


def meooe_mooee_inv(h, d_in, d_out, out_parity):
    _check(lib().mrhs_meooe_mooee_inv(h, _ptr(d_in), _ptr(d_out), int(out_parity)))


def mooee_inv(h, d_in, d_out, parity):
    _check(lib().mrhs_mooee_inv(h, _ptr(d_in), _ptr(d_out), int(parity)))


def schur_sequence(h, d_in, d_tmp0, d_tmp1, d_out):
    _check(lib().mrhs_schur_sequence(h, _ptr(d_in), _ptr(d_tmp0), _ptr(d_tmp1), _ptr(d_out)))


def wilson_export_clover(h, clover_out):
    _check(lib().mrhs_wilson_export_clover(h, _ptr(clover_out)))


def wilson_set_tiling(h, which, tile, chunk):
    _check(lib().mrhs_wilson_set_tiling(h, int(which), _int3(*[int(v) for v in tile]), _int2(*[int(v) for v in chunk])))


def wilson_get_tiling(h, which):
    tile, chunk = _int3(), _int2()
    _check(lib().mrhs_wilson_get_tiling(h, int(which), tile, chunk))
    return list(tile), list(chunk)


def wilson_set_prefetch(h, which, distance_tiles):
    _check(lib().mrhs_wilson_set_prefetch(h, int(which), int(distance_tiles)))


def wilson_set_hop_kernel(h, which, kernel):
    _check(lib().mrhs_wilson_set_hop_kernel(h, int(which), int(kernel)))


def wilson_get_hop_kernel(h, which):
    k = ctypes.c_int()
    _check(lib().mrhs_wilson_get_hop_kernel(h, int(which), ctypes.byref(k)))
    return k.value


def wilson_set_sweep(h, which, lt, chunk):
    _check(lib().mrhs_wilson_set_sweep(h, int(which), int(lt), _int2(*[int(v) for v in chunk])))


def wilson_get_sweep(h, which):
    lt, chunk = ctypes.c_int(), _int2()
    _check(lib().mrhs_wilson_get_sweep(h, int(which), ctypes.byref(lt), chunk))
    return lt.value, list(chunk)


def wilson_apply_host(h, op, parity, h_in, h_out):
    """h_in / h_out: HOST tensors (canonical complex64, ideally pinned)."""
    _check(lib().mrhs_wilson_apply_host(h, int(op), int(parity), _ptr(h_in), _ptr(h_out)))


def wilson_apply_host_async(h, op, parity, h_in, h_out):
    """Enqueue only; h_in / h_out (pinned HOST tensors) must stay alive until wilson_host_wait(h)."""
    _check(lib().mrhs_wilson_apply_host_async(h, int(op), int(parity), _ptr(h_in), _ptr(h_out)))


def wilson_host_wait(h):
    _check(lib().mrhs_wilson_host_wait(h))


def sweep_plan(dims, nrhs, parity, num_sms):
    """Host-only: (blocks, threads, tiles, whole-line blocks, tail tiles, segments per tail tile, lt, cy, cz) of the sweep kernel."""
    plan = (ctypes.c_int * 9)()
    _check(lib().mrhs_sweep_plan(_dims(dims), int(nrhs), int(parity), int(num_sms), plan))
    return list(plan)


def sweep_blocks(dims, nrhs, parity, num_sms, first, count):
    """Host-only: [(x-block, first y, first z, first t, slices)] of the tile segments blocks first .. first + count - 1 sweep."""
    c = (ctypes.c_int * (5 * int(count)))()
    _check(lib().mrhs_sweep_blocks(_dims(dims), int(nrhs), int(parity), int(num_sms), int(first), int(count), c))
    return [tuple(c[5 * i:5 * i + 5]) for i in range(int(count))]


def wilson_destroy(h):
    _check(lib().mrhs_wilson_destroy(h))


# ------------------------------------------------------------------ coarse level

def coarse_create(cdims, nbasis, nrhs, links, math_mode=0, stream=None):
    h = _vp()
    _check(lib().mrhs_coarse_create(ctypes.byref(h), _dims(cdims), int(nbasis), int(nrhs), _ptr(links),
                                    int(math_mode), _stream_ptr(stream)))
    return h


def coarse_apply(h, d_in, d_out):
    _check(lib().mrhs_coarse_apply(h, _ptr(d_in), _ptr(d_out)))


def coarse_apply_points(h, d_in, d_out, point_mask):
    _check(lib().mrhs_coarse_apply_points(h, _ptr(d_in), _ptr(d_out), int(point_mask)))


def coarse_meooe(h, d_in, d_out, out_parity):
    _check(lib().mrhs_coarse_meooe(h, _ptr(d_in), _ptr(d_out), int(out_parity)))


def coarse_apply_host(h, h_in, h_out):
    _check(lib().mrhs_coarse_apply_host(h, _ptr(h_in), _ptr(h_out)))


def coarse_apply_host_async(h, h_in, h_out):
    _check(lib().mrhs_coarse_apply_host_async(h, _ptr(h_in), _ptr(h_out)))


def coarse_host_wait(h):
    _check(lib().mrhs_coarse_host_wait(h))


def coarse_destroy(h):
    _check(lib().mrhs_coarse_destroy(h))


# ------------------------------------------------------------------ handle owners

class Wilson:
    """Owns a fine-level handle (packed gauge + clover on the device)."""

    def __init__(self, dims, nrhs, mass, csw, gauge, clover=None, stream=None):
        self.dims = [int(d) for d in dims]
        self.nrhs = int(nrhs)
        self.h = wilson_create(dims, nrhs, mass, csw, gauge, clover, stream)

    def close(self):
        if self.h is not None:
            wilson_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def empty(self, parity, device="cuda"):
        return empty_field(self.dims, 12, self.nrhs, parity, device)

    def import_field(self, canonical, parity):
        return field_import(self.dims, 12, self.nrhs, parity, canonical)

    def export_field(self, native, parity):
        out = field_export(self.dims, 12, self.nrhs, parity, native)
        return out.reshape(out.shape[0], 4, 3, self.nrhs)

    def dhop(self, d_in, d_out):
        dhop(self.h, d_in, d_out)

    def meooe(self, d_in, d_out, out_parity):
        meooe(self.h, d_in, d_out, out_parity)

    def mooee(self, d_in, d_out, parity):
        mooee(self.h, d_in, d_out, parity)

    def apply(self, d_in, d_out, dagger=False):
        """out = M in (or M^+ in), the full Wilson-clover matrix on full-lattice fields."""
        (wilson_apply_dag if dagger else wilson_apply)(self.h, d_in, d_out)

    def dhop_dag(self, d_in, d_out):
        dhop_dag(self.h, d_in, d_out)

    def meooe_dag(self, d_in, d_out, out_parity):
        meooe_dag(self.h, d_in, d_out, out_parity)

    def schur_apply(self, d_in, d_tmp, d_out, dagger=False):
        """out = S in on even fields, S = C_e - H_eo C_o^-1 H_oe / 4 (d_tmp: odd scratch)."""
        schur_apply(self.h, d_in, d_tmp, d_out, dagger)

    def meooe_mooee(self, d_in, d_out, out_parity):
        meooe_mooee(self.h, d_in, d_out, out_parity)

    def meooe_mooee_inv(self, d_in, d_out, out_parity):
        meooe_mooee_inv(self.h, d_in, d_out, out_parity)

    def mooee_inv(self, d_in, d_out, parity):
        mooee_inv(self.h, d_in, d_out, parity)

    def schur_sequence(self, d_in, d_tmp0, d_tmp1, d_out):
        schur_sequence(self.h, d_in, d_tmp0, d_tmp1, d_out)


class Coarse:
    """Owns a coarse-level handle (packed link matrices on the device)."""

    def __init__(self, cdims, nbasis, nrhs, links, math_mode=0, stream=None):
        self.cdims = [int(d) for d in cdims]
        self.nbasis = int(nbasis)
        self.nrhs = int(nrhs)
        self.h = coarse_create(cdims, nbasis, nrhs, links, math_mode, stream)

    def close(self):
        if self.h is not None:
            coarse_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def empty(self, device="cuda", parity=FULL):
        return empty_field(self.cdims, self.nbasis, self.nrhs, parity, device)

    def import_field(self, canonical, parity=FULL):
        return coarse_field_import(self.cdims, self.nbasis, self.nrhs, parity, canonical)

    def export_field(self, native, parity=FULL):
        return coarse_field_export(self.cdims, self.nbasis, self.nrhs, parity, native)

    def meooe(self, d_in, d_out, out_parity):
        """out = coarse M_eooe in: the 8-point hopping term on the sites of out_parity from the other parity."""
        coarse_meooe(self.h, d_in, d_out, out_parity)

    def apply(self, d_in, d_out, point_mask=None):
        if point_mask is None:
            coarse_apply(self.h, d_in, d_out)
        else:
            coarse_apply_points(self.h, d_in, d_out, point_mask)

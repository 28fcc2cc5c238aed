"""fp64 CPU oracle for the MRHS Wilson-clover stencils -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin numpy/ctypes front end of ``mrhs_oracle.c`` (the arithmetic lives there, in plain C,
see its header for the definitions and the paper passages they restate).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs
may import this package.  It imports nothing from ``paper_2211_13719_b200`` and shares no
code with the CUDA path.

All arrays are complex128 in the canonical layouts of SURVEY.md Sec. 8(b):
  spinor [V][4][3][N], gauge [V][4][3][3], clover [V][2][6][6],
  coarse links [V][9][nb][nb], coarse vector [V][nb][N]; site lex = x + X(y + Y(z + Z t)).

Versus the paper's own code (absent from this container): parity unpinned.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mrhs_oracle.c")
_LIB = os.path.join(_HERE, "libmrhs_oracle.so")
_lib = None

_c_int4 = ctypes.c_int * 4
_dp = ctypes.c_void_p


def build(force=False):
    """Compile mrhs_oracle.c with gcc (OpenMP over sites).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fcx-limited-range", "-fPIC", "-shared",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.orc_neighbour.restype = ctypes.c_long
        _lib.orc_neighbour.argtypes = [_c_int4, ctypes.c_long, ctypes.c_int, ctypes.c_int]
        _lib.orc_parity.restype = ctypes.c_int
        _lib.orc_parity.argtypes = [_c_int4, ctypes.c_long]
        _lib.orc_get_threads.restype = ctypes.c_int
    return _lib


def _c128(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a


def _ptr(a):
    return ctypes.c_void_p(a.ctypes.data)


def _dims(dims):
    dims = [int(d) for d in dims]
    assert len(dims) == 4 and all(d >= 2 and d % 2 == 0 for d in dims), "extents must be even and >= 2"
    return _c_int4(*dims)


def _cdims(dims):
    """Coarse lattices need not have even extents (nothing is checkerboarded there)."""
    dims = [int(d) for d in dims]
    assert len(dims) == 4 and all(d >= 2 for d in dims), "extents must be >= 2"
    return _c_int4(*dims)


def volume(dims):
    return int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


def set_threads(n):
    _load().orc_set_threads(ctypes.c_int(int(n)))


def get_threads():
    return int(_load().orc_get_threads())


def gamma(mu):
    """4x4 gamma matrix, mu = 0..3 (x,y,z,t), 4 = gamma_5 (S2)."""
    g = np.zeros((4, 4), dtype=np.complex128)
    _load().orc_gamma(ctypes.c_int(mu), _ptr(g))
    return g


def sigma(mu, nu):
    """sigma_munu = (i/2)[gamma_mu, gamma_nu] (S6)."""
    s = np.zeros((4, 4), dtype=np.complex128)
    _load().orc_sigma(ctypes.c_int(mu), ctypes.c_int(nu), _ptr(s))
    return s


def neighbour(dims, lex, mu, sign):
    return int(_load().orc_neighbour(_dims(dims), ctypes.c_long(int(lex)), ctypes.c_int(mu), ctypes.c_int(sign)))


def parity(dims, lex):
    return int(_load().orc_parity(_dims(dims), ctypes.c_long(int(lex))))


def dhop(dims, U, psi, dirmask=0xFF):
    """D_hop on the full lattice (S3).  psi [V][4][3][N] -> same shape."""
    V = volume(dims)
    U = _c128(U); psi = _c128(psi)
    assert U.shape == (V, 4, 3, 3) and psi.shape[:3] == (V, 4, 3)
    N = psi.shape[3]
    out = np.empty_like(psi)
    _load().orc_dhop(_dims(dims), ctypes.c_int(N), _ptr(U), _ptr(psi), _ptr(out), ctypes.c_int(dirmask))
    return out


def meooe(dims, U, psi_cb, out_parity):
    """M_eooe (S4).  psi_cb [V/2][4][3][N] of parity 1-out_parity -> parity out_parity."""
    V = volume(dims)
    U = _c128(U); psi_cb = _c128(psi_cb)
    assert U.shape == (V, 4, 3, 3) and psi_cb.shape[:3] == (V // 2, 4, 3)
    assert out_parity in (0, 1)
    N = psi_cb.shape[3]
    out = np.empty_like(psi_cb)
    _load().orc_meooe(_dims(dims), ctypes.c_int(N), _ptr(U), _ptr(psi_cb), _ptr(out), ctypes.c_int(out_parity))
    return out


def dhop_sites(links, nbrs, dirmask=0xFF):
    """D_hop at isolated sites: links [n][8][3][3] (U_mu(x), then U_mu(x-mu)),
    nbrs [n][8][4][3][N] (psi(x+mu), then psi(x-mu)) -> [n][4][3][N]."""
    links = _c128(links); nbrs = _c128(nbrs)
    n = links.shape[0]
    assert links.shape == (n, 8, 3, 3) and nbrs.shape[:4] == (n, 8, 4, 3)
    N = nbrs.shape[4]
    out = np.empty((n, 4, 3, N), dtype=np.complex128)
    _load().orc_dhop_sites(ctypes.c_long(n), ctypes.c_int(N), _ptr(links), _ptr(nbrs), ctypes.c_int(dirmask), _ptr(out))
    return out


def field_strength(dims, U, lex, mu, nu):
    """F_munu(x), Hermitian 3x3 (S5)."""
    U = _c128(U)
    F = np.zeros((3, 3), dtype=np.complex128)
    _load().orc_field_strength(_dims(dims), _ptr(U), ctypes.c_long(int(lex)), ctypes.c_int(mu), ctypes.c_int(nu), _ptr(F))
    return F


def clover_site_matrix(dims, U, mass, csw, lex):
    """Full 12x12 M_ooee(x), index 3*spin + colour (S6)."""
    U = _c128(U)
    M = np.zeros((12, 12), dtype=np.complex128)
    _load().orc_clover_site_matrix(_dims(dims), _ptr(U), ctypes.c_double(mass), ctypes.c_double(csw),
                                   ctypes.c_long(int(lex)), _ptr(M))
    return M


def clover_blocks(dims, U, mass, csw):
    """Clover blocks C [V][2][6][6] (S7) and the largest |entry| outside the two blocks."""
    V = volume(dims)
    U = _c128(U)
    assert U.shape == (V, 4, 3, 3)
    C = np.zeros((V, 2, 6, 6), dtype=np.complex128)
    off = ctypes.c_double(0.0)
    _load().orc_clover_blocks(_dims(dims), _ptr(U), ctypes.c_double(mass), ctypes.c_double(csw), _ptr(C), ctypes.byref(off))
    return C, off.value


def inner_products(x, y):
    """Simultaneous inner products: result[r] = sum conj(x[..., r]) y[..., r]
    over every index but the last (the RHS index), in fp64.  x, y: canonical fields [...][N]."""
    x = _c128(x); y = _c128(y)
    assert x.shape == y.shape
    N = x.shape[-1]
    out = np.zeros(N, dtype=np.complex128)
    for r in range(N):
        out[r] = np.sum(np.conj(x[..., r]) * y[..., r])
    return out


def clover_inverse(C):
    """Inverse clover blocks: the matrix inverse of every 6x6 block,
    by the library routine (numpy.linalg.inv, fp64).  C [n][2][6][6] -> same shape."""
    return np.linalg.inv(_c128(C))


def mooee(C, psi):
    """M_ooee apply.  C [n][2][6][6], psi [n][4][3][N] -> same shape."""
    C = _c128(C); psi = _c128(psi)
    n = C.shape[0]
    assert C.shape == (n, 2, 6, 6) and psi.shape[:3] == (n, 4, 3)
    N = psi.shape[3]
    out = np.empty_like(psi)
    _load().orc_mooee(ctypes.c_long(n), ctypes.c_int(N), _ptr(C), _ptr(psi), _ptr(out))
    return out


def coarse_apply(cdims, A, v, pmask=0x1FF):
    """9-point coarse apply (S8).  A [V][9][nb][nb], v [V][nb][N] -> [V][nb][N]."""
    V = volume(cdims)
    A = _c128(A); v = _c128(v)
    nb = A.shape[2]
    assert A.shape == (V, 9, nb, nb) and v.shape[:2] == (V, nb)
    N = v.shape[2]
    out = np.empty_like(v)
    _load().orc_coarse_apply(_cdims(cdims), ctypes.c_int(nb), ctypes.c_int(N), _ptr(A), _ptr(v), _ptr(out), ctypes.c_int(pmask))
    return out


def coarse_meooe(cdims, A, v_cb, out_parity):
    """Coarse M_eooe: the 8-point hopping term at the coarse sites of parity
    out_parity from the sites of the other parity.  A [V][9][nb][nb] (full lattice), v_cb [V/2][nb][N] -> [V/2][nb][N]."""
    V = volume(cdims)
    assert all(int(d) % 2 == 0 for d in cdims), "checkerboarded coarse fields need even extents"
    A = _c128(A); v_cb = _c128(v_cb)
    nb = A.shape[2]
    assert A.shape == (V, 9, nb, nb) and v_cb.shape[:2] == (V // 2, nb)
    N = v_cb.shape[2]
    out = np.empty_like(v_cb)
    _load().orc_coarse_meooe(_cdims(cdims), ctypes.c_int(nb), ctypes.c_int(N), _ptr(A), _ptr(v_cb), _ptr(out), ctypes.c_int(out_parity))
    return out


def coarse_sites(A, nbrs):
    """Coarse apply at isolated sites: A [n][9][nb][nb], nbrs [n][9][nb][N] -> [n][nb][N]."""
    A = _c128(A); nbrs = _c128(nbrs)
    n, _, nb, _ = A.shape
    assert A.shape == (n, 9, nb, nb) and nbrs.shape[:3] == (n, 9, nb)
    N = nbrs.shape[3]
    out = np.empty((n, nb, N), dtype=np.complex128)
    _load().orc_coarse_sites(ctypes.c_long(n), ctypes.c_int(nb), ctypes.c_int(N), _ptr(A), _ptr(nbrs), _ptr(out))
    return out


# ---- checkerboard helpers of the canonical layout (pure indexing) ----

def parity_mask(dims):
    """parity[lex] = (x+y+z+t) % 2 for the canonical site order."""
    X, Y, Z, T = [int(d) for d in dims]
    x = np.arange(X).reshape(1, 1, 1, X)
    y = np.arange(Y).reshape(1, 1, Y, 1)
    z = np.arange(Z).reshape(1, Z, 1, 1)
    t = np.arange(T).reshape(T, 1, 1, 1)
    return ((x + y + z + t) % 2).reshape(-1)


def cb_split(dims, full):
    """full [V]... -> (even [V/2]..., odd [V/2]...), each ordered by increasing lex (index lex>>1)."""
    p = parity_mask(dims)
    return np.ascontiguousarray(full[p == 0]), np.ascontiguousarray(full[p == 1])


def cb_merge(dims, even, odd):
    p = parity_mask(dims)
    full = np.empty((p.size,) + even.shape[1:], dtype=even.dtype)
    full[p == 0] = even
    full[p == 1] = odd
    return full

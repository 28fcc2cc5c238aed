"""Small test-side helpers: plain numpy indexing and error metrics (no operator arithmetic)."""
import numpy as np


def read_golden_gammas(path):
    mats, rows = [], []
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        rows.append([complex(float(a), float(b)) for a, b in (e.split(",") for e in line.split())])
        if len(rows) == 4:
            mats.append(np.array(rows, dtype=np.complex128))
            rows = []
    assert len(mats) == 5
    return mats


def coords(dims):
    """x,y,z,t arrays [V] for the canonical site order lex = x + X(y + Y(z + Z t))."""
    X, Y, Z, T = [int(d) for d in dims]
    lex = np.arange(X * Y * Z * T)
    return np.stack([lex % X, (lex // X) % Y, (lex // (X * Y)) % Z, lex // (X * Y * Z)], axis=0)


def shift_index(dims, mu, sign):
    """lex of x + sign*mu for every site (periodic)."""
    c = coords(dims).copy()
    c[mu] = (c[mu] + sign) % dims[mu]
    X, Y, Z, T = [int(d) for d in dims]
    return c[0] + X * (c[1] + Y * (c[2] + Z * c[3]))


def rel_l2_per_rhs(got, want):
    """Reading S16: per RHS r, ||got[..., r] - want[..., r]||_2 / ||want[..., r]||_2, norms in fp64."""
    got = np.asarray(got, dtype=np.complex128)
    want = np.asarray(want, dtype=np.complex128)
    N = want.shape[-1]
    d = (got - want).reshape(-1, N)
    w = want.reshape(-1, N)
    return np.sqrt(np.sum(np.abs(d) ** 2, axis=0)) / np.sqrt(np.sum(np.abs(w) ** 2, axis=0))

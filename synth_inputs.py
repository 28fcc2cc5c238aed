"""Seeded synthetic inputs shaped like the paper's workloads (single precision,
random "hot" gauge fields, random sources).  Serves both the oracle tests and the CUDA path;
holds none of the method's arithmetic -- only random draws, a Gram-Schmidt to land on SU(3)
and one rounding to fp32 (readings S16 and S18).

Everything is returned as complex64 in the canonical layouts of SURVEY.md Sec. 8(b).  The
oracle promotes these fp32 values to fp64, so input rounding is not part of any error.

numpy generators (``*_np``) are used up to 24^4; the torch generators (``*_torch``) draw on a
given device with a seeded ``torch.Generator`` for the 48^4 workloads.
"""
import numpy as np


def volume(dims):
    return int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


# ---------------------------------------------------------------- numpy (host)

def _cgauss_np(rng, shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def su3_np(rng, n):
    """n Haar-random SU(3) matrices, complex128 [n][3][3] (S18): row a uniform on the unit
    sphere of C^3, row b Gaussian made orthogonal to a and normalised, row c = conj(a x b)."""
    a = _cgauss_np(rng, (n, 3))
    a /= np.linalg.norm(a, axis=1, keepdims=True)
    b = _cgauss_np(rng, (n, 3))
    b -= a * np.sum(np.conj(a) * b, axis=1, keepdims=True)
    b /= np.linalg.norm(b, axis=1, keepdims=True)
    c = np.conj(np.cross(a, b))
    return np.stack([a, b, c], axis=1)


def gauge_np(dims, seed):
    """Hot gauge field U[V][4][3][3], complex64."""
    rng = np.random.default_rng([seed, 0x6A])
    V = volume(dims)
    return su3_np(rng, V * 4).reshape(V, 4, 3, 3).astype(np.complex64)


def unit_gauge_np(dims):
    V = volume(dims)
    U = np.zeros((V, 4, 3, 3), dtype=np.complex64)
    U[:, :, 0, 0] = U[:, :, 1, 1] = U[:, :, 2, 2] = 1
    return U


def spinor_np(nsites, nrhs, seed, ncomp=(4, 3)):
    """Gaussian N(0,1) source [nsites][*ncomp][nrhs], complex64 (re and im each N(0,1))."""
    rng = np.random.default_rng([seed, 0x5B])
    shape = (nsites,) + tuple(ncomp) + (nrhs,)
    return _cgauss_np(rng, shape).astype(np.complex64)


def coarse_links_np(cdims, nbasis, seed):
    """Dense coarse link/self matrices A[V][9][nb][nb], entries N(0,1)/sqrt(nb), complex64."""
    rng = np.random.default_rng([seed, 0x7C])
    V = volume(cdims)
    out = np.empty((V, 9, nbasis, nbasis), dtype=np.complex64)
    scale = 1.0 / np.sqrt(nbasis)
    for x in range(V):                      # chunked so the fp64 temporaries stay small
        out[x] = (_cgauss_np(rng, (9, nbasis, nbasis)) * scale).astype(np.complex64)
    return out


def coarse_vector_np(cdims, nbasis, nrhs, seed):
    return spinor_np(volume(cdims), nrhs, seed, ncomp=(nbasis,))


def gauge_transform_np(dims, seed):
    """Random SU(3) gauge transformation g[V][3][3], complex128 (oracle self-checks only)."""
    rng = np.random.default_rng([seed, 0x8D])
    return su3_np(rng, volume(dims))


# --------------------------------------------------------------- torch (device)

def _cgauss_torch(gen, shape, device):
    import torch
    re = torch.randn(shape, generator=gen, device=device, dtype=torch.float32)
    im = torch.randn(shape, generator=gen, device=device, dtype=torch.float32)
    return torch.complex(re, im)


def gauge_torch(dims, seed, device):
    """Hot gauge field on ``device``: same recipe as gauge_np, drawn with torch's generator."""
    import torch
    gen = torch.Generator(device=device)
    gen.manual_seed(1000003 * seed + 0x6A)
    n = volume(dims) * 4
    a = _cgauss_torch(gen, (n, 3), device).to(torch.complex128)
    a = a / torch.linalg.vector_norm(a, dim=1, keepdim=True)
    b = _cgauss_torch(gen, (n, 3), device).to(torch.complex128)
    b = b - a * torch.sum(torch.conj(a) * b, dim=1, keepdim=True)
    b = b / torch.linalg.vector_norm(b, dim=1, keepdim=True)
    c = torch.conj(torch.linalg.cross(a, b, dim=1))
    U = torch.stack([a, b, c], dim=1).to(torch.complex64)
    return U.reshape(volume(dims), 4, 3, 3).contiguous()


def spinor_torch(nsites, nrhs, seed, device, ncomp=(4, 3)):
    import torch
    gen = torch.Generator(device=device)
    gen.manual_seed(1000003 * seed + 0x5B)
    shape = (nsites,) + tuple(ncomp) + (nrhs,)
    return _cgauss_torch(gen, shape, device).contiguous()


def coarse_links_torch(cdims, nbasis, seed, device):
    import torch
    gen = torch.Generator(device=device)
    gen.manual_seed(1000003 * seed + 0x7C)
    A = _cgauss_torch(gen, (volume(cdims), 9, nbasis, nbasis), device)
    return (A * (1.0 / float(np.sqrt(nbasis)))).contiguous()

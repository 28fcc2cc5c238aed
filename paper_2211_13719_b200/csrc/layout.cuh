// layout.cuh -- field-layout module.
// Site ordering (full and checkerboarded), RHS-fastest element order, and the index
// maps between the canonical layouts of include/mrhs.h and the native ones.
//
// Native fine layout: x-lines cut in blocks of XB sites; inside a block the order is
// [component][site in block][rhs], so the threads of a warp, which run over
// (site in block, rhs pair), read one contiguous 512-byte run per component.
#pragma once
#include "common.cuh"

namespace mrhs {

// Threads of a kernel run over (site in block, rhs pair); one x-block row of one component is
// XB * NP elements (16 B each for even N), contiguous.  XB = largest divisor d of x_eff with
// d <= 16 and d * NP <= 48, NP = threads per site: ~768 contiguous bytes per component row
// while the thread-block tile stays close to a hypercube.
inline int threads_per_site(int nrhs) { return (nrhs % 2 == 0) ? nrhs / 2 : nrhs; }
inline int xblock_host(int x_eff, int nrhs) {
    int np = threads_per_site(nrhs);
    int best = 1;
    for (int d = 1; d <= 16 && d <= x_eff; d++)
        if (x_eff % d == 0 && d * np <= 48) best = d;
    return best;
}

struct FieldGeom {
    int X, Y, Z, T;     // lattice extents
    int cb;             // 0: full lattice field, 1: one parity
    int parity;         // parity of the field when cb
    int Xe;             // sites per x-line of this field (X or X/2)
    int XB;             // layout block extent along x
    int nxb;            // Xe / XB
    int ncomp;          // 12 (fine)
    int N;              // N_rhs
    long long nsites;   // sites of this field

    __host__ __device__ long long nblocks() const { return (long long)nxb * Y * Z * T; }
    __host__ __device__ long long nfloats() const { return nsites * ncomp * 2ll * N; }
};

inline FieldGeom make_geom(const int dims[4], int ncomp, int nrhs, int parity) {
    FieldGeom g;
    g.X = dims[0]; g.Y = dims[1]; g.Z = dims[2]; g.T = dims[3];
    g.cb = parity != MRHS_FULL;
    g.parity = g.cb ? parity : 0;
    g.Xe = g.cb ? g.X / 2 : g.X;
    g.XB = xblock_host(g.Xe, nrhs);
    g.nxb = g.Xe / g.XB;
    g.ncomp = ncomp;
    g.N = nrhs;
    g.nsites = (long long)g.Xe * g.Y * g.Z * g.T;
    return g;
}

// float offset of RHS r (real part; +rhs_im_stride(N) for the imaginary part) inside one
// (site, component) group of 2N floats
__host__ __device__ __forceinline__ int rhs_elem(int N, int r, int im) {
    return (N & 1) ? 2 * r + im : 4 * (r >> 1) + (r & 1) + 2 * im;
}

// x coordinate of site xe of the line (y,z,t) of this field
__host__ __device__ __forceinline__ int x_of(const FieldGeom &g, int xe, int y, int z, int t) {
    return g.cb ? 2 * xe + ((g.parity + y + z + t) & 1) : xe;
}

// native float offset of (site (xe,y,z,t), comp, rhs 0, re)
__host__ __device__ __forceinline__ long long native_offset(const FieldGeom &g, int xe, int y, int z, int t, int comp) {
    int xb = xe / g.XB, xin = xe - xb * g.XB;
    long long b = xb + (long long)g.nxb * (y + (long long)g.Y * (z + (long long)g.Z * t));
    return ((b * g.ncomp + comp) * g.XB + xin) * 2ll * g.N;
}

}  // namespace mrhs

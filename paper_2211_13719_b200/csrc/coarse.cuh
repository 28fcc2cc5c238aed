// coarse.cuh -- host-side interface of the coarse-level 9-point stencil (SURVEY.md Sec. 8(a)
// rows a5, a6; reading S8; PAPER.md:61 nbasis, PAPER.md:75 coarse hopping term).
#pragma once
#include "common.cuh"

namespace mrhs {

struct CoarseGeom {
    int X, Y, Z, T;
    int nb, N;
    long long nsites;
};

// Which sites an apply runs over (the coarse operators exist on the full lattice and, as M_eooe, on one
// parity).  cb = 0: all sites, vectors indexed by lex.  cb = 1: the sites of parity `parity`, output indexed by lex >> 1,
// input vectors (the other parity) also by lex >> 1; the link matrices are always indexed by lex.
struct CoarseSites {
    int X, Y, Z, T;
    int cb, parity;
    long long nout;     // output sites: V or V / 2
};

#ifdef __CUDACC__
// idx-th output site -> lex
__device__ __forceinline__ long long coarse_site_lex(const CoarseSites &g, long long idx) {
    if (!g.cb) return idx;
    long long s = 2 * idx;                 // the pair (2 idx, 2 idx + 1) holds one site of each parity (X even)
    const int x = (int)(s % g.X); s /= g.X;
    const int y = (int)(s % g.Y); s /= g.Y;
    const int z = (int)(s % g.Z);
    const int t = (int)(s / g.Z);
    return 2 * idx + (((x + y + z + t) & 1) != g.parity);
}
// lex of the neighbour at stencil point p (0 self, 1..4 = +x..+t, 5..8 = -x..-t, periodic)
__device__ __forceinline__ long long coarse_neighbour_lex(const CoarseSites &g, long long lex, int p) {
    if (p == 0) return lex;
    long long s = lex;
    int c0 = (int)(s % g.X); s /= g.X;
    int c1 = (int)(s % g.Y); s /= g.Y;
    int c2 = (int)(s % g.Z);
    int c3 = (int)(s / g.Z);
    const int mu = (p - 1) & 3, d = p <= 4 ? 1 : -1;
    if (mu == 0) c0 = (c0 + d + g.X) % g.X;
    else if (mu == 1) c1 = (c1 + d + g.Y) % g.Y;
    else if (mu == 2) c2 = (c2 + d + g.Z) % g.Z;
    else c3 = (c3 + d + g.T) % g.T;
    return c0 + (long long)g.X * (c1 + (long long)g.Y * (c2 + (long long)g.Z * c3));
}
// The same two maps in 32-bit arithmetic without a division per neighbour (coarse lattices have fewer than 2^31 sites; checked at
// create): the kernels evaluate them per stencil point on the thread that issues the copies, where the 64-bit divisions of the
// functions above cost more than the copy itself.
struct CoarseSite32 { int lex, x, y, z, t; };
__device__ __forceinline__ CoarseSite32 coarse_site32(const CoarseSites &g, long long idx) {
    CoarseSite32 c;
    unsigned s = g.cb ? 2u * (unsigned)idx : (unsigned)idx;
    c.lex = (int)s;
    c.x = (int)(s % (unsigned)g.X); s /= (unsigned)g.X;
    c.y = (int)(s % (unsigned)g.Y); s /= (unsigned)g.Y;
    c.z = (int)(s % (unsigned)g.Z);
    c.t = (int)(s / (unsigned)g.Z);
    if (g.cb && (((c.x + c.y + c.z + c.t) & 1) != g.parity)) { c.lex += 1; c.x += 1; }   // the pair (2 idx, 2 idx + 1) differs in x only (X even)
    return c;
}
__device__ __forceinline__ int coarse_neighbour32(const CoarseSites &g, const CoarseSite32 &c, int p) {
    if (p == 0) return c.lex;
    const int mu = (p - 1) & 3;
    const int coord = mu == 0 ? c.x : mu == 1 ? c.y : mu == 2 ? c.z : c.t;
    const int ext = mu == 0 ? g.X : mu == 1 ? g.Y : mu == 2 ? g.Z : g.T;
    const int stride = mu == 0 ? 1 : mu == 1 ? g.X : mu == 2 ? g.X * g.Y : g.X * g.Y * g.Z;
    const int d = p <= 4 ? (coord + 1 == ext ? -(ext - 1) : 1) : (coord == 0 ? ext - 1 : -1);
    return c.lex + d * stride;
}
// The stencil points selected by a mask as a list of 4-bit entries (s-th entry = the s-th set bit), made once per kernel:
// __fns (n-th set bit) is a software loop, too slow for the thread that issues the copies of every stage.
__device__ __forceinline__ unsigned long long coarse_point_list(unsigned mask) {
    unsigned long long l = 0;
    int n = 0;
    for (int p = 0; p < 9; p++)
        if ((mask >> p) & 1u) { l |= (unsigned long long)p << (4 * n); n++; }
    return l;
}
__device__ __forceinline__ int coarse_point(unsigned long long list, int s) { return (int)((list >> (4 * s)) & 15ull); }
#endif
inline CoarseSites coarse_sites_full(const CoarseGeom &g) { return {g.X, g.Y, g.Z, g.T, 0, 0, g.nsites}; }
inline CoarseSites coarse_sites_parity(const CoarseGeom &g, int parity) { return {g.X, g.Y, g.Z, g.T, 1, parity, g.nsites / 2}; }

// canonical A[site][p][row][col] -> native A[site][p][col][row] (one bulk copy per stencil point
// lands the matrix so that a thread's TI consecutive rows of one column are contiguous).
mrhs_status_t pack_coarse_links(const CoarseGeom &g, const float2 *d_canonical, float2 *d_native, cudaStream_t st);

// true if an FP32-FMA specialisation for (nbasis, nrhs) is compiled
bool coarse_fma_supported(int nb, int nrhs);
mrhs_status_t coarse_fma_prepare(const CoarseGeom &g);   // opt in to large dynamic shared memory
// mask: bit p set = stencil point p is applied (0 self, 1..4 = +x..+t, 5..8 = -x..-t); 0x1FF = the 9-point operator
mrhs_status_t launch_coarse_fma(const CoarseGeom &g, const CoarseSites &sites, unsigned mask, const float2 *d_links, const void *d_in, void *d_out, cudaStream_t st);

// ---- tensor-core variant (row a6): tcgen05 kind::tf32 with hi/lo split operands (3 MMAs per K step)
// true if a tensor-core specialisation for (nbasis, nrhs) is compiled (even nrhs only)
bool coarse_tc_supported(int nb, int nrhs);
// canonical A[site][p][row][col] -> [site][p][Re/Im][K chunk][row][4 columns] fp32: the order the kernel's
// operand conversion reads with contiguous 128-bit loads.  Same size as the complex matrices.
mrhs_status_t pack_coarse_links_tc(const CoarseGeom &g, const float2 *d_canonical, float *d_native, cudaStream_t st);
// opt in to large dynamic shared memory and size the persistent grid (CTAs per SM limited by shared memory and TMEM)
mrhs_status_t coarse_tc_prepare(const CoarseGeom &g, int *grid);
mrhs_status_t launch_coarse_tc(const CoarseGeom &g, const CoarseSites &sites, int grid, unsigned mask, const float *d_links, const void *d_in, void *d_out, cudaStream_t st);

// ---- tensor-core variant 2 (row a6, math_mode 2): tcgen05 kind::f16 on operands split into fp16 hi + lo after a power-of-two
// scaling (coarse_h16.cu).  The links are split at create time (same bytes as fp32) with one scale per site; the input vector is
// split per apply into a scratch image of coarse_h16_vec_bytes() bytes (cleared once by the caller: its tail is a chunk of zeros), with one scale per right-hand side (d_colmax: 128 floats and one unsigned counter behind
// them, all zero on entry and zero again when the apply has finished).
bool coarse_h16_supported(int nb, int nrhs);
size_t coarse_h16_vec_bytes(const CoarseGeom &g);
mrhs_status_t pack_coarse_links_h16(const CoarseGeom &g, const float2 *d_canonical, void *d_links16, float *d_site_scale, cudaStream_t st);
mrhs_status_t coarse_h16_prepare(const CoarseGeom &g, int *grid);
mrhs_status_t launch_coarse_h16(const CoarseGeom &g, const CoarseSites &sites, int grid, unsigned mask, const void *d_links16, const float *d_site_scale,
                                const void *d_in, void *d_vec16, float *d_colmax, void *d_out, cudaStream_t st);

}  // namespace mrhs

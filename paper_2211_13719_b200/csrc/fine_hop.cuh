// fine_hop.cuh -- host-side description of the fine-level hopping kernel.  D_hop (full
// lattice) and M_eooe (checkerboarded) are the same device code with different index maps
// ("different site ordering"); reading S3/S4 of DESIGN.md.
#pragma once
#include "layout.cuh"

namespace mrhs {

// Upper bound on threads per block the hop kernel is compiled for (register budget 65536 / 384).
constexpr int kHopMaxThreads = 384;
// Threads per block the default tiling aims for.
constexpr int kHopTargetThreads = 96;

struct HopTiling {
    int by, bz, bt;   // sites per thread-block tile in y, z, t (x extent of a tile is the layout block XB)
    int cy, cz;       // tiles per L2 sweep chunk in y and z
};

struct HopParams {
    int Y, Z, T;              // lattice extents (x enters through Xe, XB, nxb)
    int XB, nxb, NP;          // layout block, blocks per x-line, threads per site
    int cb, out_parity;       // checkerboarded fields? parity of the output field
    int dagger;               // 1: apply the adjoint D_hop^+ = gamma_5 D_hop gamma_5
    int by, bz, bt;           // tile extents
    int cy, cz;               // chunk extents in tiles
    unsigned pf_dist;         // L2 prefetch distance in tiles of the sweep order (0 = off)
    FastDiv d_np, d_xb, d_by, d_bz;             // thread index -> (row, xin, pair) -> (ty, tz, tt)
    FastDiv d_nxb, d_cy, d_cz, d_ntt, d_ncy;    // block index -> tile coordinates in sweep order
    const float4 *gauge_out;  // links living on the sites of the output field, [block][18][xin] float4
    const float4 *gauge_in;   // links living on the sites of the input field
    unsigned grid, threads;
};

// Default tiling for a field geometry: as many rows as fit kHopMaxThreads,
// as cubic as the divisors allow; L2 sweep chunk sized so that the live t-slices fit l2_budget.
HopTiling default_tiling(const FieldGeom &g, size_t l2_budget);
// Fill p (except gauge pointers) from geometry + tiling; false if the tiling does not divide the lattice.
bool build_hop_params(const FieldGeom &g, int out_parity, const HopTiling &t, HopParams &p);

mrhs_status_t launch_hop(const HopParams &p, int nrhs, const void *d_in, void *d_out, cudaStream_t st);

// ---- site-diagonal data (gauge links, packed clover blocks): 72 floats per site, stored
// [block][18][xin] float4 in the block order of the field geometry g.
constexpr int kSiteF4 = 18;
// src: [lex][72] floats in canonical full-lattice site order; dst: native for geometry g.
mrhs_status_t pack_site_data(const FieldGeom &g, const float *d_src, float4 *d_dst, cudaStream_t st);
// inverse, full-lattice geometry only.
mrhs_status_t unpack_site_data(const FieldGeom &g, const float4 *d_src, float *d_dst, cudaStream_t st);

// ---- clover (rows a0, a4)
// d_gauge canonical -> d_packed [lex][72]: per chirality 6 real diagonals then the 15 lower-triangle
// entries (row-major, re,im) of the Hermitian block (readings S5-S7).
mrhs_status_t build_clover(const int dims[4], float mass, float csw, const float2 *d_gauge, float *d_packed, cudaStream_t st);
// canonical blocks [lex][2][6][6] c64 <-> [lex][72]
mrhs_status_t pack_clover_blocks(long long nsites, const float2 *d_blocks, float *d_packed, cudaStream_t st);
// packed blocks [lex][72] -> packed inverse blocks (fp64 Gauss-Jordan per 6x6 block)
mrhs_status_t invert_clover_blocks(long long nsites, const float *d_packed, float *d_packed_inv, cudaStream_t st);
mrhs_status_t unpack_clover_blocks(long long nsites, const float *d_packed, float2 *d_blocks, cudaStream_t st);
// axpy_scale != 0: out = C in + axpy_scale * out instead of out = C in (-1/2: full matrix, -1/4: Schur complement)
mrhs_status_t launch_mooee(const FieldGeom &g, const float4 *d_clover, const void *d_in, void *d_out, cudaStream_t st, float axpy_scale = 0.f);

}  // namespace mrhs

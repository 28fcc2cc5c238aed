// fine_sweep.cuh -- host-side description of the slice-sweep variant of the fine-level hopping kernel
// (readings S3, S4).  Same operator and same native
// layouts as fine_hop.cuh; what differs is how the operands reach the SM:
// a thread block owns a tile of XB x 2 x 2 sites in (x,y,z) and sweeps a segment of t, holding the
// current t-slice of the tile, its y/z/x halo and the links in shared memory (TMA bulk copies from a
// producer warp), so every input spinor crosses the L2 -> SM path about 3x instead of 7x; the two
// half-warps of a consumer warp split every site by the spin row of the projected half spinor.
#pragma once
#include "fine_hop.cuh"

namespace mrhs {

constexpr int kSweepBY = 2, kSweepBZ = 2;        // tile extent in y and z (sites)
constexpr int kSweepRows = kSweepBY * kSweepBZ;
constexpr int kSweepProducerWarps = 4;                          // tile rows, halo rows, links (two warps): one warp per stream of bulk copies
// Four warps per SM sub-partition start with 128 registers; the producer warp group hands most of its share to the three consumer
// warp groups (3 x 152 + 40 <= 512 per lane of a sub-partition).
constexpr int kSweepConsumerRegs = 152, kSweepProducerRegs = 40;
constexpr int kSweepMaxThreads = (kSweepRows * 3 + 4) * 32;   // three consumer warps per tile row, the producer warps, rounded to four warps per SM sub-partition (128 registers)

// Packed backward links of a checkerboarded field (the sweep kernel's second link stream): per site of parity p, in that field's
// block order, [block][kBackF4][xin] float4 =
//   floats 0..53   U_mu(x - mu), mu = x, y, z, each at the position it has in the own-link site data (18 floats per link)
//   floats 56..73  U_t of the site of the OTHER parity with the same checkerboarded index (x-block, xin, y, z, t): the link of the
//                  hop from that site into the slice after it (the kernel carries that hop from step to step)
// so that one contiguous bulk copy per tile row brings every backward link of the step; floats 54, 55, 74, 75 are padding.
constexpr int kBackF4 = 19, kBackT = 14;
mrhs_status_t pack_back_links(const FieldGeom &g, const float *d_gauge_canonical, float4 *d_dst, cudaStream_t st);

struct SweepTiling {
    int lt;          // t-slices one thread block sweeps (divides T)
    int cy, cz;      // tiles per concurrently scheduled chunk in y and z
};

struct SweepParams {
    int Y, Z, T;
    int XB, nxb, NP;              // layout block, blocks per x-line, threads per site (= RHS pairs)
    int cb, out_parity;
    int lt, ntseg;                // slices per segment, segments per t-line
    unsigned n_whole;             // blocks before the tail: the last tail_tiles tiles are cut into tail_seg segments each (whole-line sweeps only)
    int tail_tiles, tail_seg;
    int pf;                       // L2 prefetch distance of the producer, in slices (0 = off)
    int cy, cz;
    FastDiv d_nxb, d_cy, d_cz, d_ntseg, d_ncy;   // block index -> (x-block, tile in chunk, segment, chunk)
    const float4 *gauge_out;      // links on the sites of the output field, [block][18][xin] float4
    const float4 *gauge_in;       // links on the sites of the input field (full lattice: the same array)
    const float4 *gauge_back;     // checkerboarded: the packed backward links of the output sites (pack_back_links)
    const float4 *clover;         // packed clover blocks on the sites of the output field: non-null => out = C H (checkerboarded) or C in - H/2 (full lattice)
    const float4 *aux;            // with clover on checkerboarded fields: non-null => out = C aux - H/4 (Schur complement, second launch)
    int dagger;                   // 1: the adjoint hopping term (gamma_5 D_hop gamma_5)
    unsigned grid, threads;
    unsigned smem_bytes, smem_bytes_clover;   // dynamic shared memory without / with the clover blocks of the fused epilogues
};

// Thread block -> (x-block, first y, first z, first t, slices) of the tile segment it sweeps.  x-blocks fastest, then the tiles of a
// chunk, then segments, then chunks; the last p.tail_tiles tiles of that order are cut into p.tail_seg segments each (blocks
// n_whole, n_whole + 1, ...: the segments of a tile follow one another), so that the blocks of the last, partly filled wave are
// short ones (build_sweep_params).  Shared by the kernel and the host-side plan check (mrhs_sweep_block).
__host__ __device__ __forceinline__ void sweep_block_coords(const SweepParams &p, uint32_t block, int &xb, int &y0, int &z0, int &t0, int &lt) {
    uint32_t bi = block, tseg = 0;
    lt = p.lt;
    if (bi >= p.n_whole) {
        const uint32_t j = bi - p.n_whole, q = j / (uint32_t)p.tail_seg;
        tseg = j - q * (uint32_t)p.tail_seg;
        bi = p.n_whole + q;
        lt = p.T / p.tail_seg;
    }
    uint32_t x, yc, zc, seg, chy, chz, q0;
    p.d_nxb.divmod(bi, q0, x);
    p.d_cy.divmod(q0, q0, yc);
    p.d_cz.divmod(q0, q0, zc);
    p.d_ntseg.divmod(q0, q0, seg);
    p.d_ncy.divmod(q0, chz, chy);
    xb = (int)x;
    y0 = (int)(chy * p.cy + yc) * kSweepBY;
    z0 = (int)(chz * p.cz + zc) * kSweepBZ;
    t0 = (int)(seg + tseg) * lt;
}

// true if the sweep kernel can run this geometry (even N_rhs, shared memory fits)
bool sweep_supported(const FieldGeom &g);
SweepTiling default_sweep_tiling(const FieldGeom &g, int num_sms);
// num_sms: thread blocks resident at the same time (one per SM); 0 = do not balance the last wave
bool build_sweep_params(const FieldGeom &g, int out_parity, const SweepTiling &t, int num_sms, SweepParams &p);
mrhs_status_t sweep_prepare();    // opt in to large dynamic shared memory for every instantiation
mrhs_status_t launch_sweep(const SweepParams &p, const void *d_in, void *d_out, cudaStream_t st);

}  // namespace mrhs

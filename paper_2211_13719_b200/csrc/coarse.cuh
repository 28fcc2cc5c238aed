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

// canonical A[site][p][row][col] -> native A[site][p][col][row] (one bulk copy per stencil point
// lands the matrix so that a thread's TI consecutive rows of one column are contiguous).
mrhs_status_t pack_coarse_links(const CoarseGeom &g, const float2 *d_canonical, float2 *d_native, cudaStream_t st);

// true if an FP32-FMA specialisation for (nbasis, nrhs) is compiled
bool coarse_fma_supported(int nb, int nrhs);
mrhs_status_t coarse_fma_prepare(const CoarseGeom &g);   // opt in to large dynamic shared memory
// mask: bit p set = stencil point p is applied (0 self, 1..4 = +x..+t, 5..8 = -x..-t); 0x1FF = the 9-point operator
mrhs_status_t launch_coarse_fma(const CoarseGeom &g, unsigned mask, const float2 *d_links, const void *d_in, void *d_out, cudaStream_t st);

// ---- tensor-core variant (row a6): tcgen05 kind::tf32 with hi/lo split operands (3 MMAs per K step)
// true if a tensor-core specialisation for (nbasis, nrhs) is compiled (even nrhs only)
bool coarse_tc_supported(int nb, int nrhs);
// canonical A[site][p][row][col] -> [site][p][Re/Im][K chunk][row][4 columns] fp32: the order the kernel's
// operand conversion reads with contiguous 128-bit loads.  Same size as the complex matrices.
mrhs_status_t pack_coarse_links_tc(const CoarseGeom &g, const float2 *d_canonical, float *d_native, cudaStream_t st);
// opt in to large dynamic shared memory and size the persistent grid (CTAs per SM limited by shared memory and TMEM)
mrhs_status_t coarse_tc_prepare(const CoarseGeom &g, int *grid);
mrhs_status_t launch_coarse_tc(const CoarseGeom &g, int grid, unsigned mask, const float *d_links, const void *d_in, void *d_out, cudaStream_t st);

}  // namespace mrhs

// transfer.cuh -- MRHS intergrid operators (reading S9):
//   prolong:  fine(x)[s][c][r] = sum_k phi_k(x)[s][c] coarse(B(x))[chi(s) n_vec + k][r]
//   restrict: coarse(B)[chi n_vec + k][r] = sum_{x in B, s in chi, c} conj(phi_k(x)[s][c]) fine(x)[s][c][r]
// for all N_rhs at once: every basis entry fetched from HBM serves every right-hand side.
#pragma once
#include "layout.cuh"

namespace mrhs {

struct TransferGeom {
    int X, Y, Z, T;          // fine extents
    int bx, by, bz, bt;      // block (aggregate) extents
    int cX, cY, cZ, cT;      // coarse extents
    int nvec, N;             // basis vectors (nbasis = 2 nvec), right-hand sides
    int XB, nxb;             // fine native layout: x-block and blocks per x-line (full lattice)
    long long nsites, ncoarse;
};

// canonical basis [nvec][V][12] complex -> native [V][nvec][12] complex (the 96 bytes of one (site, k) contiguous)
mrhs_status_t pack_basis(const TransferGeom &g, const float2 *d_canonical, float2 *d_native, cudaStream_t st);
mrhs_status_t launch_prolong(const TransferGeom &g, const float2 *d_basis, const void *d_coarse, void *d_fine, cudaStream_t st);
mrhs_status_t launch_restrict(const TransferGeom &g, const float2 *d_basis, const void *d_fine, void *d_coarse, cudaStream_t st);

// ---- coarse -> coarser: the "fine" field is a coarse vector of nf components per site in the coarse
// (site-contiguous) layout, chirality chi(c) = c >= nf / 2;
//   prolong:  out(x)[c][r] = sum_k phi_k(x)[c] coarse(B(x))[chi(c) n_vec + k][r]
//   restrict: coarse(B)[chi n_vec + k][r] = sum_{x in B, c in chi} conj(phi_k(x)[c]) in(x)[c][r]
struct CoarseTransferGeom {
    int X, Y, Z, T;          // extents of the finer (intermediate) coarse lattice
    int bx, by, bz, bt;      // block (aggregate) extents
    int cX, cY, cZ, cT;      // extents of the coarser lattice
    int nf, nvec, N;         // components per finer site (multiple of 4), basis vectors (coarser nbasis = 2 nvec), right-hand sides
    long long nsites, ncoarse;
};
// canonical basis [nvec][Vf][nf] complex -> native [Vf][nvec][nf]
mrhs_status_t pack_basis_coarse(const CoarseTransferGeom &g, const float2 *d_canonical, float2 *d_native, cudaStream_t st);
mrhs_status_t launch_prolong_coarse(const CoarseTransferGeom &g, const float2 *d_basis, const void *d_coarse, void *d_fine, cudaStream_t st);
mrhs_status_t launch_restrict_coarse(const CoarseTransferGeom &g, const float2 *d_basis, const void *d_fine, void *d_coarse, cudaStream_t st);

}  // namespace mrhs

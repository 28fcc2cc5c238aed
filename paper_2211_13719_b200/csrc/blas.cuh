// blas.cuh -- block reductions over the RHS index.
#pragma once
#include "common.cuh"

namespace mrhs {

// thread blocks of the partial-sum pass; the caller provides grid * nrhs double2 of scratch
int inner_grid(int num_sms);
// result[r] = <x_r, y_r> = sum conj(x) y over all sites and components, r < nrhs (<= 256); nfloats = floats of one field
mrhs_status_t launch_inner_products(long long nfloats, int nrhs, const void *d_x, const void *d_y, double2 *d_partial,
                                    int grid, double2 *d_out, cudaStream_t st);

// The same with the partial sums in a file-scope __device__ array of inner_static_capacity() double2 (blas.cu): allocates
// nothing; MRHS_ERR_UNSUPPORTED if grid * nrhs exceeds the capacity.  Calls share the array: calls that overlap on the GPU race.
size_t inner_static_capacity();
mrhs_status_t launch_inner_products_static(long long nfloats, int nrhs, const void *d_x, const void *d_y, int grid,
                                           double2 *d_out, cudaStream_t st);

}  // namespace mrhs

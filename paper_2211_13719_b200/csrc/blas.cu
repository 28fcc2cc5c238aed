// blas.cu -- simultaneous inner products of N_rhs right-hand sides (PAPER.md:85:
// once the matrix part is fast, the block reductions of the Krylov solver become a significant share).
//   result[r] = sum over sites and components of conj(x[.., r]) y[.., r],  r = 0 .. N_rhs - 1
// on two fields in the same native layout (fine or coarse, full or checkerboarded: every native layout is a flat
// array of elements whose index modulo the number of RHS lanes is the RHS lane, layout.cuh).  One pass over both
// fields (HBM-bound: 2 x field bytes), products and sums in fp64, two kernels so that the result is deterministic:
// per-block partial sums, then one block adds the partials in a fixed order.
#include "blas.cuh"
#include <mutex>

// Scratch of the allocation-free entry (mrhs_inner_products_noalloc): the per-block partial sums live in this file-scope array
// instead of a stream-ordered allocation.  2 MiB on every GPU that loads the library, until the process exits.  In host code
// this NAME is a host-side stand-in, not a device address: the host passes kernels the address cudaGetSymbolAddress returns.
static constexpr size_t kInnerStaticPartials = 131072;     // double2 elements: thread blocks x N_rhs of one call at most
static __device__ __align__(256) double2 g_mrhs_inner_scratch[kInnerStaticPartials];

namespace mrhs {

namespace {

constexpr int kInnerMaxBlock = 256;

// R = 2: element = float4 (re0 re1 im0 im1) of one RHS pair; R = 1: float2 (re im) of one RHS
template <int R>
__global__ void __launch_bounds__(kInnerMaxBlock)
inner_partial_kernel(const typename Elem<R>::type *__restrict__ x, const typename Elem<R>::type *__restrict__ y,
                     long long nelem, int lanes, double2 *__restrict__ partial) {
    __shared__ double sh[2 * R][kInnerMaxBlock];
    const int tid = threadIdx.x;
    const long long stride = (long long)gridDim.x * blockDim.x;   // a multiple of lanes: this thread keeps its RHS lane
    double acc[2 * R];
#pragma unroll
    for (int k = 0; k < 2 * R; k++) acc[k] = 0.0;
#pragma unroll 4
    for (long long e = (long long)blockIdx.x * blockDim.x + tid; e < nelem; e += stride) {
        if constexpr (R == 2) {
            const float4 a = __ldg(x + e), b = __ldg(y + e);
            acc[0] += (double)a.x * b.x + (double)a.z * b.z;   // Re, first RHS of the pair
            acc[1] += (double)a.x * b.z - (double)a.z * b.x;   // Im
            acc[2] += (double)a.y * b.y + (double)a.w * b.w;   // second RHS
            acc[3] += (double)a.y * b.w - (double)a.w * b.y;
        } else {
            const float2 a = __ldg(x + e), b = __ldg(y + e);
            acc[0] += (double)a.x * b.x + (double)a.y * b.y;
            acc[1] += (double)a.x * b.y - (double)a.y * b.x;
        }
    }
#pragma unroll
    for (int k = 0; k < 2 * R; k++) sh[k][tid] = acc[k];
    __syncthreads();
    if (tid < lanes) {
        double s[2 * R];
#pragma unroll
        for (int k = 0; k < 2 * R; k++) s[k] = 0.0;
        for (int j = tid; j < (int)blockDim.x; j += lanes)
#pragma unroll
            for (int k = 0; k < 2 * R; k++) s[k] += sh[k][j];
        double2 *o = partial + (size_t)blockIdx.x * lanes * R + (size_t)tid * R;
#pragma unroll
        for (int a = 0; a < R; a++) o[a] = make_double2(s[2 * a], s[2 * a + 1]);
    }
}

// one block per RHS: 256 threads add the partials of their stride in block order, then a fixed-shape tree
__global__ void __launch_bounds__(256)
inner_final_kernel(const double2 *__restrict__ partial, int nblocks, int nrhs, double2 *__restrict__ out) {
    __shared__ double sre[256], sim[256];
    const int r = blockIdx.x, tid = threadIdx.x;
    double re = 0.0, im = 0.0;
    for (int b = tid; b < nblocks; b += 256) {
        const double2 v = partial[(size_t)b * nrhs + r];
        re += v.x; im += v.y;
    }
    sre[tid] = re; sim[tid] = im;
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if (tid < w) { sre[tid] += sre[tid + w]; sim[tid] += sim[tid + w]; }
        __syncthreads();
    }
    if (tid == 0) out[r] = make_double2(sre[0], sim[0]);
}

}  // namespace

int inner_grid(int num_sms) { return num_sms * 8; }

mrhs_status_t launch_inner_products(long long nfloats, int nrhs, const void *d_x, const void *d_y, double2 *d_partial,
                                    int grid, double2 *d_out, cudaStream_t st) {
    const int R = (nrhs & 1) ? 1 : 2;
    const int lanes = nrhs / R;
    const int block = lanes * (kInnerMaxBlock / lanes);
    const long long nelem = nfloats / (2 * R);
    if (R == 2) inner_partial_kernel<2><<<grid, block, 0, st>>>((const float4 *)d_x, (const float4 *)d_y, nelem, lanes, d_partial);
    else        inner_partial_kernel<1><<<grid, block, 0, st>>>((const float2 *)d_x, (const float2 *)d_y, nelem, lanes, d_partial);
    MRHS_CUDA(cudaGetLastError());
    inner_final_kernel<<<nrhs, 256, 0, st>>>(d_partial, grid, nrhs, d_out);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

size_t inner_static_capacity() { return kInnerStaticPartials; }

// The same two kernels with the partial sums in g_mrhs_inner_scratch.  No allocation: the device address of the array is
// looked up once per device (with that device current: it is the caller's current device) and cached.  Nothing has to be
// cleared between calls: the first kernel writes every one of the grid * nrhs partials the second one reads.
mrhs_status_t launch_inner_products_static(long long nfloats, int nrhs, const void *d_x, const void *d_y, int grid,
                                           double2 *d_out, cudaStream_t st) {
    if ((size_t)grid * (size_t)nrhs > kInnerStaticPartials) {
        set_error("inner products (no alloc): %d thread blocks x %d right-hand sides = %zu partial sums exceed the static scratch of %zu",
                  grid, nrhs, (size_t)grid * (size_t)nrhs, kInnerStaticPartials);
        return MRHS_ERR_UNSUPPORTED;
    }
    constexpr int kMaxDev = 64;
    static std::mutex mu;
    static double2 *addr[kMaxDev] = {};
    int dev = 0;
    MRHS_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDev) { set_error("inner products (no alloc): device ordinal %d out of range", dev); return MRHS_ERR_UNSUPPORTED; }
    double2 *partial = nullptr;
    {
        std::lock_guard<std::mutex> lock(mu);
        if (!addr[dev]) {
            void *p = nullptr;
            MRHS_CUDA(cudaGetSymbolAddress(&p, g_mrhs_inner_scratch));
            if (!p) { set_error("inner products (no alloc): cudaGetSymbolAddress returned NULL"); return MRHS_ERR_CUDA; }
            addr[dev] = (double2 *)p;
        }
        partial = addr[dev];
    }
    return launch_inner_products(nfloats, nrhs, d_x, d_y, partial, grid, d_out, st);
}

}  // namespace mrhs

// coarse_h16.cu -- coarse-level 9-point stencil, second tensor-core variant (math_mode 2):
//   out_i(x) = sum_{p=0..8} sum_j A_p(x)_ij v_j(x + delta_p)          (reading S8)
// on tcgen05.mma kind::f16 (K = 16 per instruction, half as many instructions as kind::tf32) with every fp32 number
// represented as the sum of two fp16 numbers after an exact power-of-two scaling (reading S15, split precision):
//   s x = hi + lo,   hi = fp16(s x),  lo = fp16(s x - hi),   s = 2^k chosen so that max |s x| is in [2^14, 2^15)
//   (A v) ~ (A_hi v_hi + A_hi v_lo + A_lo v_hi) / (s_A s_v)      products exact, fp32 accumulation in tensor memory
// hi carries 11 bits and lo the next 11; elements down to 2^-17 of the largest one keep full fp32 relative accuracy, smaller ones
// an absolute error of 2^-40 of the largest (fp16 subnormals).  The scale of the matrices is per site (all nine matrices of a site add
// up in one accumulator), that of the vectors per right-hand side over the whole field (the tolerance of north_star is per RHS).
//
// The split is NOT done in the stencil kernel:
//   * link matrices: split once at create time into the operand image the MMA reads (same bytes as fp32: 2 + 2 per real number);
//   * vectors: two small passes per apply (column maxima; split into the operand image, 2 x 2 N_rhs (rounded) fp16 per component),
//     instead of converting each vector nine times, once per stencil point that reads it.
// The stencil kernel is then a plain TMA -> tcgen05 -> epilogue pipeline: one persistent block per SM, one copy warp (three bulk
// copies per stencil point), one MMA warp, eight epilogue warps, operand ring of two to eight stages, two accumulator sets in
// tensor memory so that the epilogue of a site runs under the MMAs of the next.
//
// Per site the complex contraction is ONE real GEMM accumulated over the stencil points, D[128 x cols] += Aop[128 x 16] Bop[16 x cols]:
//   Aop rows (TMEM lanes): groups of 16 components, each group 16 rows of Re A followed by the same 16 rows of Im A (a last group of
//                          8 + 8 if nbasis mod 16 = 8), so Re and Im of an output component sit in the same 32-lane quarter;
//   Bop cols 0..N-1 = Re v_hi, NT/2..NT/2+N-1 = Im v_hi, NT..2NT-1 the same for v_lo     (NT = 2 N rounded up to 16)
//   stacked B (2 NT <= 256): A_hi x [v_hi | v_lo] and A_lo x v_hi, two MMAs per K step, hi*lo in accumulator columns NT..2NT-1;
//   otherwise three MMAs per K step into columns 0..NT-1;
//   stacked A (4 nbasis <= 128, i.e. nbasis 24): the A_lo rows follow the A_hi rows of the same 8 components inside a lane quarter,
//   [A_hi ; A_lo] x [v_hi | v_lo] is ONE MMA per K step (two without the stacked B), hi and lo rows added by a warp shuffle.
//   Re out = D[Re i][n] - D[Im i][NT/2 + n],  Im out = D[Re i][NT/2 + n] + D[Im i][n]   (one warp shuffle per value).
// nbasis / 8 K chunks of 16 bytes per point, an MMA takes two: with an odd count a stage holds two stencil points back to back and a
// site's last single point is followed by one chunk of zeros copied from a zero buffer (nothing is padded in HBM).
#include "coarse.cuh"
#include "tcgen05.cuh"
#include <cuda_fp16.h>
#include <cstdlib>

namespace mrhs {

namespace {

// programmatic dependent launch: wait for the preceding kernel of the stream (no-op in a normal launch); let the next one start early
__device__ __forceinline__ void grid_dependency_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void grid_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
// 8 consecutive fp32 columns of this thread's TMEM lane.  Asynchronous: the registers hold the values only after tmem_ld_wait(),
// so that the loads of one chunk (two to four) are in flight together.
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&r)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr)
                 : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// Exponent k of the scale 2^k that brings a largest magnitude m into [2^14, 2^15) (fp16 overflows at 65504); 0 for m = 0.
__device__ __forceinline__ int scale_exp(float m) {
    if (!(m > 0.f) || !(m <= 3.0e38f)) return 0;      // zero field, or Inf / NaN in the input: no scaling (the result is Inf / NaN as in fp32)
    int e = ilogbf(m);
    if (e < -100) e = -100;
    return 14 - e;
}

constexpr unsigned kH16SmemLimit = 227u * 1024u;
constexpr int kH16MaxStages = 8;

template <int NB, int N>
struct H16Cfg {
    static_assert(N % 2 == 0, "the tensor-core variants use the RHS-pair element layout (even N_rhs)");
    static_assert(NB % 8 == 0 && NB <= 64, "nbasis must be a multiple of 8 and fit 128 operand rows");
    static constexpr int NP = N / 2;                          // float4 elements per component
    static constexpr int NT = ((2 * N + 15) / 16) * 16;       // columns of one of v_hi / v_lo: Re at 0, Im at NT / 2
    static constexpr int KC = NB / 8;                         // 16-byte K chunks (8 fp16) per stencil point
    // An MMA takes K = 16 = two chunks.  With an odd chunk count per point (nbasis = 24, 40) a stage holds TWO stencil points whose
    // chunks follow each other (2 KC chunks = KC MMA steps for two points); a site's last, single point is followed by one chunk of
    // zeros in the B operand (copied from a zero buffer, not stored per site): nbasis 40: 23 K steps per site instead of 27.
    static constexpr int PP = KC % 2 ? 2 : 1;                 // stencil points per operand stage
    static constexpr int KCP = PP * KC;                       // chunks of one stage in shared memory (even)
    // Stacked A operand (4 nbasis <= 128 rows, i.e. nbasis 24): the rows of A_lo follow those of A_hi in the SAME operand, so one MMA
    // forms A_hi x B and A_lo x B at once (an MMA of this size costs a fixed ~77 cycles + ~0.6 per column whatever its row count):
    // with the stacked B operand ONE MMA per K step, all four hi / lo products (lo x lo is exact too and is simply kept).
    static constexpr bool SA = 4 * NB <= 128;
    static constexpr int NA = SA ? 1 : 2;                     // A operands per stencil point
    static constexpr int GW = SA ? 8 : 16;                    // components per TMEM lane quarter
    static constexpr int NG = (NB + GW - 1) / GW;             // TMEM lane quarters with rows
    static constexpr int ROWS = (SA ? 4 : 2) * NB;            // stored rows of one A operand
    static constexpr bool STK = 2 * NT <= 256;                // stacked B operand: two MMAs per K step
    static constexpr int D_COLS = STK ? 2 * NT : NT;          // accumulator columns of one set
    static constexpr int TMEM_COLS = pow2_cols(2 * D_COLS);   // two sets
    static constexpr int A_LBO = ROWS * 16;
    static constexpr int B_LBO = 2 * NT * 16;
    static constexpr int A_HALF = KC * A_LBO;                 // bytes of one A operand (A_hi or A_lo; stacked: both) of one matrix in HBM
    static constexpr int A_SLOT = KCP * A_LBO;                // and in shared memory
    static constexpr int B_COPY = KC * B_LBO;                 // bytes of one split vector [chunk][hi cols | lo cols][8]
    static constexpr int B_SLOT = KCP * B_LBO;
    static constexpr int STAGE = NA * A_SLOT + B_SLOT;
    static constexpr int TAIL = 512 + 256;                    // column scales (N <= 128 floats), mbarriers + TMEM slot
    static constexpr int NSTAGE = (int)((kH16SmemLimit - TAIL) / STAGE) < kH16MaxStages ? (int)((kH16SmemLimit - TAIL) / STAGE) : kH16MaxStages;
    static constexpr int SMEM_BYTES = NSTAGE * STAGE + TAIL;
    static constexpr int THREADS = 10 * 32;                   // copy, MMA, eight epilogue warps (two per TMEM lane quarter)
    static_assert(NSTAGE >= 2, "operand ring needs two stages");
    static_assert(KCP % 2 == 0, "whole MMAs per stage");
    static_assert(NT <= 256 && 2 * D_COLS <= 512 && N <= 128, "MMA N / TMEM limit");
};

// links16: [site][p][hi | lo][K chunk][row][8 fp16] (stacked A: [site][p][K chunk][row of hi or lo][8 fp16]); site_scale[site] = 1 / s_A; vec16: [site][K chunk][2 NT columns][8 fp16];
// zeros: one K chunk of the B operand (2 NT x 16 bytes) of zeros;
// colmax[n] = max |v| of RHS n (both written by the passes below; 128 floats, cleared again by this kernel), blocks_done: a zero counter; out: coarse vectors [site][component][RHS pair] float4.
// CM: the point mask at compile time (0x1FF the nine-point operator, 0x1FE the hopping term: the argument is ignored, the loops over
// the points unroll and every point index folds into the address arithmetic of the thread that issues the copies), or 0: the
// argument `mask` at run time (any subset; the point list is unpacked once)
__host__ __device__ constexpr int h16_nth_point(unsigned m, int n) {
    int c = 0;
    for (int p = 0; p < 9; p++)
        if ((m >> p) & 1u) { if (c == n) return p; c++; }
    return 0;
}
__host__ __device__ constexpr int h16_popc(unsigned m) { int c = 0; for (int p = 0; p < 9; p++) c += (m >> p) & 1u; return c; }
template <int NB, int N, unsigned CM>
__global__ void __launch_bounds__(H16Cfg<NB, N>::THREADS, 1)
coarse_h16_kernel(const CoarseSites sites, unsigned mask, const unsigned char *__restrict__ links16, const float *__restrict__ site_scale,
                  const unsigned char *__restrict__ vec16, const unsigned char *__restrict__ zeros, float *colmax,
                  unsigned *blocks_done, float4 *__restrict__ out) {
    typedef H16Cfg<NB, N> C;
    extern __shared__ __align__(128) unsigned char smem[];
    float *cinv = reinterpret_cast<float *>(smem + C::NSTAGE * C::STAGE);
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + C::NSTAGE * C::STAGE + 512);
    uint64_t *full = bars, *empty = bars + kH16MaxStages, *accfull = bars + 2 * kH16MaxStages, *accfree = accfull + 2;
    uint32_t *tslot = reinterpret_cast<uint32_t *>(accfull + 4);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < C::NSTAGE; s++) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
        for (int a = 0; a < 2; a++) { mbar_init(&accfull[a], 1); mbar_init(&accfree[a], 2 * C::NG); }
        mbar_fence_init();
    }
    // the padding chunks (and, before the first fill, everything else) read as zero
    for (int i = tid; i < C::NSTAGE * C::STAGE / 16; i += C::THREADS) reinterpret_cast<float4 *>(smem)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    fence_async_smem();
    if (warp == 0) tmem_alloc<C::TMEM_COLS>(tslot);
    // Launched with programmatic stream serialization: everything above overlaps the tail of the split pass; what follows reads its output
    grid_dependency_wait();
    for (int n = tid; n < N; n += C::THREADS) cinv[n] = ldexpf(1.f, -scale_exp(colmax[n]));
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    // The column maxima must be zero again when the next apply starts: the last block to have read them clears them (and the
    // counter), so every apply leaves the handle as it found it (no memset launch, and safe under graph replay).
    if (tid == 64) {
        __threadfence();
        if (atomicAdd(blocks_done, 1u) == gridDim.x - 1) {
            for (int n = 0; n < 128; n++) colmax[n] = 0.f;
            *blocks_done = 0u;
        }
    }
    const uint32_t tmem = *tslot;

    const long long nsites = sites.nout;       // output sites, enumerated by osite; the links of output site osite live at its lex
    const int npts = CM ? h16_popc(CM) : __popc(mask);
    const unsigned long long plist = CM ? 0ull : coarse_point_list(mask);
    auto point = [&](int s) { return CM ? h16_nth_point(CM, s) : coarse_point(plist, s); };

    if (warp == 0) {
        // ------------------------------------------------------------------ copy warp
        if (lane == 0) {
            uint32_t s = 0, ph = 1;    // stage of the next fill; parity of the release it waits for once the ring has wrapped
            bool wrapped = false;
            for (long long site = blockIdx.x; site < nsites; site += gridDim.x) {
                const CoarseSite32 sc = coarse_site32(sites, site);
                const long long lex = sc.lex;
#pragma unroll
                for (int sp = 0; sp < npts; sp += C::PP) {
                    if (wrapped) mbar_wait(&empty[s], ph);
                    unsigned char *dst = smem + (size_t)s * C::STAGE;
                    const bool two = C::PP == 2 && sp + 1 < npts;
                    mbar_expect_tx(&full[s], (two ? 2 : 1) * (C::NA * C::A_HALF + C::B_COPY) + (C::PP == 2 && !two ? C::B_LBO : 0));
#pragma unroll
                    for (int k = 0; k < C::PP; k++) {
                        if (k == 1 && !two) break;
                        const int p = point(sp + k);
                        // vector index of the neighbour at stencil point p: 0 self, 1..4 = +x..+t, 5..8 = -x..-t (periodic)
                        long long nbr = coarse_neighbour32(sites, sc, p);
                        if (sites.cb) nbr >>= 1;
                        const unsigned char *a = links16 + ((size_t)lex * 9 + p) * (C::NA * C::A_HALF);
                        bulk_g2s(dst + k * C::A_HALF, a, C::A_HALF, &full[s]);
                        if (!C::SA) bulk_g2s(dst + C::A_SLOT + k * C::A_HALF, a + C::A_HALF, C::A_HALF, &full[s]);
                        bulk_g2s(dst + C::NA * C::A_SLOT + k * C::B_COPY, vec16 + (size_t)nbr * C::B_COPY, C::B_COPY, &full[s]);
                    }
                    if (C::PP == 2 && !two) bulk_g2s(dst + C::NA * C::A_SLOT + C::B_COPY, zeros, C::B_LBO, &full[s]);     // K padding of a single point
                    if (++s == (uint32_t)C::NSTAGE) { s = 0; ph ^= 1u; wrapped = true; }
                }
            }
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA warp: the whole warp walks the stages, one elected lane issues
        constexpr uint32_t idesc = instr_desc_f16(128, C::NT), idesc2 = instr_desc_f16(128, C::STK ? 2 * C::NT : C::NT);
        uint32_t s = 0, ph = 0, sl = 0;
        for (long long site = blockIdx.x; site < nsites; site += gridDim.x, sl++) {
            const uint32_t a = sl & 1u;
            if (sl >= 2) mbar_wait(&accfree[a], ((sl >> 1) - 1) & 1u);      // the epilogue has read this accumulator set
            tc_fence_after();
            const uint32_t d = tmem + a * C::D_COLS;
            for (int sp = 0; sp < npts; sp += C::PP) {
                mbar_wait(&full[s], ph);
                tc_fence_after();
                const int steps = C::PP == 2 && sp + 1 >= npts ? (C::KC + 1) / 2 : C::KCP / 2;
                if (elect_one()) {
                    const uint32_t ah = smem_u32(smem + (size_t)s * C::STAGE), al = ah + C::A_SLOT, bh = ah + C::NA * C::A_SLOT, bl = bh + C::NT * 16;
                    for (int ks = 0; ks < steps; ks++) {
                        const uint64_t dah = smem_desc(ah + ks * 2 * C::A_LBO, C::A_LBO, 128);
                        const uint64_t dal = smem_desc(al + ks * 2 * C::A_LBO, C::A_LBO, 128);
                        const uint64_t dbh = smem_desc(bh + ks * 2 * C::B_LBO, C::B_LBO, 128);
                        if (C::SA) {
                            mma_f16(d, dah, dbh, idesc2, (sp | ks) != 0);     // [hi ; lo] x [hi | lo], or [hi ; lo] x hi
                            if (!C::STK) mma_f16(d, dah, smem_desc(bl + ks * 2 * C::B_LBO, C::B_LBO, 128), idesc, 1);    // [hi ; lo] x lo, same columns
                        } else if (C::STK) {
                            mma_f16(d, dah, dbh, idesc2, (sp | ks) != 0);     // hi x [hi | lo]
                            mma_f16(d, dal, dbh, idesc, 1);                    // lo x hi
                        } else {
                            const uint64_t dbl = smem_desc(bl + ks * 2 * C::B_LBO, C::B_LBO, 128);
                            mma_f16(d, dal, dbh, idesc, (sp | ks) != 0);
                            mma_f16(d, dah, dbl, idesc, 1);
                            mma_f16(d, dah, dbh, idesc, 1);
                        }
                    }
                    mma_commit(&empty[s]);                           // the operand stage is free once these MMAs have read it
                    if (sp + C::PP >= npts) mma_commit(&accfull[a]); // all points of the site accumulated
                }
                __syncwarp();
                if (++s == (uint32_t)C::NSTAGE) { s = 0; ph ^= 1u; }
            }
        }
    } else {
        // ------------------------------------------------------------------ epilogue warps: a warp reads the TMEM lane quarter warp & 3;
        // the two warps of a quarter take the even and the odd chunks of eight columns
        const int g = warp & 3, half = (warp - 2) >> 2;
        if (g < C::NG) {
            // rows of a quarter: w components x (Re, Im); stacked A: 8 components x (Re, Im) of A_hi, then the same of A_lo
            const int w = C::SA ? 8 : (NB - 16 * g < 16 ? NB - 16 * g : 16);
            const int part = (lane / w) & 1, i = C::GW * g + lane % w;
            const bool live = lane < 2 * w;
            uint32_t sl = 0;
            for (long long site = blockIdx.x; site < nsites; site += gridDim.x, sl++) {
                const uint32_t a = sl & 1u;
                const float sa = site_scale[coarse_site32(sites, site).lex];
                mbar_wait(&accfull[a], (sl >> 1) & 1u);
                tc_fence_after();
                float *o = reinterpret_cast<float *>(out + ((size_t)site * NB + (live ? i : 0)) * C::NP) + 2 * part;
                const uint32_t t0 = tmem + ((uint32_t)(g * 32) << 16) + a * C::D_COLS;
                constexpr int NCH = (N + 7) / 8, NCHW = (NCH + 1) / 2;
#pragma unroll
                for (int c = 0; c < NCHW; c++) {
                    const int ch = 2 * c + half;
                    uint32_t rx[8], ry[8], rxa[8], rya[8];
                    if (ch < NCH) {
                        tmem_ld8(t0 + ch * 8, rx);
                        tmem_ld8(t0 + C::NT / 2 + ch * 8, ry);
                        if (C::STK) {
                            tmem_ld8(t0 + C::NT + ch * 8, rxa);
                            tmem_ld8(t0 + C::NT + C::NT / 2 + ch * 8, rya);
                        }
                        tmem_ld_wait();
                    }
                    if (c == NCHW - 1) {
                        // the accumulator has been read: hand it back before the arithmetic and the stores
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(&accfree[a]);
                    }
                    if (ch < NCH) {
                        float x[8], y[8];
#pragma unroll
                        for (int k = 0; k < 8; k++) {
                            x[k] = __uint_as_float(rx[k]);
                            y[k] = __uint_as_float(ry[k]);
                            if (C::STK) { x[k] += __uint_as_float(rxa[k]); y[k] += __uint_as_float(rya[k]); }
                            if (C::SA) {      // the A_lo rows sit 16 lanes further
                                x[k] += __shfl_xor_sync(0xffffffffu, x[k], 16);
                                y[k] += __shfl_xor_sync(0xffffffffu, y[k], 16);
                            }
                        }
#pragma unroll
                        for (int k = 0; k < 8; k += 2) {
                            const int n = ch * 8 + k;
                            const float r0 = __shfl_xor_sync(0xffffffffu, y[k], w);          // the partner row's Im-column value
                            const float r1 = __shfl_xor_sync(0xffffffffu, y[k + 1], w);
                            if (n < N && live) {
                                // Re row: Re out = D[Re i][n] - D[Im i][NT/2 + n];  Im row: Im out = D[Re i][NT/2 + n] + D[Im i][n]
                                const float v0 = (part ? r0 + x[k] : x[k] - r0) * sa * cinv[n];          // two exact power-of-two factors, applied one after the other
                                const float v1 = (part ? r1 + x[k + 1] : x[k + 1] - r1) * sa * cinv[n + 1];
                                *reinterpret_cast<float2 *>(o + 2 * n) = make_float2(v0, v1);      // element n / 2 = (re0 re1 im0 im1)
                            }
                        }
                    }
                }
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_free<C::TMEM_COLS>(tmem);
}

// ---- passes over the input vector: column maxima, then the split operand image
__device__ __forceinline__ void atomic_max_abs(float *addr, float m) {
    atomicMax(reinterpret_cast<unsigned int *>(addr), __float_as_uint(m));     // non-negative floats order like their bit patterns
}
// grid * block is a multiple of np, so a thread sees one RHS pair only
__global__ void h16_colmax_kernel(const float4 *__restrict__ in, long long total, int np, float *__restrict__ colmax) {
    grid_launch_dependents();      // the split pass may be scheduled now; it waits for this grid before it reads colmax
    const long long stride = (long long)gridDim.x * blockDim.x;
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int q = (int)(e % np);
    float m0 = 0.f, m1 = 0.f;
    for (; e < total; e += stride) {
        const float4 v = __ldg(in + e);
        m0 = fmaxf(m0, fmaxf(fabsf(v.x), fabsf(v.z)));
        m1 = fmaxf(m1, fmaxf(fabsf(v.y), fabsf(v.w)));
    }
    // lanes with the same q: every np-th thread; reduce through shared memory per block
    __shared__ float sm[2 * 64];
    for (int i = threadIdx.x; i < 2 * np; i += blockDim.x) sm[i] = 0.f;
    __syncthreads();
    atomic_max_abs(&sm[2 * q], m0);
    atomic_max_abs(&sm[2 * q + 1], m1);
    __syncthreads();
    for (int i = threadIdx.x; i < 2 * np; i += blockDim.x) atomic_max_abs(&colmax[i], sm[i]);
}
__device__ __forceinline__ void split_h16(float x, __half &hi, __half &lo) {
    hi = __float2half_rn(x);
    lo = __float2half_rn(x - __half2float(hi));
}
union H8 { uint4 u; __half h[8]; };
// one thread per (site, K chunk, column pair): 8 components of one RHS pair -> Re / Im rows of both RHS, hi and lo; the column
// pairs past N_rhs are the zero padding of the operand
__global__ void h16_split_vec_kernel(const float4 *__restrict__ in, long long nsites, int nb, int np, int nt, const float *__restrict__ colmax,
                                     uint4 *__restrict__ vec16) {
    grid_launch_dependents();      // the stencil kernel may start its set-up; it waits for this grid before it reads vec16
    grid_dependency_wait();        // launched with programmatic stream serialization after the column-maximum pass
    const int kcn = nb / 8, qn = nt / 4;
    const long long total = nsites * kcn * qn;
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int q = (int)(idx % qn);
    const long long r = idx / qn;
    const int kc = (int)(r % kcn);
    const long long site = r / kcn;
    uint4 *dst = vec16 + (size_t)(site * kcn + kc) * 2 * nt;
    H8 o[8];      // [hi, lo] x [Re 2q, Re 2q+1, Im 2q, Im 2q+1]
#pragma unroll
    for (int k = 0; k < 8; k++) o[k].u = make_uint4(0u, 0u, 0u, 0u);
    if (q < np) {
        const float s0 = ldexpf(1.f, scale_exp(colmax[2 * q])), s1 = ldexpf(1.f, scale_exp(colmax[2 * q + 1]));
#pragma unroll
        for (int j = 0; j < 8; j++) {
            const float4 v = __ldg(in + ((size_t)site * nb + 8 * kc + j) * np + q);
            split_h16(v.x * s0, o[0].h[j], o[4].h[j]);
            split_h16(v.y * s1, o[1].h[j], o[5].h[j]);
            split_h16(v.z * s0, o[2].h[j], o[6].h[j]);
            split_h16(v.w * s1, o[3].h[j], o[7].h[j]);
        }
    }
    dst[2 * q] = o[0].u;
    dst[2 * q + 1] = o[1].u;
    dst[nt / 2 + 2 * q] = o[2].u;
    dst[nt / 2 + 2 * q + 1] = o[3].u;
    dst[nt + 2 * q] = o[4].u;
    dst[nt + 2 * q + 1] = o[5].u;
    dst[nt + nt / 2 + 2 * q] = o[6].u;
    dst[nt + nt / 2 + 2 * q + 1] = o[7].u;
}

// ---- create time: per-site maximum of the nine matrices, then the split operand image
__global__ void h16_site_max_kernel(const float2 *__restrict__ src, int per_site, float *__restrict__ site_max) {
    const long long site = blockIdx.x;
    float m = 0.f;
    for (int i = threadIdx.x; i < per_site; i += blockDim.x) {
        const float2 a = src[site * per_site + i];
        m = fmaxf(m, fmaxf(fabsf(a.x), fabsf(a.y)));
    }
    __shared__ float sm;
    if (threadIdx.x == 0) sm = 0.f;
    __syncthreads();
    atomic_max_abs(&sm, m);
    __syncthreads();
    if (threadIdx.x == 0) site_max[site] = sm;
}
// canonical A[site][p][row][col] complex -> [site][p][hi | lo][K chunk][operand row][8 fp16]; one thread per (matrix, chunk, operand row);
// site_scale: in = the site maximum, out (by the thread of the site's first unit) = 1 / s_A
__global__ void h16_pack_links_kernel(int nb, const float2 *__restrict__ src, uint4 *__restrict__ dst, float *__restrict__ site_scale, long long total) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int kcn = nb / 8, rows = 2 * nb;
    const bool sa = 4 * nb <= 128;         // stacked A operand (H16Cfg::SA)
    const int u = (int)(idx % (kcn * rows));
    const long long mat = idx / (kcn * rows);
    const long long site = mat / 9;
    const int kc = u / rows, rr = u - kc * rows;
    // operand row rr -> (part, component); stacked: rr enumerates the hi rows, (part, component) = (rr / 8 & 1, 8 (rr / 16) + rr % 8)
    const int g = sa ? rr >> 4 : rr >> 5, w = sa ? 8 : (nb - 16 * g < 16 ? nb - 16 * g : 16);
    const int part = sa ? (rr >> 3) & 1 : (rr - 32 * g) / w, i = sa ? 8 * g + (rr & 7) : 16 * g + (rr - 32 * g) % w;
    const int k = scale_exp(site_scale[site]);
    const float s = ldexpf(1.f, k);
    H8 hi, lo;
#pragma unroll
    for (int j = 0; j < 8; j++) {
        const float2 a = src[(mat * nb + i) * nb + 8 * kc + j];
        split_h16((part ? a.y : a.x) * s, hi.h[j], lo.h[j]);
    }
    uint4 *d = dst + (size_t)mat * 2 * kcn * rows;
    if (sa) {       // [K chunk][quarter: 8 Re hi, 8 Im hi, 8 Re lo, 8 Im lo][8 fp16]
        const int r4 = 32 * g + 8 * part + (rr & 7);
        d[kc * 2 * rows + r4] = hi.u;
        d[kc * 2 * rows + r4 + 16] = lo.u;
    } else {
        d[kc * rows + rr] = hi.u;
        d[(kcn + kc) * rows + rr] = lo.u;
    }
}
__global__ void h16_site_scale_kernel(float *__restrict__ site_scale, long long nsites) {
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s < nsites) site_scale[s] = ldexpf(1.f, -scale_exp(site_scale[s]));
}

template <int NB, int N>
mrhs_status_t h16_prepare_t() {
    typedef H16Cfg<NB, N> C;
    MRHS_CUDA(cudaFuncSetAttribute(coarse_h16_kernel<NB, N, 0x1FFu>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
    MRHS_CUDA(cudaFuncSetAttribute(coarse_h16_kernel<NB, N, 0x1FEu>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
    MRHS_CUDA(cudaFuncSetAttribute(coarse_h16_kernel<NB, N, 0u>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
    return MRHS_OK;
}
template <int NB, int N>
mrhs_status_t h16_launch_t(const CoarseSites &sites, int grid, unsigned mask, const void *links16, const float *site_scale, const void *vec16,
                           const void *zeros, float *colmax, unsigned *blocks_done, void *out, cudaStream_t st) {
    typedef H16Cfg<NB, N> C;
    if ((long long)grid > sites.nout) grid = (int)sites.nout;
    // programmatic stream serialization: the kernel's set-up (shared memory, barriers, tensor memory) runs under the tail of the split pass
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(C::THREADS);
    cfg.dynamicSmemBytes = C::SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const unsigned char *l = (const unsigned char *)links16, *v = (const unsigned char *)vec16, *z = (const unsigned char *)zeros;
    float4 *o = (float4 *)out;
    if (mask == 0x1FFu)      MRHS_CUDA(cudaLaunchKernelEx(&cfg, coarse_h16_kernel<NB, N, 0x1FFu>, sites, mask, l, site_scale, v, z, colmax, blocks_done, o));
    else if (mask == 0x1FEu) MRHS_CUDA(cudaLaunchKernelEx(&cfg, coarse_h16_kernel<NB, N, 0x1FEu>, sites, mask, l, site_scale, v, z, colmax, blocks_done, o));
    else                     MRHS_CUDA(cudaLaunchKernelEx(&cfg, coarse_h16_kernel<NB, N, 0u>, sites, mask, l, site_scale, v, z, colmax, blocks_done, o));
    return MRHS_OK;
}

#define MRHS_H16_N_LIST(F, NB) F(NB, 2) F(NB, 4) F(NB, 8) F(NB, 12) F(NB, 16) F(NB, 24) F(NB, 32) F(NB, 48) F(NB, 64) F(NB, 96)

}  // namespace

bool coarse_h16_supported(int nb, int nrhs) {
#define MRHS_CASE(NB, NN) if (nb == NB && nrhs == NN) return true;
    MRHS_H16_N_LIST(MRHS_CASE, 24)
    MRHS_H16_N_LIST(MRHS_CASE, 40)
#undef MRHS_CASE
    return false;
}

// the split image of a full-lattice vector, followed by one K chunk of zeros (the caller clears the buffer once)
static size_t h16_image_bytes(const CoarseGeom &g) {
    const int nt = (2 * g.N + 15) / 16 * 16;
    return (size_t)g.nsites * (g.nb / 8) * 2 * nt * 16;
}
size_t coarse_h16_vec_bytes(const CoarseGeom &g) {
    const int nt = (2 * g.N + 15) / 16 * 16;
    return h16_image_bytes(g) + (size_t)2 * nt * 16;
}

mrhs_status_t coarse_h16_prepare(const CoarseGeom &g, int *grid) {
    int dev = 0, sms = 0;
    MRHS_CUDA(cudaGetDevice(&dev));
    MRHS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    mrhs_status_t s = MRHS_ERR_UNSUPPORTED;
#define MRHS_CASE(NB, NN) if (g.nb == NB && g.N == NN) s = h16_prepare_t<NB, NN>();
    MRHS_H16_N_LIST(MRHS_CASE, 24)
    MRHS_H16_N_LIST(MRHS_CASE, 40)
#undef MRHS_CASE
    if (s == MRHS_ERR_UNSUPPORTED) set_error("coarse apply: no fp16-split tensor-core specialisation for nbasis=%d nrhs=%d", g.nb, g.N);
    if (s != MRHS_OK) return s;
    *grid = (int)((long long)sms < g.nsites ? sms : g.nsites);     // one persistent block per SM (it owns all of the SM's tensor memory)
    return MRHS_OK;
}

mrhs_status_t pack_coarse_links_h16(const CoarseGeom &g, const float2 *d_canonical, void *d_links16, float *d_site_scale, cudaStream_t st) {
    const int per_site = 9 * g.nb * g.nb;
    h16_site_max_kernel<<<(unsigned)g.nsites, 256, 0, st>>>(d_canonical, per_site, d_site_scale);
    MRHS_CUDA(cudaGetLastError());
    const long long total = g.nsites * 9 * (g.nb / 8) * 2 * g.nb;
    h16_pack_links_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(g.nb, d_canonical, (uint4 *)d_links16, d_site_scale, total);
    MRHS_CUDA(cudaGetLastError());
    h16_site_scale_kernel<<<(unsigned)((g.nsites + 255) / 256), 256, 0, st>>>(d_site_scale, g.nsites);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

mrhs_status_t launch_coarse_h16(const CoarseGeom &g, const CoarseSites &sites, int grid, unsigned mask, const void *d_links16, const float *d_site_scale,
                                const void *d_in, void *d_vec16, float *d_colmax, void *d_out, cudaStream_t st) {
    const int np = g.N / 2, nt = (2 * g.N + 15) / 16 * 16;
    const long long nin = sites.cb ? g.nsites / 2 : g.nsites;      // sites of the input vector
    const long long total = nin * g.nb * np;
    // d_colmax (128 floats + the block counter behind them) is zero: cleared at create and by the stencil kernel of every apply
    {
        // a multiple of 3 blocks of 256 threads: the thread count is a multiple of every supported N_rhs / 2
        long long blocks = (total + 255) / 256;
        if (blocks > 3 * 148 * 2) blocks = 3 * 148 * 2;
        blocks = (blocks + 2) / 3 * 3;
        h16_colmax_kernel<<<(unsigned)blocks, 256, 0, st>>>((const float4 *)d_in, total, np, d_colmax);
        MRHS_CUDA(cudaGetLastError());
    }
    {
        const long long items = nin * (g.nb / 8) * (nt / 4);
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)((items + 255) / 256));
        cfg.blockDim = dim3(256);
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        MRHS_CUDA(cudaLaunchKernelEx(&cfg, h16_split_vec_kernel, (const float4 *)d_in, nin, g.nb, np, nt, (const float *)d_colmax, (uint4 *)d_vec16));
    }
    const void *zeros = (const unsigned char *)d_vec16 + h16_image_bytes(g);
#define MRHS_CASE(NB, NN) if (g.nb == NB && g.N == NN) return h16_launch_t<NB, NN>(sites, grid, mask, d_links16, d_site_scale, d_vec16, zeros, d_colmax, reinterpret_cast<unsigned *>(d_colmax + 128), d_out, st);
    MRHS_H16_N_LIST(MRHS_CASE, 24)
    MRHS_H16_N_LIST(MRHS_CASE, 40)
#undef MRHS_CASE
    set_error("coarse apply: no fp16-split tensor-core specialisation for nbasis=%d nrhs=%d", g.nb, g.N);
    return MRHS_ERR_UNSUPPORTED;
}

}  // namespace mrhs

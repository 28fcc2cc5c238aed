// coarse_tc.cu -- coarse-level 9-point stencil, tensor-core variant:
//   out_i(x) = sum_{p=0..8} sum_j A_p(x)_ij v_j(x + delta_p)          (reading S8)
// evaluated on the 5th-generation tensor cores (tcgen05.mma kind::tf32, accumulator in TMEM)
// with split-precision operands so that the fp32 tolerance of north_star holds (reading S15):
//   a = a_hi + a_lo,  a_hi = tf32(a), a_lo = tf32(a - a_hi);   a*b ~ a_hi*b_hi + a_hi*b_lo + a_lo*b_hi
// (three MMAs per K step, fp32 accumulation; the dropped a_lo*b_lo term is ~2^-22 relative).
//
// Per coarse site the complex contraction is written as ONE real GEMM accumulated over the nine
// stencil points and the nb columns:
//   D[128 x NT] += Aop[128 x nb] * Bop[nb x NT]
//   Aop rows 0..nb-1      = Re A_p,   rows nb..2nb-1   = Im A_p            (rows 2nb..127: whatever follows in shared memory; their D lanes are never read)
//   Bop cols 0..N-1       = Re v,     cols N..2N-1     = Im v              (NT = 2N rounded up to 16; inside each half the
//                                                                        even RHS come first, then the odd ones)
// so D holds Re A Re v, Re A Im v, Im A Re v, Im A Im v and the epilogue forms
//   Re out = D[i][n] - D[nb+i][N+n],   Im out = D[i][N+n] + D[nb+i][n].
// Every matrix entry read from HBM serves all N_rhs columns (PAPER.md:23 (i)).
//
// Data path: fp32 links and vectors go global -> registers (coalesced 128-bit loads) -> hi/lo split
// -> shared memory in the no-swizzle K-major core-matrix layout tcgen05.mma reads (8 rows x 16 bytes
// per core matrix, 16-byte K chunks LBO apart).  One elected thread issues the MMAs; completion comes
// back on an mbarrier via tcgen05.commit.  Several CTAs share an SM, so one CTA's operand conversion
// overlaps another's MMAs.
#include "coarse.cuh"
#include "tcgen05.cuh"
#include <cstdlib>

namespace mrhs {

namespace {

// 16 consecutive fp32 columns of this thread's TMEM lane
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 16; i++) v[i] = __uint_as_float(r[i]);
}

// round-to-nearest tf32 (low 13 mantissa bits cleared) and the remainder, itself rounded to tf32
__device__ __forceinline__ void split_tf32(float x, float &hi, float &lo) {
    uint32_t h;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(h) : "f"(x));
    hi = __uint_as_float(h);
    uint32_t l;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(l) : "f"(x - hi));
    lo = __uint_as_float(l);
}
__device__ __forceinline__ void split4(float4 x, float4 &hi, float4 &lo) {
    split_tf32(x.x, hi.x, lo.x);
    split_tf32(x.y, hi.y, lo.y);
    split_tf32(x.z, hi.z, lo.z);
    split_tf32(x.w, hi.w, lo.w);
}

template <int NB, int N>
struct TcCfg {
    static_assert(N % 2 == 0, "the tensor-core variant uses the RHS-pair element layout (even N_rhs)");
    static_assert(NB % 8 == 0 && NB <= 64, "nbasis must be a multiple of the MMA K (8) and fit 64 rows");
    static constexpr int NP = N / 2;                          // float4 elements per component
    static constexpr int NT = ((2 * N + 15) / 16) * 16;       // MMA N: Re and Im columns of every RHS
    static constexpr int KC = NB / 4;                         // 16-byte K chunks per stencil point
    static constexpr int KS = NB / 8;                         // MMA K steps per stencil point
    static constexpr int THREADS = NT <= 64 ? 128 : 256;
    static constexpr int A_LBO = 2 * NB * 16;                 // bytes between K chunks of the A operand: only the 2 nb used rows are stored
    // Stacked B operand (2 NT <= 256 columns): the hi and lo parts of the vectors are the columns 0..NT-1 and NT..2NT-1 of ONE operand,
    // so A_hi x [B_hi | B_lo] is one MMA of 2 NT columns and A_lo x B_hi a second one of NT columns on the same buffer: two
    // instructions per K step instead of three (an MMA of this size costs a fixed ~77 cycles + ~0.6 per column);
    // hi*hi and lo*hi land in accumulator columns 0..NT-1, hi*lo in NT..2NT-1, summed in the epilogue.
    // Used where it measured faster (6^3x32: nb = 40, N = 12: 0.270 -> 0.252 ms): the doubled accumulator must not cost resident blocks
    // (N = 24: 128 instead of 64 TMEM columns, N = 48: 256 instead of 128: 0.31 -> 0.52 and 0.43 -> 0.60 ms), and with the three K steps
    // of nb = 24 there is nothing to gain (0.109 -> 0.113 ms).
    static constexpr bool STK = NT <= 32 && NB >= 40;
    static constexpr int B_ROWS = STK ? 2 * NT : NT;          // rows of one K chunk of the B operand
    static constexpr int D_COLS = STK ? 2 * NT : NT;          // accumulator columns
    static constexpr int B_LBO = B_ROWS * 16 + 16;                 // + 16: consecutive K chunks of the B operand start in different banks (operand stores of one warp span several chunks)
    static constexpr int A_BYTES = KC * A_LBO;                // one of hi / lo
    static constexpr int B_BYTES = KC * B_LBO;                // stacked: hi and lo together; else one of hi / lo
    static constexpr int OPER_BYTES = 2 * A_BYTES + (STK ? 1 : 2) * B_BYTES;
    static constexpr int S_PITCH = 128 + (32 + NP - 1) / NP;  // epilogue scratch S[col][lane], floats; the combine reads NP columns x 32 / NP lanes per warp: distinct banks
    static constexpr int S_BYTES = NT * S_PITCH * 4;
    static constexpr int DATA_BYTES = OPER_BYTES > S_BYTES ? OPER_BYTES : S_BYTES;
    static constexpr int SMEM_BYTES = DATA_BYTES + 32;        // + mbarrier + TMEM address slot
    static constexpr int TMEM_COLS = pow2_cols(D_COLS);
    static constexpr int A_UNITS = 2 * KC * NB;               // 16-byte units of one link matrix
    static constexpr int B_UNITS = KC * NP;                   // (K chunk, RHS pair) work items of one vector
    static_assert(NT <= 256, "MMA N limit");
};

// links: native tensor-core layout [site][p][part Re/Im][K chunk][row][4 columns] fp32 (pack_coarse_links_tc)
// in/out: coarse vectors [site][component][RHS pair] float4 = (re0 re1 im0 im1), as in the FMA variant
// ALL: the nine-point operator (mask ignored; compile-time stage count)
template <int NB, int N, bool ALL>
__global__ void __launch_bounds__(TcCfg<NB, N>::THREADS)
coarse_tc_kernel(const CoarseSites sites, unsigned mask, const float4 *__restrict__ links,
                 const float4 *__restrict__ in, float4 *__restrict__ out) {
    typedef TcCfg<NB, N> C;
    constexpr int A_IT = (C::A_UNITS + C::THREADS - 1) / C::THREADS;
    constexpr int B_IT = (C::B_UNITS + C::THREADS - 1) / C::THREADS;
    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char *a_hi = smem, *a_lo = smem + C::A_BYTES;
    unsigned char *b_hi = smem + 2 * C::A_BYTES, *b_lo = b_hi + (C::STK ? C::NT * 16 : C::B_BYTES);     // stacked: the lo rows follow the hi rows inside every K chunk
    float *S = reinterpret_cast<float *>(smem);
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem + C::DATA_BYTES);
    uint32_t *tslot = reinterpret_cast<uint32_t *>(smem + C::DATA_BYTES + 8);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    // one-time setup: barrier, zeroed operand area (so that the unused MMA rows / columns never see NaN patterns), TMEM accumulator
    if (tid == 0) {
        mbar_init(bar, 1);
        mbar_fence_init();
    }
    for (int i = tid; i < C::OPER_BYTES / 16; i += C::THREADS) reinterpret_cast<float4 *>(smem)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (warp == 0) tmem_alloc<C::TMEM_COLS>(tslot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tslot;
    constexpr uint32_t idesc = instr_desc_tf32(128, C::NT), idesc2 = instr_desc_tf32(128, 2 * C::NT);

    uint32_t nstage = 0;   // operand stages handed to the tensor core so far (same in every thread)
    // raw fp32 operands of one stage (stencil point p of a site) in registers; loaded one stage ahead, right after
    // the previous stage has been handed to the tensor core, so the load latency overlaps its MMAs and the next wait
    float4 ra[A_IT];
    float4 rb[B_IT][4];
    const long long nsites = sites.nout;       // output sites, enumerated by osite; the links of output site osite live at its lex
    // vector index of the neighbour at stencil point p: 0 self, 1..4 = +x..+t, 5..8 = -x..-t (periodic)
    auto neighbour = [&](const CoarseSite32 &c, int p) -> long long {
        const int n = coarse_neighbour32(sites, c, p);
        return sites.cb ? n >> 1 : n;
    };
    // one thread asks the copy engine to bring a later stage's matrix and neighbour vector into L2 (each is one
    // contiguous block), so that the register loads of that stage find them there
    auto prefetch_stage = [&](const CoarseSite32 &c, int p) {
        bulk_prefetch_l2(links + ((size_t)c.lex * 9 + p) * C::A_UNITS, C::A_UNITS * 16);
        bulk_prefetch_l2(in + (size_t)neighbour(c, p) * NB * C::NP, NB * C::NP * 16);
    };
    auto load_stage = [&](const CoarseSite32 &c, int p) {
        const float4 *lp = links + ((size_t)c.lex * 9 + p) * C::A_UNITS;
        const float4 *vp = in + (size_t)neighbour(c, p) * NB * C::NP;
#pragma unroll
        for (int it = 0; it < A_IT; it++) {
            const int u = tid + it * C::THREADS;
            if (u < C::A_UNITS) ra[it] = __ldg(lp + u);
        }
#pragma unroll
        for (int it = 0; it < B_IT; it++) {
            const int w = tid + it * C::THREADS;
            if (w < C::B_UNITS) {
                const int kc = w / C::NP, q = w - kc * C::NP;
#pragma unroll
                for (int e = 0; e < 4; e++) rb[it][e] = __ldg(vp + (size_t)(4 * kc + e) * C::NP + q);
            }
        }
    };
    // For wide operands (two blocks per SM) the load runs one stage ahead; for narrow ones the extra live registers
    // would cost resident blocks, which hide the latency better, so the load sits at the top of its own stage.
    constexpr bool AHEAD = C::NT > 96;
    constexpr int kPfAhead = AHEAD ? 3 : 2;
    // the stencil points of this apply: bit p of mask; stage s of a site handles the s-th set bit
    const int npts = ALL ? 9 : __popc(mask);
    const unsigned long long plist = ALL ? 0ull : coarse_point_list(mask);
    auto point = [&](int s) { return ALL ? s : coarse_point(plist, s); };
    // site coordinates once per site (this site and the block's next one), neighbours from them without divisions
    CoarseSite32 cur = coarse_site32(sites, blockIdx.x), nxt = cur;
    if (AHEAD && (long long)blockIdx.x < nsites) load_stage(cur, point(0));
    for (long long site = blockIdx.x; site < nsites; site += gridDim.x) {
        if (site + gridDim.x < nsites) nxt = coarse_site32(sites, site + gridDim.x);
        for (int sp = 0; sp < npts; sp++) {
            const int p = point(sp);
            if (!AHEAD) load_stage(cur, p);
            // the single operand buffer is free once the previous stage's MMAs have completed
            if (nstage > 0) mbar_wait(bar, (nstage - 1) & 1);
#pragma unroll
            for (int it = 0; it < A_IT; it++) {
                const int u = tid + it * C::THREADS;
                if (u < C::A_UNITS) {
                    const int part = u / (C::KC * NB), r = u - part * (C::KC * NB);
                    const int kc = r / NB, row = r - kc * NB;
                    float4 hi, lo;
                    split4(ra[it], hi, lo);
                    const int off = kc * C::A_LBO + (part * NB + row) * 16;
                    *reinterpret_cast<float4 *>(a_hi + off) = hi;
                    *reinterpret_cast<float4 *>(a_lo + off) = lo;
                }
            }
#pragma unroll
            for (int it = 0; it < B_IT; it++) {
                const int w = tid + it * C::THREADS;
                if (w < C::B_UNITS) {
                    const int kc = w / C::NP, q = w - kc * C::NP;
                    const float4 x0 = rb[it][0], x1 = rb[it][1], x2 = rb[it][2], x3 = rb[it][3];
                    float4 hi, lo;
                    const int base = kc * C::B_LBO;
                    split4(make_float4(x0.x, x1.x, x2.x, x3.x), hi, lo);        // Re, RHS 2q
                    *reinterpret_cast<float4 *>(b_hi + base + (q) * 16) = hi;
                    *reinterpret_cast<float4 *>(b_lo + base + (q) * 16) = lo;
                    split4(make_float4(x0.y, x1.y, x2.y, x3.y), hi, lo);        // Re, RHS 2q+1
                    *reinterpret_cast<float4 *>(b_hi + base + (C::NP + q) * 16) = hi;
                    *reinterpret_cast<float4 *>(b_lo + base + (C::NP + q) * 16) = lo;
                    split4(make_float4(x0.z, x1.z, x2.z, x3.z), hi, lo);        // Im, RHS 2q
                    *reinterpret_cast<float4 *>(b_hi + base + (N + q) * 16) = hi;
                    *reinterpret_cast<float4 *>(b_lo + base + (N + q) * 16) = lo;
                    split4(make_float4(x0.w, x1.w, x2.w, x3.w), hi, lo);        // Im, RHS 2q+1
                    *reinterpret_cast<float4 *>(b_hi + base + (N + C::NP + q) * 16) = hi;
                    *reinterpret_cast<float4 *>(b_lo + base + (N + C::NP + q) * 16) = lo;
                }
            }
            fence_async_smem();
            __syncthreads();
            if (tid == 0) {
                tc_fence_after();
                const uint32_t ah = smem_u32(a_hi), al = smem_u32(a_lo), bh = smem_u32(b_hi), bl = smem_u32(b_lo);
#pragma unroll
                for (int ks = 0; ks < C::KS; ks++) {
                    const uint64_t dah = smem_desc(ah + ks * 2 * C::A_LBO, C::A_LBO, 128);
                    const uint64_t dal = smem_desc(al + ks * 2 * C::A_LBO, C::A_LBO, 128);
                    const uint64_t dbh = smem_desc(bh + ks * 2 * C::B_LBO, C::B_LBO, 128);
                    const uint64_t dbl = smem_desc(bl + ks * 2 * C::B_LBO, C::B_LBO, 128);
                    if (C::STK) {
                        mma_tf32(tmem, dah, dbh, idesc2, (sp | ks) != 0);     // hi x [hi | lo]
                        mma_tf32(tmem, dal, dbh, idesc, 1);                    // lo x hi
                    } else {
                        mma_tf32(tmem, dal, dbh, idesc, (sp | ks) != 0);
                        mma_tf32(tmem, dah, dbl, idesc, 1);
                        mma_tf32(tmem, dah, dbh, idesc, 1);
                    }
                }
                mma_commit(bar);
                // L2 prefetch kPfAhead stages ahead (possibly into the next site of this block)
                int sp2 = sp + kPfAhead;
                long long site2 = site;
                while (sp2 >= npts) { sp2 -= npts; site2 += gridDim.x; }
                if (site2 == site) prefetch_stage(cur, point(sp2));
                else if (site2 == site + gridDim.x && site2 < nsites) prefetch_stage(nxt, point(sp2));
            }
            nstage++;
            if (AHEAD) {
                if (sp + 1 < npts) load_stage(cur, point(sp + 1));
                else if (site + gridDim.x < nsites) load_stage(nxt, point(0));
            }
        }
        // all nine points accumulated: TMEM -> shared scratch S[col][lane] -> combine -> global
        mbar_wait(bar, (nstage - 1) & 1);
        tc_fence_after();
        {
            const int quarter = warp & 3;
            for (int ch = warp >> 2; ch < C::NT / 16; ch += C::THREADS / 128) {
                float v[16];
                tmem_ld16(tmem + ((uint32_t)(quarter * 32) << 16) + ch * 16, v);
                if (C::STK) {       // the hi*lo part sits NT columns further
                    float w[16];
                    tmem_ld16(tmem + ((uint32_t)(quarter * 32) << 16) + C::NT + ch * 16, w);
#pragma unroll
                    for (int k = 0; k < 16; k++) v[k] += w[k];
                }
#pragma unroll
                for (int k = 0; k < 16; k++) S[(ch * 16 + k) * C::S_PITCH + quarter * 32 + lane] = v[k];
            }
        }
        tc_fence_before();
        __syncthreads();
        for (int idx = tid; idx < NB * C::NP; idx += C::THREADS) {
            const int i = idx / C::NP, q = idx - i * C::NP;
            const int n0 = q, n1 = C::NP + q;   // column order of D: Re even RHS | Re odd RHS | Im even | Im odd (conflict-free operand stores)
            auto d = [&](int col, int row) { return S[col * C::S_PITCH + row]; };
            float4 o;
            o.x = d(n0, i) - d(N + n0, NB + i);
            o.y = d(n1, i) - d(N + n1, NB + i);
            o.z = d(N + n0, i) + d(n0, NB + i);
            o.w = d(N + n1, i) + d(n1, NB + i);
            out[((size_t)site * NB + i) * C::NP + q] = o;
        }
        __syncthreads();   // S (aliasing the operand buffer) is free for the next site
        cur = nxt;
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_free<C::TMEM_COLS>(tmem);
}

// canonical A[site][p][row][col] complex -> [site][p][part][K chunk][row][4 columns] fp32; one thread per float
__global__ void pack_links_tc_kernel(int nb, const float2 *__restrict__ src, float *__restrict__ dst, long long total) {
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int kcn = nb / 4;
    int e = (int)(idx & 3);
    long long q = idx >> 2;
    int row = (int)(q % nb); q /= nb;
    int kc = (int)(q % kcn); q /= kcn;
    int part = (int)(q & 1);
    long long mat = q >> 1;
    float2 a = src[(mat * nb + row) * nb + 4 * kc + e];
    dst[idx] = part ? a.y : a.x;
}

template <int NB, int N>
mrhs_status_t tc_prepare_t(int *ctas_per_sm) {
    typedef TcCfg<NB, N> C;
    MRHS_CUDA(cudaFuncSetAttribute(coarse_tc_kernel<NB, N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
    MRHS_CUDA(cudaFuncSetAttribute(coarse_tc_kernel<NB, N, true>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    MRHS_CUDA(cudaFuncSetAttribute(coarse_tc_kernel<NB, N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
    MRHS_CUDA(cudaFuncSetAttribute(coarse_tc_kernel<NB, N, false>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    // Resident CTAs per SM from the resources themselves (the occupancy API reports 1 for a kernel that
    // allocates tensor memory): shared memory (+1 KB reserved per CTA), registers, threads, TMEM columns.
    cudaFuncAttributes fa;
    MRHS_CUDA(cudaFuncGetAttributes(&fa, coarse_tc_kernel<NB, N, false>));
    int dev = 0, smem_sm = 0, regs_sm = 0;
    MRHS_CUDA(cudaGetDevice(&dev));
    MRHS_CUDA(cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev));
    MRHS_CUDA(cudaDeviceGetAttribute(&regs_sm, cudaDevAttrMaxRegistersPerMultiprocessor, dev));
    int occ = smem_sm / (C::SMEM_BYTES + (int)fa.sharedSizeBytes + 1024);
    const int regs_cta = ((fa.numRegs + 7) / 8 * 8) * C::THREADS;
    if (regs_cta > 0 && occ > regs_sm / regs_cta) occ = regs_sm / regs_cta;
    if (occ > 2048 / C::THREADS) occ = 2048 / C::THREADS;
    if (occ > 512 / C::TMEM_COLS) occ = 512 / C::TMEM_COLS;
    if (occ > 8) occ = 8;
    if (occ < 1) { set_error("coarse tensor-core kernel does not fit an SM (nbasis=%d nrhs=%d)", NB, N); return MRHS_ERR_UNSUPPORTED; }
    *ctas_per_sm = occ;
    return MRHS_OK;
}
template <int NB, int N>
mrhs_status_t tc_launch_t(const CoarseSites &sites, int grid, unsigned mask, const float *links, const void *in, void *out, cudaStream_t st) {
    typedef TcCfg<NB, N> C;
    if ((long long)grid > sites.nout) grid = (int)sites.nout;
    if (mask == 0x1FFu)
        coarse_tc_kernel<NB, N, true><<<grid, C::THREADS, C::SMEM_BYTES, st>>>(sites, mask, (const float4 *)links, (const float4 *)in, (float4 *)out);
    else
        coarse_tc_kernel<NB, N, false><<<grid, C::THREADS, C::SMEM_BYTES, st>>>(sites, mask, (const float4 *)links, (const float4 *)in, (float4 *)out);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

#define MRHS_TC_N_LIST(F, NB) F(NB, 2) F(NB, 4) F(NB, 8) F(NB, 12) F(NB, 16) F(NB, 24) F(NB, 32) F(NB, 48) F(NB, 64) F(NB, 96)

}  // namespace

bool coarse_tc_supported(int nb, int nrhs) {
#define MRHS_CASE(NB, NN) if (nb == NB && nrhs == NN) return true;
    MRHS_TC_N_LIST(MRHS_CASE, 24)
    MRHS_TC_N_LIST(MRHS_CASE, 40)
#undef MRHS_CASE
    return false;
}

mrhs_status_t coarse_tc_prepare(const CoarseGeom &g, int *grid) {
    int dev = 0, sms = 0, per_sm = 0;
    MRHS_CUDA(cudaGetDevice(&dev));
    MRHS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    mrhs_status_t s = MRHS_ERR_UNSUPPORTED;
#define MRHS_CASE(NB, NN) if (g.nb == NB && g.N == NN) s = tc_prepare_t<NB, NN>(&per_sm);
    MRHS_TC_N_LIST(MRHS_CASE, 24)
    MRHS_TC_N_LIST(MRHS_CASE, 40)
#undef MRHS_CASE
    if (s != MRHS_OK) {
        if (per_sm == 0 && !coarse_tc_supported(g.nb, g.N))
            set_error("coarse apply: no tensor-core specialisation for nbasis=%d nrhs=%d", g.nb, g.N);
        return s;
    }
    long long want = (long long)per_sm * sms;
    *grid = (int)(want < g.nsites ? want : g.nsites);
    if (getenv("MRHS_DEBUG")) fprintf(stderr, "[mrhs] coarse tensor-core kernel nb=%d N=%d: %d CTAs/SM x %d SMs, grid %d\n", g.nb, g.N, per_sm, sms, *grid);
    return MRHS_OK;
}

mrhs_status_t launch_coarse_tc(const CoarseGeom &g, const CoarseSites &sites, int grid, unsigned mask, const float *d_links, const void *d_in, void *d_out, cudaStream_t st) {
#define MRHS_CASE(NB, NN) if (g.nb == NB && g.N == NN) return tc_launch_t<NB, NN>(sites, grid, mask, d_links, d_in, d_out, st);
    MRHS_TC_N_LIST(MRHS_CASE, 24)
    MRHS_TC_N_LIST(MRHS_CASE, 40)
#undef MRHS_CASE
    set_error("coarse apply: no tensor-core specialisation for nbasis=%d nrhs=%d", g.nb, g.N);
    return MRHS_ERR_UNSUPPORTED;
}

mrhs_status_t pack_coarse_links_tc(const CoarseGeom &g, const float2 *d_canonical, float *d_native, cudaStream_t st) {
    long long total = g.nsites * 9 * g.nb * g.nb * 2;
    long long blocks = (total + 255) / 256;
    pack_links_tc_kernel<<<(unsigned)blocks, 256, 0, st>>>(g.nb, d_canonical, d_native, total);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

}  // namespace mrhs

// coarse.cu -- coarse-level 9-point stencil, FP32-FMA variant:
//   out_i(x) = sum_{p=0..8} sum_j A_p(x)_ij v_j(x + delta_p)          (reading S8)
// with nine independent dense nb x nb complex matrices per site, applied to N_rhs vectors at
// once: each matrix entry fetched from HBM serves every RHS (PAPER.md:23 (i)).
//
// One thread block per coarse site.  The nine (A_p, v(x+delta_p)) pairs are streamed through a
// ring of shared-memory stages with bulk async copies (one contiguous copy per matrix and per
// neighbour vector) signalled on mbarriers.  A thread owns a TI x TP register tile of (rows, RHS
// pairs) and, for small N_rhs, one of KS slices of the column range; slices are summed through
// shared memory at the end.
#include "async_copy.cuh"
#include "coarse.cuh"
#include "layout.cuh"

namespace mrhs {

namespace {

template <int R> __device__ __forceinline__ CVec<R> czero_c();
template <> __device__ __forceinline__ CVec<1> czero_c<1>() { return {{0.f}, {0.f}}; }
template <> __device__ __forceinline__ CVec<2> czero_c<2>() { return {{0ull}, {0ull}}; }

constexpr int largest_ks(int nb, int groups) {
    int best = 1;
    for (int k = 1; k <= nb; k++)
        if (nb % k == 0 && groups * k <= 256) best = k;
    return best;
}

// Register tile of (rows, RHS lanes) per thread, chosen from measurements at nbasis 24 / 40: up to
// N_rhs = 16 the small 2 x 1 tile with many column slices keeps more warps busy per site (few lanes to spread over
// threads; 4 x 1, 2 x 2, 4 x 2, 2 x 3, 4 x 3 and 8-row tiles all measured slower there); at N_rhs = 24 a 4 x 1 tile (10 % faster
// at nbasis 24 and 40); from N_rhs = 32 the 4-row tile with 2 or 3 lanes (per column 2 + TP shared-memory loads of 16 bytes feed
// 16 TP FFMA2) relieves the shared-memory pipe, as long as the block keeps at least six warps.
constexpr int pick_ti(int nb, int np, int r) { return np * r >= 24 || nb * np / 2 > 256 ? 4 : 2; }
constexpr int pick_tp(int nb, int np, int r) {
    if (np * r < 32) return (nb * np / 2 > 256 && np % 2 == 0) ? 2 : 1;
    return (np % 3 == 0 && nb / 4 * (np / 3) >= 192) ? 3 : 2;
}

template <int NB, int N>
struct CoarseCfg {
    static constexpr int R = (N % 2 == 0) ? 2 : 1;
    static constexpr int NP = N / R;                       // RHS lanes (elements) per component
    static constexpr int TI = pick_ti(NB, NP, R);
    static constexpr int TP = pick_tp(NB, NP, R);
    static constexpr int NPG = NP / TP;                    // lane groups
    static constexpr int NRG = NB / TI;                    // row groups
    static constexpr int GROUPS = NPG * NRG;
    static constexpr int KS = largest_ks(NB, GROUPS);
    static constexpr int THREADS = GROUPS * KS;
    static constexpr int JS = NB / KS;                     // columns per slice
    static constexpr int A_BYTES = NB * NB * 8;
    static constexpr int V_BYTES = NB * N * 8;
    static constexpr int STAGE_BYTES = A_BYTES + V_BYTES;
    static constexpr int NSTAGE = STAGE_BYTES < 24 * 1024 ? 4 : 3;
    static constexpr int RED_BYTES = (KS > 1 ? KS : 0) * GROUPS * TI * TP * R * 8;
    static constexpr int DATA_BYTES = NSTAGE * STAGE_BYTES > RED_BYTES ? NSTAGE * STAGE_BYTES : RED_BYTES;
    static constexpr int SMEM_BYTES = DATA_BYTES + 64;     // + mbarriers
    static_assert(NB % TI == 0 && NP % TP == 0, "tile must divide the site");
    static_assert(GROUPS <= 256 && THREADS <= 256, "too many work items for one block");
    static_assert(A_BYTES % 16 == 0 && V_BYTES % 16 == 0, "bulk copies need 16-byte multiples");
};

// ALL: the nine-point operator (mask ignored; the stage loop has a compile-time trip count)
template <int NB, int N, bool ALL>
__global__ void __launch_bounds__(CoarseCfg<NB, N>::THREADS)
coarse_fma_kernel(const CoarseSites sites, unsigned mask, const float2 *__restrict__ links,
                  const typename Elem<CoarseCfg<NB, N>::R>::type *__restrict__ in,
                  typename Elem<CoarseCfg<NB, N>::R>::type *__restrict__ out) {
    typedef CoarseCfg<NB, N> C;
    constexpr int R = C::R, TI = C::TI, TP = C::TP;
    typedef typename Elem<R>::type E;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + C::DATA_BYTES);

    const int tid = threadIdx.x;
    const int pg = tid % C::NPG;
    const int rg = (tid / C::NPG) % C::NRG;
    const int ks = tid / C::GROUPS;

    const long long osite = blockIdx.x;                       // output site; its links live at lex
    const CoarseSite32 sc = coarse_site32(sites, osite);
    const long long site = sc.lex;
    // vector index of the neighbour at stencil point p: 0 self, 1..4 = +x..+t, 5..8 = -x..-t
    auto neighbour = [&](int p) -> long long {
        const int n = coarse_neighbour32(sites, sc, p);
        return sites.cb ? n >> 1 : n;
    };
    // the stencil points of this apply: bit p of mask (all nine for the full operator, bit 0 = self term alone,
    // bits 1..8 = the 8-point hopping term); stage s handles the s-th set bit
    const int npts = ALL ? 9 : __popc(mask);
    const unsigned long long plist = ALL ? 0ull : coarse_point_list(mask);
    auto issue = [&](int s) {
        const int p = ALL ? s : coarse_point(plist, s);
        const int slot = s % C::NSTAGE;
        unsigned char *dst = smem + (size_t)slot * C::STAGE_BYTES;
        mbar_expect_tx(&full[slot], C::STAGE_BYTES);
        bulk_g2s(dst, links + ((size_t)site * 9 + p) * NB * NB, C::A_BYTES, &full[slot]);
        bulk_g2s(dst + C::A_BYTES, in + (size_t)neighbour(p) * NB * C::NP, C::V_BYTES, &full[slot]);
    };

    if (tid == 0) {
        for (int s = 0; s < C::NSTAGE; s++) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0)
        for (int s = 0; s < C::NSTAGE && s < npts; s++) issue(s);

    CVec<R> acc[TI][TP];
#pragma unroll
    for (int a = 0; a < TI; a++)
#pragma unroll
        for (int b = 0; b < TP; b++) acc[a][b] = czero_c<R>();

    for (int p = 0; p < npts; p++) {
        const int slot = p % C::NSTAGE;
        mbar_wait(&full[slot], (p / C::NSTAGE) & 1);
        const float2 *As = reinterpret_cast<const float2 *>(smem + (size_t)slot * C::STAGE_BYTES);   // [col][row]
        const E *vs = reinterpret_cast<const E *>(smem + (size_t)slot * C::STAGE_BYTES + C::A_BYTES);  // [col][lane]
        const float2 *ap = As + (size_t)(ks * C::JS) * NB + rg * TI;
        const E *vp = vs + (size_t)(ks * C::JS) * C::NP + pg * TP;
#pragma unroll 4
        for (int j = 0; j < C::JS; j++) {
            float2 a[TI];
#pragma unroll
            for (int i = 0; i < TI; i += 2) {
                float4 t = *reinterpret_cast<const float4 *>(ap + j * NB + i);
                a[i] = make_float2(t.x, t.y);
                a[i + 1] = make_float2(t.z, t.w);
            }
            CVec<R> v[TP];
#pragma unroll
            for (int b = 0; b < TP; b++) v[b] = to_cvec(vp[j * C::NP + b]);
#pragma unroll
            for (int i = 0; i < TI; i++)
#pragma unroll
                for (int b = 0; b < TP; b++) acc[i][b] = cfma(a[i].x, a[i].y, v[b], acc[i][b]);
        }
        __syncthreads();   // every thread is done with this slot
        if (tid == 0 && p + C::NSTAGE < npts) issue(p + C::NSTAGE);
    }

    // sum the column slices (the stage ring is free: the last __syncthreads above covers it): every slice leaves its tile in
    // shared memory as [slice][group][TI x TP], then thread e adds element e of all slices in a fixed order and stores it
    constexpr int TILE = TI * TP, ELEMS = C::GROUPS * TILE;
    if (C::KS > 1) {
        E *red = reinterpret_cast<E *>(smem);
        E *r = red + ((size_t)ks * C::GROUPS + (tid % C::GROUPS)) * TILE;
#pragma unroll
        for (int i = 0; i < TI; i++)
#pragma unroll
            for (int b = 0; b < TP; b++) r[i * TP + b] = from_cvec(acc[i][b]);
        __syncthreads();
        for (int e = tid; e < ELEMS; e += C::THREADS) {
            CVec<R> sum = to_cvec(red[e]);
            for (int k = 1; k < C::KS; k++) sum = cadd(sum, to_cvec(red[(size_t)k * ELEMS + e]));
            const int grp = e / TILE, w = e - grp * TILE, i = w / TP, b = w - i * TP;
            const int epg = grp % C::NPG, erg = grp / C::NPG;
            out[((size_t)osite * NB + erg * TI + i) * C::NP + epg * TP + b] = from_cvec(sum);
        }
    } else {
        E *o = out + ((size_t)osite * NB + rg * TI) * C::NP + pg * TP;
#pragma unroll
        for (int i = 0; i < TI; i++)
#pragma unroll
            for (int b = 0; b < TP; b++) o[(size_t)i * C::NP + b] = from_cvec(acc[i][b]);
    }
}

__global__ void pack_links_kernel(int nb, const float2 *__restrict__ src, float2 *__restrict__ dst, long long total) {
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;   // native order: [mat][col][row]
    if (idx >= total) return;
    int row = (int)(idx % nb);
    long long q = idx / nb;
    int col = (int)(q % nb);
    long long mat = q / nb;
    dst[idx] = src[(mat * nb + row) * nb + col];
}

template <int NB, int N>
mrhs_status_t launch_t(const CoarseSites &sites, unsigned mask, const float2 *links, const void *in, void *out, cudaStream_t st) {
    typedef CoarseCfg<NB, N> C;
    typedef typename Elem<C::R>::type E;
    if (mask == 0x1FFu) coarse_fma_kernel<NB, N, true><<<(unsigned)sites.nout, C::THREADS, C::SMEM_BYTES, st>>>(sites, mask, links, (const E *)in, (E *)out);
    else coarse_fma_kernel<NB, N, false><<<(unsigned)sites.nout, C::THREADS, C::SMEM_BYTES, st>>>(sites, mask, links, (const E *)in, (E *)out);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}
template <int NB, int N>
mrhs_status_t prepare_t() {
    typedef CoarseCfg<NB, N> C;
    MRHS_CUDA(cudaFuncSetAttribute(coarse_fma_kernel<NB, N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
    MRHS_CUDA(cudaFuncSetAttribute(coarse_fma_kernel<NB, N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES));
    return MRHS_OK;
}

#define MRHS_COARSE_N_LIST(F, NB) \
    F(NB, 1) F(NB, 2) F(NB, 4) F(NB, 8) F(NB, 12) F(NB, 16) F(NB, 24) F(NB, 32) F(NB, 48) F(NB, 64) F(NB, 96)

}  // namespace

bool coarse_fma_supported(int nb, int nrhs) {
#define MRHS_CASE(NB, NN) if (nb == NB && nrhs == NN) return true;
    MRHS_COARSE_N_LIST(MRHS_CASE, 24)
    MRHS_COARSE_N_LIST(MRHS_CASE, 40)
#undef MRHS_CASE
    return false;
}

mrhs_status_t coarse_fma_prepare(const CoarseGeom &g) {
#define MRHS_CASE(NB, NN) if (g.nb == NB && g.N == NN) return prepare_t<NB, NN>();
    MRHS_COARSE_N_LIST(MRHS_CASE, 24)
    MRHS_COARSE_N_LIST(MRHS_CASE, 40)
#undef MRHS_CASE
    set_error("coarse apply: no FP32-FMA specialisation for nbasis=%d nrhs=%d", g.nb, g.N);
    return MRHS_ERR_UNSUPPORTED;
}

mrhs_status_t launch_coarse_fma(const CoarseGeom &g, const CoarseSites &sites, unsigned mask, const float2 *d_links, const void *d_in, void *d_out, cudaStream_t st) {
#define MRHS_CASE(NB, NN) if (g.nb == NB && g.N == NN) return launch_t<NB, NN>(sites, mask, d_links, d_in, d_out, st);
    MRHS_COARSE_N_LIST(MRHS_CASE, 24)
    MRHS_COARSE_N_LIST(MRHS_CASE, 40)
#undef MRHS_CASE
    set_error("coarse apply: no FP32-FMA specialisation for nbasis=%d nrhs=%d", g.nb, g.N);
    return MRHS_ERR_UNSUPPORTED;
}

mrhs_status_t pack_coarse_links(const CoarseGeom &g, const float2 *d_canonical, float2 *d_native, cudaStream_t st) {
    long long total = g.nsites * 9 * g.nb * g.nb;
    long long blocks = (total + 255) / 256;
    pack_links_kernel<<<(unsigned)blocks, 256, 0, st>>>(g.nb, d_canonical, d_native, total);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

}  // namespace mrhs

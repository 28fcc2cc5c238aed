// transfer.cu -- prolongation and restriction between the fine level and the first coarse level for N_rhs
// right-hand sides at once (reading S9).  First correct version:
// FP32 FMA (FFMA2 over RHS pairs), operands through L1/L2; fields in the library's native layouts.
#include "transfer.cuh"
#include "async_copy.cuh"

#include <cooperative_groups.h>

namespace mrhs {

namespace {

constexpr int kRestrictAhead = 4;   // restriction: L2 prefetch distance in sites of a slice

template <int R> __device__ __forceinline__ CVec<R> czero_t();
template <> __device__ __forceinline__ CVec<1> czero_t<1>() { return {{0.f}, {0.f}}; }
template <> __device__ __forceinline__ CVec<2> czero_t<2>() { return {{0ull}, {0ull}}; }

__global__ void pack_basis_kernel(int nvec, long long V, const float2 *__restrict__ src, float2 *__restrict__ dst, long long total) {
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;   // native order [lex][k][12]
    if (idx >= total) return;
    const int c = (int)(idx % 12);
    long long q = idx / 12;
    const int k = (int)(q % nvec);
    const long long lex = q / nvec;
    dst[idx] = src[((long long)k * V + lex) * 12 + c];
}

// One thread = one fine site and R right-hand sides (the thread order of the fine native layout, as in M_ooee):
// the 2 nvec coarse coefficients of the site's block are read once per k and serve all twelve components.
template <int R>
__global__ void __launch_bounds__(256)
prolong_kernel(TransferGeom g, int NP, long long nthreads, const float4 *__restrict__ basis,
               const typename Elem<R>::type *__restrict__ coarse, typename Elem<R>::type *__restrict__ fine) {
    typedef typename Elem<R>::type E;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= nthreads) return;
    const int CS = g.XB * NP;
    long long b = gid / CS;
    const int rem = (int)(gid - b * CS);
    const int xin = rem / NP, pair = rem - xin * NP;
    E *po = fine + (size_t)b * 12 * CS + rem;
    const int xb = (int)(b % g.nxb); b /= g.nxb;
    const int y = (int)(b % g.Y); b /= g.Y;
    const int z = (int)(b % g.Z);
    const int t = (int)(b / g.Z);
    const int x = xb * g.XB + xin;
    const long long lex = x + (long long)g.X * (y + (long long)g.Y * (z + (long long)g.Z * t));
    const long long B = (x / g.bx) + (long long)g.cX * ((y / g.by) + (long long)g.cY * ((z / g.bz) + (long long)g.cZ * (t / g.bt)));
    const E *vc = coarse + (size_t)B * 2 * g.nvec * NP + pair;
    const float4 *ph = basis + (size_t)lex * g.nvec * 6;
    CVec<R> acc[12];
#pragma unroll
    for (int c = 0; c < 12; c++) acc[c] = czero_t<R>();
#pragma unroll 4
    for (int k = 0; k < g.nvec; k++) {
        const CVec<R> v0 = to_cvec(__ldg(vc + (size_t)k * NP)), v1 = to_cvec(__ldg(vc + (size_t)(g.nvec + k) * NP));
#pragma unroll
        for (int j = 0; j < 6; j++) {
            const float4 a = __ldg(ph + k * 6 + j);   // components 2j, 2j+1
            const CVec<R> &v = j < 3 ? v0 : v1;
            acc[2 * j] = cfma(a.x, a.y, v, acc[2 * j]);
            acc[2 * j + 1] = cfma(a.z, a.w, v, acc[2 * j + 1]);
        }
    }
#pragma unroll
    for (int c = 0; c < 12; c++) po[(size_t)c * CS] = from_cvec(acc[c]);
}

// The same map with the basis staged in shared memory: a thread block owns ROWS consecutive block rows of the fine
// native layout (XB sites each, ROWS XB NP threads); the basis of a row is one contiguous run of XB nvec 96 bytes, brought
// in by one bulk async copy per row (completion on an mbarrier), so the HBM stream of the basis has tens of KB in flight
// per SM instead of one 16-byte load per thread.  Sites read their k in a staggered order to spread shared-memory banks.
template <int R>
__global__ void __launch_bounds__(256)
prolong_smem_kernel(TransferGeom g, int NP, int rows, long long nblk, const float4 *__restrict__ basis,
                    const typename Elem<R>::type *__restrict__ coarse, typename Elem<R>::type *__restrict__ fine) {
    typedef typename Elem<R>::type E;
    extern __shared__ __align__(128) unsigned char sm[];
    __shared__ uint64_t bar;
    const float4 *sb = reinterpret_cast<const float4 *>(sm);
    const int CS = g.XB * NP;
    const int tid = threadIdx.x;
    const long long b0 = (long long)blockIdx.x * rows;
    const uint32_t row_bytes = (uint32_t)g.XB * g.nvec * 96u;
    auto row_lex0 = [&](long long b) {
        const int xb = (int)(b % g.nxb); b /= g.nxb;
        const int y = (int)(b % g.Y); b /= g.Y;
        const int z = (int)(b % g.Z);
        const int t = (int)(b / g.Z);
        return (long long)xb * g.XB + (long long)g.X * (y + (long long)g.Y * (z + (long long)g.Z * t));
    };
    if (tid == 0) {
        mbar_init(&bar, 1);
        mbar_fence_init();
        int nrow = 0;
        for (int r = 0; r < rows; r++) nrow += b0 + r < nblk;
        mbar_expect_tx(&bar, nrow * row_bytes);
        for (int r = 0; r < nrow; r++)
            bulk_g2s(sm + (size_t)r * row_bytes, basis + (size_t)row_lex0(b0 + r) * g.nvec * 6, row_bytes, &bar);
    }
    __syncthreads();
    const int row = tid / CS, rem = tid - row * CS;
    const long long b = b0 + row;
    const bool active = row < rows && b < nblk;
    const int xin = rem / NP, pair = rem - xin * NP;
    const E *vc = coarse;
    int x = 0, y = 0, z = 0, t = 0;
    if (active) {
        long long q = b;
        const int xb = (int)(q % g.nxb); q /= g.nxb;
        y = (int)(q % g.Y); q /= g.Y;
        z = (int)(q % g.Z);
        t = (int)(q / g.Z);
        x = xb * g.XB + xin;
        const long long B = (x / g.bx) + (long long)g.cX * ((y / g.by) + (long long)g.cY * ((z / g.bz) + (long long)g.cZ * (t / g.bt)));
        vc = coarse + (size_t)B * 2 * g.nvec * NP + pair;
    }
    mbar_wait(&bar, 0);      // the basis rows have landed
    if (!active) return;
    const int site = row * g.XB + xin;
    const float4 *ph = sb + (size_t)site * g.nvec * 6;
    CVec<R> acc[12];
#pragma unroll
    for (int c = 0; c < 12; c++) acc[c] = czero_t<R>();
    int k = site % g.nvec;
#pragma unroll 10
    for (int i = 0; i < g.nvec; i++) {
        const CVec<R> v0 = to_cvec(__ldg(vc + (size_t)k * NP)), v1 = to_cvec(__ldg(vc + (size_t)(g.nvec + k) * NP));
#pragma unroll
        for (int j = 0; j < 6; j++) {
            const float4 a = ph[k * 6 + j];
            const CVec<R> &v = j < 3 ? v0 : v1;
            acc[2 * j] = cfma(a.x, a.y, v, acc[2 * j]);
            acc[2 * j + 1] = cfma(a.z, a.w, v, acc[2 * j + 1]);
        }
        k = k + 1 == g.nvec ? 0 : k + 1;
    }
    E *po = fine + (size_t)b * 12 * CS + rem;
#pragma unroll
    for (int c = 0; c < 12; c++) po[(size_t)c * CS] = from_cvec(acc[c]);
}

// One thread block = one aggregate and a chunk of PC x LT RHS lanes; a thread owns one (slice, group of KT basis vectors,
// group of LT lanes) and sums its slice of the aggregate's sites into the 2 KT LT chiral coefficients: every field element
// loaded serves KT basis vectors and every basis entry LT lanes from registers.  Slices are added through shared memory in
// a fixed order (bit-reproducible).
template <int R, int KT, int LT>
__global__ void __launch_bounds__(256)
restrict_kernel(TransferGeom g, int NP, int PC, int S, const float4 *__restrict__ basis,
                const typename Elem<R>::type *__restrict__ fine, typename Elem<R>::type *__restrict__ coarse) {
    typedef typename Elem<R>::type E;
    extern __shared__ __align__(16) unsigned char sm[];
    const int nagg = g.bx * g.by * g.bz * g.bt;
    long long *s_lex = reinterpret_cast<long long *>(sm);                 // [nagg] canonical site index (basis)
    long long *s_off = s_lex + nagg;                                      // [nagg] native element offset of component 0, lane 0
    E *red = reinterpret_cast<E *>(s_off + nagg);                         // [S-1][items][2 KT LT]
    const int CS = g.XB * NP;
    const long long B = blockIdx.x;
    const int c0x = (int)(B % g.cX), c0y = (int)((B / g.cX) % g.cY), c0z = (int)((B / ((long long)g.cX * g.cY)) % g.cZ);
    const int c0t = (int)(B / ((long long)g.cX * g.cY * g.cZ));
    for (int i = threadIdx.x; i < nagg; i += blockDim.x) {
        int q = i;
        const int ix = q % g.bx; q /= g.bx;
        const int iy = q % g.by; q /= g.by;
        const int iz = q % g.bz;
        const int it = q / g.bz;
        const int x = c0x * g.bx + ix, y = c0y * g.by + iy, z = c0z * g.bz + iz, t = c0t * g.bt + it;
        s_lex[i] = x + (long long)g.X * (y + (long long)g.Y * (z + (long long)g.Z * t));
        const long long b = (x / g.XB) + (long long)g.nxb * (y + (long long)g.Y * (z + (long long)g.Z * t));
        s_off[i] = b * 12 * CS + (long long)(x % g.XB) * NP;
    }
    __syncthreads();
    const int items = (g.nvec / KT) * PC;
    const int tid = threadIdx.x;
    const int s = tid / items, item = tid - s * items;
    const int k0 = (item / PC) * KT, lane = (blockIdx.y * PC + (item - (item / PC) * PC)) * LT;
    const bool active = s < S && lane < NP;   // NP is a multiple of LT
    CVec<R> a0[KT][LT], a1[KT][LT];
#pragma unroll
    for (int kk = 0; kk < KT; kk++)
#pragma unroll
        for (int l = 0; l < LT; l++) { a0[kk][l] = czero_t<R>(); a1[kk][l] = czero_t<R>(); }
    if (active) {
        for (int i = s; i < nagg; i += S) {
            // the threads of a slice ask for the lines of the site some iterations ahead (L2 prefetch), so that the loads
            // below pay L2 instead of HBM latency: the basis of the site and the 12 component runs of the field
            const int ip = i + kRestrictAhead * S;
            if (ip < nagg) {
                if (item * 128 < g.nvec * 96) asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char *>(basis + (size_t)s_lex[ip] * g.nvec * 6) + item * 128));
                if (item < 12) asm volatile("prefetch.global.L2 [%0];" ::"l"(fine + s_off[ip] + (size_t)item * CS + blockIdx.y * PC * LT));
            }
            const float4 *ph = basis + ((size_t)s_lex[i] * g.nvec + k0) * 6;
            const E *pf = fine + s_off[i] + lane;
#pragma unroll
            for (int j = 0; j < 6; j++) {
                CVec<R> f0[LT], f1[LT];
#pragma unroll
                for (int l = 0; l < LT; l++) {
                    f0[l] = to_cvec(__ldg(pf + (size_t)(2 * j) * CS + l));
                    f1[l] = to_cvec(__ldg(pf + (size_t)(2 * j + 1) * CS + l));
                }
#pragma unroll
                for (int kk = 0; kk < KT; kk++) {
                    const float4 a = __ldg(ph + kk * 6 + j);
#pragma unroll
                    for (int l = 0; l < LT; l++) {
                        if (j < 3) { a0[kk][l] = cfma_conj(a.x, a.y, f0[l], a0[kk][l]); a0[kk][l] = cfma_conj(a.z, a.w, f1[l], a0[kk][l]); }
                        else       { a1[kk][l] = cfma_conj(a.x, a.y, f0[l], a1[kk][l]); a1[kk][l] = cfma_conj(a.z, a.w, f1[l], a1[kk][l]); }
                    }
                }
            }
        }
        if (s > 0) {
            E *rp = red + ((size_t)(s - 1) * items + item) * 2 * KT * LT;
#pragma unroll
            for (int kk = 0; kk < KT; kk++)
#pragma unroll
                for (int l = 0; l < LT; l++) {
                    rp[2 * (kk * LT + l)] = from_cvec(a0[kk][l]);
                    rp[2 * (kk * LT + l) + 1] = from_cvec(a1[kk][l]);
                }
        }
    }
    __syncthreads();
    if (active && s == 0) {
        for (int q = 1; q < S; q++) {
            const E *rp = red + ((size_t)(q - 1) * items + item) * 2 * KT * LT;
#pragma unroll
            for (int kk = 0; kk < KT; kk++)
#pragma unroll
                for (int l = 0; l < LT; l++) {
                    a0[kk][l] = cadd(a0[kk][l], to_cvec(rp[2 * (kk * LT + l)]));
                    a1[kk][l] = cadd(a1[kk][l], to_cvec(rp[2 * (kk * LT + l) + 1]));
                }
        }
        E *po = coarse + (size_t)B * 2 * g.nvec * NP + lane;
#pragma unroll
        for (int kk = 0; kk < KT; kk++)
#pragma unroll
            for (int l = 0; l < LT; l++) {
                po[(size_t)(k0 + kk) * NP + l] = from_cvec(a0[kk][l]);
                po[(size_t)(g.nvec + k0 + kk) * NP + l] = from_cvec(a1[kk][l]);
            }
    }
}


// Restriction with both operands staged in shared memory (even N_rhs, block extent in x dividing the layout block XB).
// A thread block owns the XB / bx aggregates that share an x-block and walks their by x bz x bt rows; a row is ONE contiguous run in
// the field (the layout block row: 12 components x XB sites x NP lanes) and ONE in the basis (XB sites x n_vec x 96 bytes), brought
// in by two bulk async copies per row into a ring of stages (a producer warp, mbarriers), so each SM has tens of KB of both streams
// in flight.  A consumer warp is one slice of the sites (position of the site inside its aggregate's x-run, row index modulo RS);
// its lanes are the (aggregate, chirality, group of KT basis vectors, group of LT lanes) tiles, each summing KT x LT coefficients in
// registers: per site and tile 3 KT + 6 LT shared-memory loads of 16 bytes feed 24 KT LT FFMA2.  Slices are added through shared
// memory in a fixed order (bit-reproducible).
constexpr int kRestrictStages = 4;
template <int KT, int LT>
__global__ void __launch_bounds__(288, 2)
restrict_staged_kernel(TransferGeom g, int NP, int RS, const float4 *__restrict__ basis, const float4 *__restrict__ fine, float4 *__restrict__ coarse) {
    extern __shared__ __align__(128) unsigned char sm[];
    const int XB = g.XB, CS = XB * NP;
    const uint32_t f_bytes = 12u * CS * 16u, b_bytes = (uint32_t)XB * g.nvec * 96u, st_bytes = f_bytes + b_bytes;
    uint64_t *full = reinterpret_cast<uint64_t *>(sm + (size_t)kRestrictStages * st_bytes), *empty = full + kRestrictStages;
    const int agx = XB / g.bx;                                  // aggregates per block
    const int kgs = g.nvec / KT, lgs = NP / LT, tiles = agx * 2 * kgs * lgs;   // tiles = lanes with work in a consumer warp (<= 32)
    const int S = g.bx * RS, NR = g.by * g.bz * g.bt;           // site slices = consumer warps; rows
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // block -> (x-block, coarse y, z, t)
    long long q = blockIdx.x;
    const int xb = (int)(q % g.nxb); q /= g.nxb;
    const int cy = (int)(q % g.cY); q /= g.cY;
    const int cz = (int)(q % g.cZ);
    const int ct = (int)(q / g.cZ);
    if (tid == 0) {
        for (int i = 0; i < kRestrictStages; i++) { mbar_init(&full[i], 1); mbar_init(&empty[i], S); }
        mbar_fence_init();
    }
    __syncthreads();
    if (warp == S) {
        // ------------------------------------------------ producer
        if (lane == 0) {
            for (int r = 0; r < NR; r++) {
                const int st = r % kRestrictStages;
                if (r >= kRestrictStages) mbar_wait(&empty[st], ((r / kRestrictStages) - 1) & 1);
                int w = r;
                const int iy = w % g.by; w /= g.by;
                const int iz = w % g.bz;
                const int it = w / g.bz;
                const long long yzt = (cy * g.by + iy) + (long long)g.Y * ((cz * g.bz + iz) + (long long)g.Z * (ct * g.bt + it));
                unsigned char *dst = sm + (size_t)st * st_bytes;
                mbar_expect_tx(&full[st], st_bytes);
                bulk_g2s(dst, fine + ((size_t)xb + (size_t)g.nxb * yzt) * 12 * CS, f_bytes, &full[st]);
                bulk_g2s(dst + f_bytes, basis + ((size_t)xb * XB + (size_t)g.X * yzt) * g.nvec * 6, b_bytes, &full[st]);
            }
        }
    } else if (warp < S) {
        // ------------------------------------------------ consumers
        const int xs = warp % g.bx, rp = warp / g.bx;          // position in the aggregate's x-run, row class
        // lane -> tile; the aggregate and the chirality are the high bits so that the eight lanes of a quarter-warp share them
        // (their field rows are a multiple of 128 bytes apart: the same banks)
        const bool has = lane < tiles;
        const int tl = has ? lane : 0;
        const int a = tl / (2 * kgs * lgs), chi = (tl / (kgs * lgs)) & 1, kg = (tl / lgs) % kgs, lg = tl % lgs;
        const int xin = a * g.bx + xs;
        CVec<2> acc[KT][LT];
#pragma unroll
        for (int kk = 0; kk < KT; kk++)
#pragma unroll
            for (int l = 0; l < LT; l++) acc[kk][l] = czero_t<2>();
        for (int r = 0; r < NR; r++) {
            const int st = r % kRestrictStages;
            // every warp waits for every row, also the rows of other row classes: a warp that ran ahead would arrive twice in one
            // phase of the stage's empty barrier
            mbar_wait(&full[st], (r / kRestrictStages) & 1);
            if (r % RS == rp) {
                const float4 *sf = reinterpret_cast<const float4 *>(sm + (size_t)st * st_bytes) + ((size_t)(chi * 6) * XB + xin) * NP + lg * LT;
                const float4 *sb = reinterpret_cast<const float4 *>(sm + (size_t)st * st_bytes + f_bytes) + ((size_t)xin * g.nvec + kg * KT) * 6 + chi * 3;
#pragma unroll
                for (int j = 0; j < 3; j++) {
                    CVec<2> f0[LT], f1[LT];
#pragma unroll
                    for (int l = 0; l < LT; l++) {
                        f0[l] = to_cvec(sf[(size_t)(2 * j) * CS + l]);
                        f1[l] = to_cvec(sf[(size_t)(2 * j + 1) * CS + l]);
                    }
#pragma unroll
                    for (int kk = 0; kk < KT; kk++) {
                        const float4 p = sb[kk * 6 + j];           // components 2j, 2j+1 of this chirality
#pragma unroll
                        for (int l = 0; l < LT; l++) {
                            acc[kk][l] = cfma_conj(p.x, p.y, f0[l], acc[kk][l]);
                            acc[kk][l] = cfma_conj(p.z, p.w, f1[l], acc[kk][l]);
                        }
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[st]);
        }
        // every row has been consumed by every warp (the arrivals above): the ring is free for the slice sums
        // [slice][tile][KT LT] float4
        float4 *red = reinterpret_cast<float4 *>(sm);
        asm volatile("bar.sync 1, %0;" ::"r"(S * 32) : "memory");
        if (has && warp > 0) {
            float4 *rp4 = red + ((size_t)(warp - 1) * tiles + tl) * KT * LT;
#pragma unroll
            for (int kk = 0; kk < KT; kk++)
#pragma unroll
                for (int l = 0; l < LT; l++) rp4[kk * LT + l] = from_cvec(acc[kk][l]);
        }
        asm volatile("bar.sync 1, %0;" ::"r"(S * 32) : "memory");
        if (has && warp == 0) {
            for (int w = 1; w < S; w++) {
                const float4 *rp4 = red + ((size_t)(w - 1) * tiles + tl) * KT * LT;
#pragma unroll
                for (int kk = 0; kk < KT; kk++)
#pragma unroll
                    for (int l = 0; l < LT; l++) acc[kk][l] = cadd(acc[kk][l], to_cvec(rp4[kk * LT + l]));
            }
            const long long B = (xb * agx + a) + (long long)g.cX * (cy + (long long)g.cY * (cz + (long long)g.cZ * ct));
            float4 *po = coarse + ((size_t)B * 2 * g.nvec + (size_t)chi * g.nvec + kg * KT) * NP + lg * LT;
#pragma unroll
            for (int kk = 0; kk < KT; kk++)
#pragma unroll
                for (int l = 0; l < LT; l++) po[(size_t)kk * NP + l] = from_cvec(acc[kk][l]);
        }
    }
}


// Prolongation with the basis streamed through a ring of shared-memory stages (even N_rhs, block extent in x dividing XB): the same
// block / row decomposition as restrict_staged_kernel.  The 2 n_vec coefficient vectors of the block's XB / bx aggregates are staged
// once; a basis row (XB sites x n_vec x 96 bytes, contiguous) arrives by one bulk async copy per row.  A consumer warp takes every
// NW-th row; its lanes are the (site of the row, chirality, group of LT lanes) tiles, each producing the six components of its
// chirality for LT lanes: per basis vector 3 + LT shared-memory loads of 16 bytes feed 24 LT FFMA2.
template <int LT>
__global__ void __launch_bounds__(160, 3)
prolong_staged_kernel(TransferGeom g, int NP, int NW, const float4 *__restrict__ basis, const float4 *__restrict__ coarse, float4 *__restrict__ fine) {
    extern __shared__ __align__(128) unsigned char sm[];
    const int XB = g.XB, CS = XB * NP;
    // a site's basis (n_vec x 96 bytes) is copied on its own and lands one float4 further than a dense row would put it: the lanes of
    // a quarter-warp read four sites at the same (k, component), 1920 bytes apart in a dense row = the same banks
    const uint32_t site_bytes = (uint32_t)g.nvec * 96u, site_pitch = site_bytes + 16u, b_bytes = (uint32_t)XB * site_pitch;
    const int agx = XB / g.bx, lgs = NP / LT, tiles = XB * 2 * lgs, NR = g.by * g.bz * g.bt;
    const uint32_t c_bytes = (uint32_t)agx * 2u * g.nvec * NP * 16u;
    float4 *sc = reinterpret_cast<float4 *>(sm + (size_t)kRestrictStages * b_bytes);                    // [aggregate][2 n_vec][NP]
    uint64_t *full = reinterpret_cast<uint64_t *>(sm + (size_t)kRestrictStages * b_bytes + c_bytes), *empty = full + kRestrictStages, *cfull = empty + kRestrictStages;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    long long q = blockIdx.x;
    const int xb = (int)(q % g.nxb); q /= g.nxb;
    const int cy = (int)(q % g.cY); q /= g.cY;
    const int cz = (int)(q % g.cZ);
    const int ct = (int)(q / g.cZ);
    if (tid == 0) {
        for (int i = 0; i < kRestrictStages; i++) { mbar_init(&full[i], 1); mbar_init(&empty[i], 1); }
        mbar_init(cfull, 1);
        mbar_fence_init();
    }
    __syncthreads();
    auto row_yzt = [&](int r) {
        const int iy = r % g.by; r /= g.by;
        const int iz = r % g.bz;
        const int it = r / g.bz;
        return (long long)(cy * g.by + iy) + (long long)g.Y * ((cz * g.bz + iz) + (long long)g.Z * (ct * g.bt + it));
    };
    if (warp == NW) {
        // ------------------------------------------------ producer
        if (lane == 0) {
            mbar_expect_tx(cfull, c_bytes);
            for (int a = 0; a < agx; a++) {
                const long long B = (xb * agx + a) + (long long)g.cX * (cy + (long long)g.cY * (cz + (long long)g.cZ * ct));
                bulk_g2s(sc + (size_t)a * 2 * g.nvec * NP, coarse + (size_t)B * 2 * g.nvec * NP, c_bytes / agx, cfull);
            }
        }
        for (int r = 0; r < NR; r++) {
            const int st = r % kRestrictStages;
            if (r >= kRestrictStages) mbar_wait(&empty[st], ((r / kRestrictStages) - 1) & 1);
            if (lane == 0) mbar_expect_tx(&full[st], XB * site_bytes);
            __syncwarp();
            if (lane < XB)
                bulk_g2s(sm + (size_t)st * b_bytes + (size_t)lane * site_pitch, basis + ((size_t)xb * XB + lane + (size_t)g.X * row_yzt(r)) * g.nvec * 6, site_bytes, &full[st]);
        }
    } else if (warp < NW) {
        // ------------------------------------------------ consumers: warp w takes rows w, w + NW, ...; each row is read by one warp only
        const bool has = lane < tiles;
        const int tl = has ? lane : 0;
        const int chi = tl / (XB * lgs), xin = (tl / lgs) % XB, lg = tl % lgs;
        const float4 *vc = sc + ((size_t)(xin / g.bx) * 2 * g.nvec + (size_t)chi * g.nvec) * NP + lg * LT;
        mbar_wait(cfull, 0);
        for (int r = warp; r < NR; r += NW) {
            const int st = r % kRestrictStages;
            mbar_wait(&full[st], (r / kRestrictStages) & 1);
            const float4 *sb = reinterpret_cast<const float4 *>(sm + (size_t)st * b_bytes + (size_t)xin * site_pitch) + chi * 3;
            CVec<2> acc[6][LT];
#pragma unroll
            for (int c = 0; c < 6; c++)
#pragma unroll
                for (int l = 0; l < LT; l++) acc[c][l] = czero_t<2>();
#pragma unroll 4
            for (int k = 0; k < g.nvec; k++) {
                CVec<2> v[LT];
#pragma unroll
                for (int l = 0; l < LT; l++) v[l] = to_cvec(vc[(size_t)k * NP + l]);
#pragma unroll
                for (int j = 0; j < 3; j++) {
                    const float4 p = sb[k * 6 + j];
#pragma unroll
                    for (int l = 0; l < LT; l++) {
                        acc[2 * j][l] = cfma(p.x, p.y, v[l], acc[2 * j][l]);
                        acc[2 * j + 1][l] = cfma(p.z, p.w, v[l], acc[2 * j + 1][l]);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[st]);
            if (has) {
                float4 *po = fine + ((size_t)xb + (size_t)g.nxb * row_yzt(r)) * 12 * CS + ((size_t)(chi * 6) * XB + xin) * NP + lg * LT;
#pragma unroll
                for (int c = 0; c < 6; c++)
#pragma unroll
                    for (int l = 0; l < LT; l++) __stcs(po + (size_t)c * CS + l, from_cvec(acc[c][l]));
            }
        }
    }
}

// ------------------------------------------------------------------ coarse -> coarser
__global__ void pack_basis_coarse_kernel(int nvec, int nf, long long V, const float2 *__restrict__ src, float2 *__restrict__ dst, long long total) {
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;   // native order [x][k][c]
    if (idx >= total) return;
    const int c = (int)(idx % nf);
    long long q = idx / nf;
    const int k = (int)(q % nvec);
    const long long x = q / nvec;
    dst[idx] = src[((long long)k * V + x) * nf + c];
}

__device__ __forceinline__ long long coarser_block(const CoarseTransferGeom &g, long long x) {
    const int ix = (int)(x % g.X); x /= g.X;
    const int iy = (int)(x % g.Y); x /= g.Y;
    const int iz = (int)(x % g.Z);
    const int it = (int)(x / g.Z);
    return (ix / g.bx) + (long long)g.cX * ((iy / g.by) + (long long)g.cY * ((iz / g.bz) + (long long)g.cZ * (it / g.bt)));
}

// One thread = one finer site, two components (same chirality: nf / 2 is even) and TP RHS lanes; per basis vector k one
// 16-byte load of phi_k(x)[2 cp .. 2 cp + 1] and TP loads of the block's coarser coefficients feed 2 TP complex FMAs.
template <int R, int TP>
__global__ void __launch_bounds__(256, 4)       // 64 registers: four blocks per SM; with eight basis loads in flight per thread 0.068 -> 0.051 ms at 6^3x32, N = 12
prolong_coarse_kernel(CoarseTransferGeom g, int NP, int items, long long nthreads, const float4 *__restrict__ basis,
                      const typename Elem<R>::type *__restrict__ coarse, typename Elem<R>::type *__restrict__ fine) {
    typedef typename Elem<R>::type E;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= nthreads) return;
    const long long x = gid / items;
    const int item = (int)(gid - x * items);
    const int lgs = NP / TP, cp = item / lgs, lane = (item - cp * lgs) * TP;
    const int chi = 2 * cp >= g.nf / 2;
    const E *vc = coarse + ((size_t)coarser_block(g, x) * 2 * g.nvec + (size_t)chi * g.nvec) * NP + lane;
    const float4 *ph = basis + ((size_t)x * g.nvec * g.nf) / 2 + cp;          // float4 = two complex components
    CVec<R> acc[2][TP];
#pragma unroll
    for (int l = 0; l < TP; l++) { acc[0][l] = czero_t<R>(); acc[1][l] = czero_t<R>(); }
#pragma unroll 8
    for (int k = 0; k < g.nvec; k++) {
        const float4 a = __ldg(ph + (size_t)k * (g.nf / 2));
#pragma unroll
        for (int l = 0; l < TP; l++) {
            const CVec<R> v = to_cvec(__ldg(vc + (size_t)k * NP + l));
            acc[0][l] = cfma(a.x, a.y, v, acc[0][l]);
            acc[1][l] = cfma(a.z, a.w, v, acc[1][l]);
        }
    }
    E *po = fine + ((size_t)x * g.nf + 2 * cp) * NP + lane;
#pragma unroll
    for (int l = 0; l < TP; l++) { po[l] = from_cvec(acc[0][l]); po[NP + l] = from_cvec(acc[1][l]); }
}

// One thread block cluster of G blocks = one aggregate (a coarse level has few aggregates: 128 at 6^3x32 / 3x3x3x2, fewer than SMs);
// a thread owns one (site slice, chirality, KT basis vectors, LT RHS lanes) and sums its slice of the aggregate's sites over the
// nf / 2 components of its chirality; the slices of a block are added through shared memory, the blocks of the cluster through
// distributed shared memory by block 0, both in a fixed order (bit-reproducible).
template <int R, int KT, int LT>
__global__ void __launch_bounds__(256)
restrict_coarse_kernel(CoarseTransferGeom g, int NP, int S, int G, const float2 *__restrict__ basis,
                       const typename Elem<R>::type *__restrict__ fine, typename Elem<R>::type *__restrict__ coarse) {
    typedef typename Elem<R>::type E;
    extern __shared__ __align__(16) unsigned char sm[];
    const int nagg = g.bx * g.by * g.bz * g.bt, h = g.nf / 2;
    const int kgs = g.nvec / KT, lgs = NP / LT, items = 2 * kgs * lgs;
    E *part = reinterpret_cast<E *>(sm);                                  // [items][KT LT]: this block's sums, read by block 0 of the cluster
    E *red = part + (size_t)items * KT * LT;                              // [S-1][items][KT LT]
    const long long B = blockIdx.x / G;
    const int crank = (int)(blockIdx.x - B * G);                          // rank in the cluster: blocks B G .. B G + G - 1
    const int c0x = (int)(B % g.cX) * g.bx, c0y = (int)((B / g.cX) % g.cY) * g.by, c0z = (int)((B / ((long long)g.cX * g.cY)) % g.cZ) * g.bz;
    const int c0t = (int)(B / ((long long)g.cX * g.cY * g.cZ)) * g.bt;
    const int tid = threadIdx.x, s = tid / items, item = tid - s * items;
    const int chi = item / (kgs * lgs), rem = item - chi * (kgs * lgs), k0 = (rem / lgs) * KT, lane = (rem - (rem / lgs) * lgs) * LT;
    const bool active = s < S;
    CVec<R> acc[KT][LT];
#pragma unroll
    for (int kk = 0; kk < KT; kk++)
#pragma unroll
        for (int l = 0; l < LT; l++) acc[kk][l] = czero_t<R>();
    if (active) {
        for (int i = crank * S + s; i < nagg; i += S * G) {
            int q = i;
            const int ix = q % g.bx; q /= g.bx;
            const int iy = q % g.by; q /= g.by;
            const int iz = q % g.bz;
            const int it = q / g.bz;
            const long long x = (c0x + ix) + (long long)g.X * ((c0y + iy) + (long long)g.Y * ((c0z + iz) + (long long)g.Z * (c0t + it)));
            const float2 *ph = basis + ((size_t)x * g.nvec + k0) * g.nf + chi * h;
            const E *pf = fine + ((size_t)x * g.nf + chi * h) * NP + lane;
#pragma unroll 20       // all of nf / 2 = 20 components of config 4 (0.119 -> 0.100 ms at 6^3x32, N = 12)
            for (int c = 0; c < h; c++) {
                CVec<R> f[LT];
#pragma unroll
                for (int l = 0; l < LT; l++) f[l] = to_cvec(__ldg(pf + (size_t)c * NP + l));
#pragma unroll
                for (int kk = 0; kk < KT; kk++) {
                    const float2 a = __ldg(ph + (size_t)kk * g.nf + c);
#pragma unroll
                    for (int l = 0; l < LT; l++) acc[kk][l] = cfma_conj(a.x, a.y, f[l], acc[kk][l]);
                }
            }
        }
        if (s > 0) {
            E *rp = red + ((size_t)(s - 1) * items + item) * KT * LT;
#pragma unroll
            for (int kk = 0; kk < KT; kk++)
#pragma unroll
                for (int l = 0; l < LT; l++) rp[kk * LT + l] = from_cvec(acc[kk][l]);
        }
    }
    __syncthreads();
    if (active && s == 0) {
        for (int q = 1; q < S; q++) {
            const E *rp = red + ((size_t)(q - 1) * items + item) * KT * LT;
#pragma unroll
            for (int kk = 0; kk < KT; kk++)
#pragma unroll
                for (int l = 0; l < LT; l++) acc[kk][l] = cadd(acc[kk][l], to_cvec(rp[kk * LT + l]));
        }
        if (G > 1) {
#pragma unroll
            for (int kk = 0; kk < KT; kk++)
#pragma unroll
                for (int l = 0; l < LT; l++) part[(size_t)item * KT * LT + kk * LT + l] = from_cvec(acc[kk][l]);
        }
    }
    if (G > 1) {
        namespace cg = cooperative_groups;
        cg::cluster_group cluster = cg::this_cluster();
        cluster.sync();                                    // every block of the cluster has written its sums
        if (crank == 0 && active && s == 0) {
            for (int r = 1; r < G; r++) {
                const E *rp = cluster.map_shared_rank(part, r) + (size_t)item * KT * LT;
#pragma unroll
                for (int kk = 0; kk < KT; kk++)
#pragma unroll
                    for (int l = 0; l < LT; l++) acc[kk][l] = cadd(acc[kk][l], to_cvec(rp[kk * LT + l]));
            }
        }
        cluster.sync();                                    // block 0 has read them: the other blocks may exit
    }
    if (crank == 0 && active && s == 0) {
        E *po = coarse + ((size_t)B * 2 * g.nvec + (size_t)chi * g.nvec + k0) * NP + lane;
#pragma unroll
        for (int kk = 0; kk < KT; kk++)
#pragma unroll
            for (int l = 0; l < LT; l++) po[(size_t)kk * NP + l] = from_cvec(acc[kk][l]);
    }
}

}  // namespace

mrhs_status_t pack_basis(const TransferGeom &g, const float2 *d_canonical, float2 *d_native, cudaStream_t st) {
    const long long total = g.nsites * g.nvec * 12;
    pack_basis_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(g.nvec, g.nsites, d_canonical, d_native, total);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

namespace {
template <int LT>
bool try_prolong_staged(const TransferGeom &g, int np, const float2 *d_basis, const void *d_coarse, void *d_fine, cudaStream_t st, mrhs_status_t *status) {
    if ((g.N & 1) || g.XB % g.bx || np % LT) return false;
    const int tiles = g.XB * 2 * (np / LT);
    if (tiles > 32 || tiles < 16) return false;
    const int agx = g.XB / g.bx, NR = g.by * g.bz * g.bt;
    const int NW = NR < 4 ? NR : 4;      // four consumer warps + the producer: three blocks per SM at 136 registers
    const size_t smem = (size_t)kRestrictStages * g.XB * (g.nvec * 96 + 16) + (size_t)agx * 2 * g.nvec * np * 16 + (2 * kRestrictStages + 1) * 8;
    if (smem > 72 * 1024) return false;
    *status = MRHS_OK;
    cudaError_t e = cudaFuncSetAttribute(prolong_staged_kernel<LT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 72 * 1024);
    if (e != cudaSuccess) { *status = cuda_fail(e, "cudaFuncSetAttribute", __FILE__, __LINE__); return true; }
    const long long grid = (long long)g.nxb * g.cY * g.cZ * g.cT;
    prolong_staged_kernel<LT><<<(unsigned)grid, (NW + 1) * 32, smem, st>>>(g, np, NW, (const float4 *)d_basis, (const float4 *)d_coarse, (float4 *)d_fine);
    e = cudaGetLastError();
    if (e != cudaSuccess) *status = cuda_fail(e, "prolong_staged_kernel", __FILE__, __LINE__);
    return true;
}
}  // namespace

mrhs_status_t launch_prolong(const TransferGeom &g, const float2 *d_basis, const void *d_coarse, void *d_fine, cudaStream_t st) {
    const int np = threads_per_site(g.N);
    {
        mrhs_status_t status = MRHS_OK;
        if (try_prolong_staged<3>(g, np, d_basis, d_coarse, d_fine, st, &status)) return status;
        if (try_prolong_staged<2>(g, np, d_basis, d_coarse, d_fine, st, &status)) return status;
    }
    const long long nthreads = g.nsites * np;
    // shared-memory staging when at least two blocks fit an SM; the plain kernel otherwise
    const int cs = g.XB * np;
    const int rows = cs <= 256 ? (256 / cs < 2 ? 256 / cs : 2) : 0;   // two rows (96 threads at XB NP = 48) measured best: many small blocks per SM
    const size_t smem = (size_t)rows * g.XB * g.nvec * 96;
    if (rows >= 1 && smem <= 100 * 1024) {
        const long long nblk = (long long)g.nxb * g.Y * g.Z * g.T;
        const unsigned grid = (unsigned)((nblk + rows - 1) / rows);
        const int threads = rows * cs;
        if (g.N & 1) {
            MRHS_CUDA(cudaFuncSetAttribute(prolong_smem_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
            prolong_smem_kernel<1><<<grid, threads, smem, st>>>(g, np, rows, nblk, (const float4 *)d_basis, (const float2 *)d_coarse, (float2 *)d_fine);
        } else {
            MRHS_CUDA(cudaFuncSetAttribute(prolong_smem_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
            prolong_smem_kernel<2><<<grid, threads, smem, st>>>(g, np, rows, nblk, (const float4 *)d_basis, (const float4 *)d_coarse, (float4 *)d_fine);
        }
        MRHS_CUDA(cudaGetLastError());
        return MRHS_OK;
    }
    const unsigned blocks = (unsigned)((nthreads + 255) / 256);
    if (g.N & 1) prolong_kernel<1><<<blocks, 256, 0, st>>>(g, np, nthreads, (const float4 *)d_basis, (const float2 *)d_coarse, (float2 *)d_fine);
    else         prolong_kernel<2><<<blocks, 256, 0, st>>>(g, np, nthreads, (const float4 *)d_basis, (const float4 *)d_coarse, (float4 *)d_fine);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

namespace {
// the staged kernel where its tiling fits: even N_rhs, whole aggregate x-runs inside a layout block, at most 32 tiles per slice
// and 8 slices, four stages + the slice sums in shared memory.  Returns false if it does not apply (nothing launched).
template <int KT, int LT>
bool try_restrict_staged(const TransferGeom &g, int np, const float2 *d_basis, const void *d_fine, void *d_coarse, cudaStream_t st, mrhs_status_t *status) {
    if ((g.N & 1) || g.XB % g.bx || g.nvec % KT || np % LT) return false;
    const int agx = g.XB / g.bx, tiles = agx * 2 * (g.nvec / KT) * (np / LT);
    if (tiles > 32 || tiles < 16 || g.bx > 8) return false;
    const int NR = g.by * g.bz * g.bt;
    int RS = 8 / g.bx;
    while (RS > 1 && NR % RS) RS--;
    const int S = g.bx * RS;
    const size_t st_bytes = (size_t)12 * g.XB * np * 16 + (size_t)g.XB * g.nvec * 96;
    const size_t red = (size_t)(S - 1) * tiles * KT * LT * 16;
    const size_t smem = kRestrictStages * st_bytes + 2 * kRestrictStages * 8;
    if (smem > 110 * 1024 || red > kRestrictStages * st_bytes) return false;
    *status = MRHS_OK;
    cudaError_t e = cudaFuncSetAttribute(restrict_staged_kernel<KT, LT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 110 * 1024);
    if (e != cudaSuccess) { *status = cuda_fail(e, "cudaFuncSetAttribute", __FILE__, __LINE__); return true; }
    const long long grid = (long long)g.nxb * g.cY * g.cZ * g.cT;
    restrict_staged_kernel<KT, LT><<<(unsigned)grid, (S + 1) * 32, smem, st>>>(g, np, RS, (const float4 *)d_basis, (const float4 *)d_fine, (float4 *)d_coarse);
    e = cudaGetLastError();
    if (e != cudaSuccess) *status = cuda_fail(e, "restrict_staged_kernel", __FILE__, __LINE__);
    return true;
}
}  // namespace

mrhs_status_t launch_restrict(const TransferGeom &g, const float2 *d_basis, const void *d_fine, void *d_coarse, cudaStream_t st) {
    const int np = threads_per_site(g.N);
    if (g.nvec > 256) { set_error("restrict: nvec = %d exceeds 256", g.nvec); return MRHS_ERR_UNSUPPORTED; }
    {
        mrhs_status_t status = MRHS_OK;
        if (try_restrict_staged<5, 3>(g, np, d_basis, d_fine, d_coarse, st, &status)) return status;
        if (try_restrict_staged<4, 3>(g, np, d_basis, d_fine, d_coarse, st, &status)) return status;
        if (try_restrict_staged<4, 2>(g, np, d_basis, d_fine, d_coarse, st, &status)) return status;
        if (try_restrict_staged<3, 3>(g, np, d_basis, d_fine, d_coarse, st, &status)) return status;
    }
    const int kt = g.nvec % 4 == 0 ? 4 : (g.nvec % 2 == 0 ? 2 : 1);   // basis vectors per thread
    const int lt = np % 2 == 0 ? 2 : 1;                              // RHS lanes per thread
    const int groups = g.nvec / kt, lgroups = np / lt;
    int pc = 256 / groups;                                           // lane groups per thread block
    if (pc > lgroups) pc = lgroups;
    const int items = groups * pc;
    const int nagg = g.bx * g.by * g.bz * g.bt;
    int S = 256 / items;
    if (S > nagg) S = nagg;
    if (S < 1) S = 1;
    const int threads = S * items;
    const int esz = (g.N & 1) ? 8 : 16;
    const size_t smem = (size_t)nagg * 16 + (size_t)(S - 1) * items * 2 * kt * lt * esz;
    if (smem > 100 * 1024) { set_error("restrict: aggregate of %d sites needs %zu bytes of shared memory (max 100 KB)", nagg, smem); return MRHS_ERR_UNSUPPORTED; }
    dim3 grid((unsigned)g.ncoarse, (unsigned)((lgroups + pc - 1) / pc));
#define MRHS_RESTRICT(RR, KT, LT, ET) MRHS_CUDA(cudaFuncSetAttribute(restrict_kernel<RR, KT, LT>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024)); \
    restrict_kernel<RR, KT, LT><<<grid, threads, smem, st>>>(g, np, pc, S, (const float4 *)d_basis, (const ET *)d_fine, (ET *)d_coarse)
#define MRHS_RESTRICT_KT(RR, LT, ET) do { if (kt == 4) { MRHS_RESTRICT(RR, 4, LT, ET); } else if (kt == 2) { MRHS_RESTRICT(RR, 2, LT, ET); } else { MRHS_RESTRICT(RR, 1, LT, ET); } } while (0)
    if (g.N & 1) {
        if (lt == 2) MRHS_RESTRICT_KT(1, 2, float2); else MRHS_RESTRICT_KT(1, 1, float2);
    } else {
        if (lt == 2) MRHS_RESTRICT_KT(2, 2, float4); else MRHS_RESTRICT_KT(2, 1, float4);
    }
#undef MRHS_RESTRICT_KT
#undef MRHS_RESTRICT
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

mrhs_status_t pack_basis_coarse(const CoarseTransferGeom &g, const float2 *d_canonical, float2 *d_native, cudaStream_t st) {
    const long long total = g.nsites * g.nvec * g.nf;
    pack_basis_coarse_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(g.nvec, g.nf, g.nsites, d_canonical, d_native, total);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

mrhs_status_t launch_prolong_coarse(const CoarseTransferGeom &g, const float2 *d_basis, const void *d_coarse, void *d_fine, cudaStream_t st) {
    const int np = threads_per_site(g.N);
    const int tp = np % 3 == 0 ? 3 : (np % 2 == 0 ? 2 : 1);
    const int items = (g.nf / 2) * (np / tp);
    const long long nthreads = g.nsites * items;
    const unsigned blocks = (unsigned)((nthreads + 255) / 256);
#define MRHS_PC(RR, TP, ET) prolong_coarse_kernel<RR, TP><<<blocks, 256, 0, st>>>(g, np, items, nthreads, (const float4 *)d_basis, (const ET *)d_coarse, (ET *)d_fine)
    if (g.N & 1) { if (tp == 3) MRHS_PC(1, 3, float2); else if (tp == 2) MRHS_PC(1, 2, float2); else MRHS_PC(1, 1, float2); }
    else         { if (tp == 3) MRHS_PC(2, 3, float4); else if (tp == 2) MRHS_PC(2, 2, float4); else MRHS_PC(2, 1, float4); }
#undef MRHS_PC
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

mrhs_status_t launch_restrict_coarse(const CoarseTransferGeom &g, const float2 *d_basis, const void *d_fine, void *d_coarse, cudaStream_t st) {
    const int np = threads_per_site(g.N);
    const int kt = g.nvec % 2 == 0 ? 2 : 1;
    const int lt = np % 3 == 0 ? 3 : (np % 2 == 0 ? 2 : 1);
    const int items = 2 * (g.nvec / kt) * (np / lt);
    if (items > 256) { set_error("restrict (coarse level): %d work items per aggregate exceed one thread block (nvec = %d, nrhs = %d)", items, g.nvec, g.N); return MRHS_ERR_UNSUPPORTED; }
    const int nagg = g.bx * g.by * g.bz * g.bt;
    int S = 256 / items;
    if (S > nagg) S = nagg;
    const int threads = S * items;
    const int esz = (g.N & 1) ? 8 : 16;
    // blocks per aggregate (one cluster): enough to give every SM work when the coarse lattice has few aggregates
    int G = 1;
    while (G < 8 && nagg >= 2 * G * S && g.ncoarse * G < 1024) G *= 2;
    const size_t smem = (size_t)S * items * kt * lt * esz;
    if (smem > 48 * 1024) { set_error("restrict (coarse level): %zu bytes of shared memory needed (max 48 KB)", smem); return MRHS_ERR_UNSUPPORTED; }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(g.ncoarse * G));
    cfg.blockDim = dim3((unsigned)threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)G; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
#define MRHS_RC(RR, KT, LT, ET) MRHS_CUDA(cudaLaunchKernelEx(&cfg, restrict_coarse_kernel<RR, KT, LT>, g, np, S, G, d_basis, (const ET *)d_fine, (ET *)d_coarse))
#define MRHS_RC_LT(RR, KT, ET) do { if (lt == 3) MRHS_RC(RR, KT, 3, ET); else if (lt == 2) MRHS_RC(RR, KT, 2, ET); else MRHS_RC(RR, KT, 1, ET); } while (0)
    if (g.N & 1) { if (kt == 2) MRHS_RC_LT(1, 2, float2); else MRHS_RC_LT(1, 1, float2); }
    else         { if (kt == 2) MRHS_RC_LT(2, 2, float4); else MRHS_RC_LT(2, 1, float4); }
#undef MRHS_RC_LT
#undef MRHS_RC
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

}  // namespace mrhs

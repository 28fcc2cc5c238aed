// fine_hop.cu -- the fine-level hopping kernel:
//   out(x) = sum_mu (1-gamma_mu) U_mu(x) in(x+mu) + (1+gamma_mu) U_mu(x-mu)^+ in(x-mu)
// (reading S3) for N_rhs right-hand sides at once.  One thread owns one output
// site and R right-hand sides (R = 2 packed in FFMA2 lanes for even N_rhs), so the 18 reals of
// a link are fetched once per site and reused by every RHS (PAPER.md:23 (i)).  Gamma matrices:
// Hermitian chiral basis of reading S2; the spin projection to two-component half spinors and
// the reconstruction are written out per direction below.
#include "fine_hop.cuh"
#include "hop_math.cuh"

namespace mrhs {

namespace {

template <int R, int MU, bool FWD>
__device__ __forceinline__ void hop_dir(const typename Elem<R>::type *__restrict__ nb, size_t cs,
                                        const float4 *__restrict__ g, int XB, CVec<R> (&acc)[12], float dg) {
    HopOperands<R> o;
    hop_load<R, MU>(o, nb, cs, g, XB);
    hop_compute<R, MU, FWD>(o, acc, dg);
}

// blk -> origin of its tile.  Sweep order: x-blocks, then y and z tiles inside a chunk, then t, then chunks.
__device__ __forceinline__ void tile_origin(const HopParams &p, uint32_t blk, uint32_t &xb, uint32_t &y0, uint32_t &z0, uint32_t &t0) {
    uint32_t q, yc, zc, ttile, chy, chz;
    p.d_nxb.divmod(blk, q, xb);
    p.d_cy.divmod(q, q, yc);
    p.d_cz.divmod(q, q, zc);
    p.d_ntt.divmod(q, q, ttile);
    p.d_ncy.divmod(q, chz, chy);
    y0 = (chy * p.cy + yc) * p.by;
    z0 = (chz * p.cz + zc) * p.bz;
    t0 = ttile * p.bt;
}

// one instruction asks the copy engine to bring [ptr, ptr+bytes) into L2 (bytes % 16 == 0)
__device__ __forceinline__ void l2_prefetch(const void *ptr, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(ptr), "r"(bytes) : "memory");
}

// XB_, NP_: compile-time layout block and threads per site (0 = take them from p at run time).
// With both fixed every component and link load is base register + immediate offset.
template <int R, bool CB, int XB_, int NP_, int MAXT>
__global__ void __launch_bounds__(MAXT, 1)
hop_kernel(const HopParams p, const typename Elem<R>::type *__restrict__ in, typename Elem<R>::type *__restrict__ out) {
    typedef typename Elem<R>::type E;
    const int XB = XB_ ? XB_ : p.XB;
    const int NP = NP_ ? NP_ : p.NP;
    // thread -> (site in tile, rhs lane)
    uint32_t q, pair, xin, row, ty, tz, tt;
    if (NP_) { q = threadIdx.x / (uint32_t)NP; pair = threadIdx.x - q * NP; }
    else p.d_np.divmod(threadIdx.x, q, pair);
    if (XB_) { row = q / (uint32_t)XB; xin = q - row * XB; }
    else p.d_xb.divmod(q, row, xin);
    p.d_by.divmod(row, q, ty);
    p.d_bz.divmod(q, tt, tz);
    // block -> tile, in sweep order: x-blocks, then y and z tiles inside a chunk, then t, then chunks
    uint32_t xb, ty0, tz0, tt0;
    tile_origin(p, blockIdx.x, xb, ty0, tz0, tt0);
    const int y = (int)(ty0 + ty);
    const int z = (int)(tz0 + tz);
    const int t = (int)(tt0 + tt);

    // L2 prefetch of the rows a later tile in the sweep owns (spinor row of the input field at the
    // same coordinates plus the rows of both link arrays): every input byte of the launch is
    // requested once, pf_dist tiles before its first use, by one bulk-prefetch instruction per
    // contiguous row, so the loads below find their data in L2 instead of waiting on HBM.
    if (p.pf_dist && threadIdx.x < (unsigned)(p.by * p.bz * p.bt) && blockIdx.x + p.pf_dist < gridDim.x) {
        uint32_t fxb, fy0, fz0, ft0, r = threadIdx.x, ry, rz, rt, qq;
        tile_origin(p, blockIdx.x + p.pf_dist, fxb, fy0, fz0, ft0);
        p.d_by.divmod(r, qq, ry);
        p.d_bz.divmod(qq, rt, rz);
        const size_t fb = (size_t)fxb + (size_t)p.nxb * ((fy0 + ry) + (size_t)p.Y * ((fz0 + rz) + (size_t)p.Z * (ft0 + rt)));
        l2_prefetch(in + fb * 12 * XB * NP, (uint32_t)(12 * XB * NP * sizeof(E)));
        l2_prefetch(p.gauge_out + fb * kSiteF4 * XB, (uint32_t)(kSiteF4 * XB * sizeof(float4)));
        if (CB) l2_prefetch(p.gauge_in + fb * kSiteF4 * XB, (uint32_t)(kSiteF4 * XB * sizeof(float4)));
    }

    const int nxb = p.nxb;
    const int sy = nxb, sz = nxb * p.Y, st = nxb * p.Y * p.Z;   // block strides
    const int b = (int)xb + sy * y + sz * z + st * t;
    const size_t cs = (size_t)XB * NP;                        // component stride in elements
    const size_t lane = pair;

    // x neighbours: (block, xin) of x+1 and x-1 in the input field
    int bxp = b, xinp = (int)xin, bxm = b, xinm = (int)xin;
    {
        bool stepp = true, stepm = true;   // does the site index along the line change?
        if (CB) {
            int s = (p.out_parity + y + z + t) & 1;   // x = 2 xe + s on this line of the output field
            stepp = s != 0;                           // x+1 -> xe + s
            stepm = s == 0;                           // x-1 -> xe + s - 1
        }
        if (stepp) {
            if (xinp + 1 < XB) xinp++;
            else { xinp = 0; bxp = ((int)xb + 1 == nxb) ? b - (nxb - 1) : b + 1; }
        }
        if (stepm) {
            if (xinm > 0) xinm--;
            else { xinm = XB - 1; bxm = (xb == 0) ? b + (nxb - 1) : b - 1; }
        }
    }
    const int byp = (y + 1 == p.Y) ? b - (p.Y - 1) * sy : b + sy;
    const int bym = (y == 0) ? b + (p.Y - 1) * sy : b - sy;
    const int bzp = (z + 1 == p.Z) ? b - (p.Z - 1) * sz : b + sz;
    const int bzm = (z == 0) ? b + (p.Z - 1) * sz : b - sz;
    const int btp = (t + 1 == p.T) ? b - (p.T - 1) * st : b + st;
    const int btm = (t == 0) ? b + (p.T - 1) * st : b - st;

#define MRHS_ELEM(bb, xx) (in + ((size_t)(bb) * 12 * XB + (xx)) * NP + lane)
#define MRHS_LINK(base, bb, xx) ((base) + (size_t)(bb) * kSiteF4 * XB + (xx))

    CVec<R> acc[12];
#pragma unroll
    for (int c = 0; c < 12; c++) acc[c] = czero<R>();

    const float dg = p.dagger ? -1.f : 1.f;      // -1: the adjoint (projector signs exchanged, hop_math.cuh)
    const float4 *gown = MRHS_LINK(p.gauge_out, b, xin);
    const E *n0p = MRHS_ELEM(bxp, xinp), *n0m = MRHS_ELEM(bxm, xinm);
    const E *n1p = MRHS_ELEM(byp, xin), *n1m = MRHS_ELEM(bym, xin);
    const E *n2p = MRHS_ELEM(bzp, xin), *n2m = MRHS_ELEM(bzm, xin);
    const E *n3p = MRHS_ELEM(btp, xin), *n3m = MRHS_ELEM(btm, xin);
    const float4 *g0m = MRHS_LINK(p.gauge_in, bxm, xinm), *g1m = MRHS_LINK(p.gauge_in, bym, xin);
    const float4 *g2m = MRHS_LINK(p.gauge_in, bzm, xin), *g3m = MRHS_LINK(p.gauge_in, btm, xin);
    if constexpr (MAXT <= 288) {
        // two hops' operands in flight: the loads of hop k+2 are issued before the arithmetic of hop k
        HopOperands<R> A, B;
        hop_load<R, 0>(A, n0p, cs, gown, XB);
        hop_load<R, 0>(B, n0m, cs, g0m, XB);
        hop_compute<R, 0, true >(A, acc, dg);  hop_load<R, 1>(A, n1p, cs, gown, XB);
        hop_compute<R, 0, false>(B, acc, dg);  hop_load<R, 1>(B, n1m, cs, g1m, XB);
        hop_compute<R, 1, true >(A, acc, dg);  hop_load<R, 2>(A, n2p, cs, gown, XB);
        hop_compute<R, 1, false>(B, acc, dg);  hop_load<R, 2>(B, n2m, cs, g2m, XB);
        hop_compute<R, 2, true >(A, acc, dg);  hop_load<R, 3>(A, n3p, cs, gown, XB);
        hop_compute<R, 2, false>(B, acc, dg);  hop_load<R, 3>(B, n3m, cs, g3m, XB);
        hop_compute<R, 3, true >(A, acc, dg);
        hop_compute<R, 3, false>(B, acc, dg);
    } else {
        hop_dir<R, 0, true >(n0p, cs, gown, XB, acc, dg);
        hop_dir<R, 0, false>(n0m, cs, g0m, XB, acc, dg);
        hop_dir<R, 1, true >(n1p, cs, gown, XB, acc, dg);
        hop_dir<R, 1, false>(n1m, cs, g1m, XB, acc, dg);
        hop_dir<R, 2, true >(n2p, cs, gown, XB, acc, dg);
        hop_dir<R, 2, false>(n2m, cs, g2m, XB, acc, dg);
        hop_dir<R, 3, true >(n3p, cs, gown, XB, acc, dg);
        hop_dir<R, 3, false>(n3m, cs, g3m, XB, acc, dg);
    }

    E *o = out + ((size_t)b * 12 * XB + xin) * NP + lane;
#pragma unroll
    for (int c = 0; c < 12; c++) o[c * cs] = from_cvec(acc[c]);
#undef MRHS_ELEM
#undef MRHS_LINK
}

// ------------------------------------------------------------- site data packing
// one thread per float of the native array
__global__ void pack_site_kernel(FieldGeom g, const float *__restrict__ src, float *__restrict__ dst, long long total) {
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    int k = (int)(idx & 3);
    long long q = idx >> 2;
    int xin = (int)(q % g.XB); q /= g.XB;
    int j = (int)(q % kSiteF4);
    long long b = q / kSiteF4;
    int xb = (int)(b % g.nxb); b /= g.nxb;
    int y = (int)(b % g.Y); b /= g.Y;
    int z = (int)(b % g.Z);
    int t = (int)(b / g.Z);
    int x = x_of(g, xb * g.XB + xin, y, z, t);
    long long lex = x + (long long)g.X * (y + (long long)g.Y * (z + (long long)g.Z * t));
    dst[idx] = src[lex * 72 + 4 * j + k];
}
__global__ void unpack_site_kernel(FieldGeom g, const float *__restrict__ src, float *__restrict__ dst, long long total) {
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    int k = (int)(idx & 3);
    long long q = idx >> 2;
    int xin = (int)(q % g.XB); q /= g.XB;
    int j = (int)(q % kSiteF4);
    long long b = q / kSiteF4;
    int xb = (int)(b % g.nxb); b /= g.nxb;
    int y = (int)(b % g.Y); b /= g.Y;
    int z = (int)(b % g.Z);
    int t = (int)(b / g.Z);
    int x = x_of(g, xb * g.XB + xin, y, z, t);
    long long lex = x + (long long)g.X * (y + (long long)g.Y * (z + (long long)g.Z * t));
    dst[lex * 72 + 4 * j + k] = src[idx];
}

}  // namespace

mrhs_status_t pack_site_data(const FieldGeom &g, const float *d_src, float4 *d_dst, cudaStream_t st) {
    long long total = g.nsites * 72;
    long long blocks = (total + 255) / 256;
    pack_site_kernel<<<(unsigned)blocks, 256, 0, st>>>(g, d_src, (float *)d_dst, total);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

mrhs_status_t unpack_site_data(const FieldGeom &g, const float4 *d_src, float *d_dst, cudaStream_t st) {
    long long total = g.nsites * 72;
    long long blocks = (total + 255) / 256;
    unpack_site_kernel<<<(unsigned)blocks, 256, 0, st>>>(g, (const float *)d_src, d_dst, total);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

// ------------------------------------------------------------------ tiling
HopTiling default_tiling(const FieldGeom &g, size_t l2_budget) {
    const int np = threads_per_site(g.N);
    const int per_row = g.XB * np;
    // Small thread blocks (about three warps, several resident per SM) measured faster than one large
    // block per SM at 48^4: their load and arithmetic phases drift apart instead of all warps of an
    // SM waiting on the same neighbour rows at once (measured in round 1).
    int rows_max = kHopTargetThreads / per_row;
    if (rows_max < 1) rows_max = 1;
    HopTiling best = {1, 1, 1, 1, 1};
    double best_score = -1.0;
    for (int by = 1; by <= g.Y; by++) {
        if (g.Y % by) continue;
        for (int bz = 1; bz <= g.Z; bz++) {
            if (g.Z % bz) continue;
            for (int bt = 1; bt <= g.T; bt++) {
                if (g.T % bt) continue;
                int rows = by * bz * bt;
                if (rows > rows_max) continue;
                // prefer full warps and many rows, then the smallest surface (neighbour rows outside the tile)
                int thr = rows * per_row;
                double fill = (double)thr / (double)(((thr + 31) / 32) * 32);
                double surf = 1.0 / by + 1.0 / bz + 1.0 / bt;
                double score = rows * fill * 16.0 - surf;
                if (score > best_score) { best_score = score; best.by = by; best.bz = bz; best.bt = bt; }
            }
        }
    }
    // L2 sweep chunk: the kernel walks t inside a (y,z) chunk; about six t-slices of the chunk are
    // live (t-1, t, t+1 of the tiles in flight), each site costing 96 N bytes of input.
    const int nty = g.Y / best.by, ntz = g.Z / best.bz;
    const double slice_site_bytes = 96.0 * g.N * 6.0;
    double best_c = -1.0;
    for (int cy = 1; cy <= nty; cy++) {
        if (nty % cy) continue;
        for (int cz = 1; cz <= ntz; cz++) {
            if (ntz % cz) continue;
            double sites = (double)g.Xe * cy * best.by * cz * best.bz;
            bool fits = sites * slice_site_bytes <= (double)l2_budget;
            if (!fits && !(cy == 1 && cz == 1)) continue;
            // halo re-read of the chunk faces: 2/extent per chunked direction
            double ey = cy * best.by, ez = cz * best.bz;
            double over = (cy == nty ? 0.0 : 2.0 / ey) + (cz == ntz ? 0.0 : 2.0 / ez);
            double score = 1.0 / (1.0 + over) + 1e-9 * sites;
            if (score > best_c) { best_c = score; best.cy = cy; best.cz = cz; }
        }
    }
    return best;
}

bool build_hop_params(const FieldGeom &g, int out_parity, const HopTiling &t, HopParams &p) {
    if (t.by < 1 || t.bz < 1 || t.bt < 1 || t.cy < 1 || t.cz < 1) return false;
    if (g.Y % t.by || g.Z % t.bz || g.T % t.bt) return false;
    const int nty = g.Y / t.by, ntz = g.Z / t.bz, ntt = g.T / t.bt;
    if (nty % t.cy || ntz % t.cz) return false;
    const int np = threads_per_site(g.N);
    const long long threads = (long long)t.by * t.bz * t.bt * g.XB * np;
    if (threads > kHopMaxThreads) return false;
    const long long grid = (long long)g.nxb * nty * ntz * ntt;
    if (grid >= (1ll << 31)) return false;
    p.Y = g.Y; p.Z = g.Z; p.T = g.T;
    p.XB = g.XB; p.nxb = g.nxb; p.NP = np;
    p.cb = g.cb; p.out_parity = out_parity;
    p.dagger = 0;
    p.by = t.by; p.bz = t.bz; p.bt = t.bt; p.cy = t.cy; p.cz = t.cz;
    bool ok = true;
    ok &= make_fastdiv(np, kHopMaxThreads, p.d_np);
    ok &= make_fastdiv(g.XB, kHopMaxThreads, p.d_xb);
    ok &= make_fastdiv(t.by, kHopMaxThreads, p.d_by);
    ok &= make_fastdiv(t.bz, kHopMaxThreads, p.d_bz);
    ok &= make_fastdiv(g.nxb, grid, p.d_nxb);
    ok &= make_fastdiv(t.cy, grid, p.d_cy);
    ok &= make_fastdiv(t.cz, grid, p.d_cz);
    ok &= make_fastdiv(ntt, grid, p.d_ntt);
    ok &= make_fastdiv(nty / t.cy, grid, p.d_ncy);
    if (!ok) return false;
    p.gauge_out = p.gauge_in = nullptr;
    // default prefetch distance: one t-step of the chunk (the t+1 rows a tile reads) plus two waves of tiles
    // default prefetch distance: about half of the tiles resident on the GPU at once (two per SM).  Farther
    // ahead the prefetched rows are evicted again before their tile runs and DRAM reads double (measured).
    p.pf_dist = 2u * 148u;      // the handle replaces this with twice its SM count
    p.grid = (unsigned)grid;
    p.threads = (unsigned)threads;
    return true;
}

namespace {
template <int R, int XB_, int NP_>
void launch_hop_t(const HopParams &p, const void *d_in, void *d_out, cudaStream_t st) {
    typedef typename Elem<R>::type E;
    // CTAs of 193..288 threads get the 224-register build (deeper load pipelining); everything else the
    // 168-register one, which also lets several small CTAs share an SM.
    if (p.threads > 192 && p.threads <= 288) {
        if (p.cb) hop_kernel<R, true, XB_, NP_, 288><<<p.grid, p.threads, 0, st>>>(p, (const E *)d_in, (E *)d_out);
        else      hop_kernel<R, false, XB_, NP_, 288><<<p.grid, p.threads, 0, st>>>(p, (const E *)d_in, (E *)d_out);
    } else {
        if (p.cb) hop_kernel<R, true, XB_, NP_, kHopMaxThreads><<<p.grid, p.threads, 0, st>>>(p, (const E *)d_in, (E *)d_out);
        else      hop_kernel<R, false, XB_, NP_, kHopMaxThreads><<<p.grid, p.threads, 0, st>>>(p, (const E *)d_in, (E *)d_out);
    }
}
}  // namespace

mrhs_status_t launch_hop(const HopParams &p, int nrhs, const void *d_in, void *d_out, cudaStream_t st) {
    const int key = p.XB * 1000 + p.NP;
    if (nrhs & 1) {
        switch (key) {
            case 16001: launch_hop_t<1, 16, 1>(p, d_in, d_out, st); break;
            case 12001: launch_hop_t<1, 12, 1>(p, d_in, d_out, st); break;
            default:    launch_hop_t<1, 0, 0>(p, d_in, d_out, st); break;
        }
    } else {
        switch (key) {
            case 8006:  launch_hop_t<2, 8, 6>(p, d_in, d_out, st); break;     // N = 12
            case 6006:  launch_hop_t<2, 6, 6>(p, d_in, d_out, st); break;     // N = 12, 24^4 checkerboarded
            case 4012:  launch_hop_t<2, 4, 12>(p, d_in, d_out, st); break;    // N = 24
            case 2024:  launch_hop_t<2, 2, 24>(p, d_in, d_out, st); break;    // N = 48
            case 1048:  launch_hop_t<2, 1, 48>(p, d_in, d_out, st); break;    // N = 96
            case 16002: launch_hop_t<2, 16, 2>(p, d_in, d_out, st); break;    // N = 4
            case 12002: launch_hop_t<2, 12, 2>(p, d_in, d_out, st); break;    // N = 4
            default:    launch_hop_t<2, 0, 0>(p, d_in, d_out, st); break;
        }
    }
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

}  // namespace mrhs

// fine_sweep.cu -- slice-sweep variant of the fine-level hopping kernel:
//   out(x) = sum_mu (1-gamma_mu) U_mu(x) in(x+mu) + (1+gamma_mu) U_mu(x-mu)^+ in(x-mu)
// (reading S3) for N_rhs right-hand sides at once, D_hop and M_eooe from one body with
// different index maps ("different site ordering").
//
// Why a second kernel: ncu shows the gather kernel of fine_hop.cu at the L2 -> SM crossbar limit
// (12.2 TB/s), not at the HBM limit: every neighbour spinor is fetched from L2 again by each of its
// eight users.  Here a thread block owns a tile of XB x 2 x 2 sites in (x,y,z) and sweeps a segment
// of t, and every operand of a step is staged in shared memory once:
//   * tile rows of the current slice and the links: cp.async.bulk by a producer warp, double buffered,
//     completion on mbarriers (the only block-wide synchronisation of a step);
//   * the +t hop reads the next slice, which is resident already because it is the next centre slice;
//   * the -t hop of slice s+1 is computed while slice s is the centre and carried in registers (it is
//     the initial value of the next accumulator), so no slice is loaded twice along t;
//   * y, z and x halo neighbours: every thread owns a private shared-memory slot per direction and
//     refills it itself with 16-byte cp.async right after reading it, for the next slice; only that
//     thread ever touches the slot, so cp.async.wait_group is all the synchronisation it needs.
// One thread still owns one output site and one RHS pair (FFMA2 lanes); links are broadcast reads.
#include "fine_sweep.cuh"
#include "hop_math.cuh"

namespace mrhs {

namespace {

constexpr int BY = kSweepBY, BZ = kSweepBZ, ROWS = kSweepRows;
static_assert(BY == 2 && BZ == 2, "every thread has exactly one halo neighbour in y and one in z");

__device__ __forceinline__ uint32_t s_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void bar_init(uint64_t *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(s_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void bar_expect_tx(uint64_t *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(s_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(s_u32(bar)) : "memory");
}
__device__ __forceinline__ void bar_wait(uint64_t *bar, unsigned parity) {
    uint32_t ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok)
                     : "r"(s_u32(bar)), "r"(parity)
                     : "memory");
    } while (!ok);
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(s_u32(dst)),
                 "l"(src), "r"(bytes), "r"(s_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void *src, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
// 16 bytes global -> shared, asynchronously, bypassing L1 (no reuse on this SM)
__device__ __forceinline__ void cp16(const float4 *dst_smem, const float4 *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s_u32(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ void zero_acc(CVec<2> (&acc)[12]) {
#pragma unroll
    for (int c = 0; c < 12; c++) acc[c] = czero<2>();
}

// Byte sizes of the shared-memory regions for a layout block of XB sites and NP RHS pairs.
struct SweepSmem {
    uint32_t RB, GO, GW, GROW;              // tile row, own links of a row, one link window, all links of one row
    uint32_t I_BYTES, G_BYTES;              // per buffer (two buffers each)
    uint32_t H_BYTES, XH_BYTES;             // thread-private halo slots: y and z (every thread), x (edge threads)
    uint32_t C_BYTES;                       // packed clover blocks of the tile rows (fused M_ooee epilogue), per buffer
    uint32_t off_G, off_H, off_XH, off_C, off_bar, total;
    __host__ __device__ SweepSmem(int XB, int NP) {
        RB = 12u * XB * NP * 16u;
        GO = 18u * XB * 16u;
        GW = 5u * XB * 16u;
        GROW = GO + 5u * GW;
        I_BYTES = ROWS * RB;
        G_BYTES = ROWS * GROW;
        H_BYTES = 2u * ROWS * RB;           // 2 slots x 12 components x (ROWS XB NP) threads x 16 bytes
        XH_BYTES = 2u * ROWS * 12u * NP * 16u;
        off_G = 2u * I_BYTES;
        off_H = off_G + 2u * G_BYTES;
        off_XH = off_H + H_BYTES;
        C_BYTES = ROWS * GO;
        off_C = off_XH + XH_BYTES;
        off_bar = off_C + 2u * C_BYTES;
        total = off_bar + 64u;
    }
};

// A neighbour's position in shared memory, in float4 units: component 0 of this thread's element, what to add
// for buffer 1, and the component stride.
struct Nbr {
    int o, bs, cs;
};

// out = C in for the two packed Hermitian 6x6 blocks of one site (6 real diagonals + 15 complex lower-triangle entries
// each, reading S7); pc: float4 0 of the site's 72 packed floats (stride XB), broadcast reads from shared memory
__device__ __forceinline__ void clover_mul(const float4 *pc, int XB, const CVec<2> (&in)[12], CVec<2> (&out)[12]) {
#pragma unroll
    for (int ch = 0; ch < 2; ch++) {
        float a[36];
#pragma unroll
        for (int j = 0; j < 9; j++) {
            const float4 v = pc[(9 * ch + j) * XB];
            a[4 * j] = v.x; a[4 * j + 1] = v.y; a[4 * j + 2] = v.z; a[4 * j + 3] = v.w;
        }
#pragma unroll
        for (int i = 0; i < 6; i++) {
            CVec<2> v = rmul(a[i], in[6 * ch + i]);
#pragma unroll
            for (int j = 0; j < 6; j++) {
                if (j < i) v = cfma(a[6 + 2 * (i * (i - 1) / 2 + j)], a[6 + 2 * (i * (i - 1) / 2 + j) + 1], in[6 * ch + j], v);
                else if (j > i) v = cfma_conj(a[6 + 2 * (j * (j - 1) / 2 + i)], a[6 + 2 * (j * (j - 1) / 2 + i) + 1], in[6 * ch + j], v);
            }
            out[6 * ch + i] = v;
        }
    }
}

// EPI, what happens to the hopping sum H before it is stored (the clover blocks of the output sites come in with the links):
//   0: out = H                                  D_hop, M_eooe
//   1: out = C H                                 M_ooee M_eooe, the first two steps of the Schur sequence (row a7), checkerboarded
//   2: out = C in - H / 2                        the full Wilson-clover matrix M (reading S6), full lattice: the centre
//                                                slice holds in(x) itself, so C in(x) is formed first and the hops add to it
template <int XB_, int NP_, bool CB, int EPI>
__global__ void __launch_bounds__(224, 1)
hop_sweep_kernel(const SweepParams p, const float4 *__restrict__ in, float4 *__restrict__ out) {
    const int XB = XB_ ? XB_ : p.XB;
    const int NP = NP_ ? NP_ : p.NP;
    const int cs = XB * NP;
    const SweepSmem L(XB, NP);
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + L.off_bar);
    uint64_t *fullI = bars, *freeI = bars + 2, *freeG = bars + 4, *fullG = bars + 6;

    constexpr bool CLOV = EPI != 0;
    static_assert(EPI == 0 || (EPI == 1 && CB) || (EPI == 2 && !CB), "fused epilogues: C H on checkerboarded fields, C in - H/2 on the full lattice");
    const int tid = threadIdx.x;
    const int NC = ROWS * cs, NCpad = (NC + 31) & ~31;
    const int Y = p.Y, Z = p.Z, T = p.T, nxb = p.nxb, lt = p.lt;

    // block -> (x-block, tile, t-segment): x-blocks fastest, then the tiles of a chunk, then segments, then chunks
    uint32_t xb, yc, zc, seg, chy, chz, q0;
    p.d_nxb.divmod(blockIdx.x, q0, xb);
    p.d_cy.divmod(q0, q0, yc);
    p.d_cz.divmod(q0, q0, zc);
    p.d_ntseg.divmod(q0, q0, seg);
    p.d_ncy.divmod(q0, chz, chy);
    const int y0 = (int)(chy * p.cy + yc) * BY, z0 = (int)(chz * p.cz + zc) * BZ, t0 = (int)seg * lt;

    if (tid == 0) {
        bar_init(&fullI[0], 1); bar_init(&fullI[1], 1);
        bar_init(&freeI[0], NC); bar_init(&freeI[1], NC);
        bar_init(&freeG[0], NC); bar_init(&freeG[1], NC);
        bar_init(&fullG[0], 1); bar_init(&fullG[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    auto tw = [&](int j) { int t = (t0 + j) % T; return t < 0 ? t + T : t; };
    auto blk = [&](int xbb, int y, int z, int t) -> size_t { return (size_t)xbb + (size_t)nxb * (y + (size_t)Y * (z + (size_t)Z * t)); };
    auto wrap = [](int v, int n) { return v < 0 ? v + n : (v >= n ? v - n : v); };
    const int xbm = xb == 0 ? nxb - 1 : (int)xb - 1, xbp = (int)xb + 1 == nxb ? 0 : (int)xb + 1;

    if (tid >= NCpad) {
        // ------------------------------------------------------------------ producer warp
        // slice j of the segment (j = -1 .. lt): the tile rows; for 0 <= j < lt also the links; for j = -1 the t-links
        const int lane = tid - NCpad;
        auto issue_rows = [&](int j) {
            const int t = tw(j);
            const uint32_t b = (uint32_t)(j + 1) & 1u;
            const bool mid = j >= 0 && j < lt;
            if (lane == 0) bar_expect_tx(&fullI[b], L.I_BYTES);
            __syncwarp();
            unsigned char *Ib = smem + b * L.I_BYTES;
            if (lane < ROWS) {
                const int ty = lane % BY, tz = lane / BY;
                bulk_g2s(Ib + lane * L.RB, in + blk(xb, y0 + ty, z0 + tz, t) * 12 * cs, L.RB, &fullI[b]);
            }
            // ask for the rows of a later slice to be brought into L2 now, so that their copy hits L2
            const int jp = j + p.pf;
            if (p.pf > 0 && jp <= lt && lane < 2 * ROWS) {
                const int r = lane % ROWS, tp = tw(jp);
                const size_t bb = blk(xb, y0 + r % BY, z0 + r / BY, tp);
                if (lane < ROWS) bulk_prefetch_l2(in + bb * 12 * cs, L.RB);
                else if (jp < lt) bulk_prefetch_l2(p.gauge_out + bb * kSiteF4 * XB, L.GO);
            }
        };
        auto issue_links = [&](int j) {
            const int t = tw(j);
            const uint32_t b = (uint32_t)(j + 1) & 1u;
            const bool mid = j >= 0 && j < lt;
            constexpr int NG = CB ? 6 : 4;   // link copies per row: on the full lattice U_x and U_t of the input row are the own links
            unsigned char *Gb = smem + L.off_G + b * L.G_BYTES;
            if (mid || j == -1) {
                if (lane == 0) bar_expect_tx(&fullG[b], mid ? ROWS * (L.GO + (NG - 1) * L.GW + (CLOV ? L.GO : 0u)) : ROWS * (CB ? L.GW : L.GO));
                __syncwarp();
                for (int idx = lane; idx < ROWS * 6; idx += 32) {
                    const int r = idx / 6, w = idx - r * 6;
                    if (!CB && (w == 1 || w == 5)) continue;
                    if (j == -1 && w != (CB ? 5 : 0)) continue;
                    const int y = y0 + r % BY, z = z0 + r / BY;
                    unsigned char *dst = Gb + r * L.GROW;
                    const float4 *src;
                    uint32_t bytes = L.GW;
                    switch (w) {
                        case 0: src = p.gauge_out + blk(xb, y, z, t) * kSiteF4 * XB; bytes = L.GO; break;                       // own links
                        case 1: src = p.gauge_in + blk(xb, y, z, t) * kSiteF4 * XB; dst += L.GO; break;                        // U_x at the -x neighbours in this x-block
                        case 2: src = p.gauge_in + blk(xbm, y, z, t) * kSiteF4 * XB; dst += L.GO + L.GW; break;                // ... and in the x-block before it
                        case 3: src = p.gauge_in + (blk(xb, wrap(y - 1, Y), z, t) * kSiteF4 + 4) * XB; dst += L.GO + 2 * L.GW; break;   // U_y at y-1
                        case 4: src = p.gauge_in + (blk(xb, y, wrap(z - 1, Z), t) * kSiteF4 + 9) * XB; dst += L.GO + 3 * L.GW; break;   // U_z at z-1
                        default: src = p.gauge_in + (blk(xb, y, z, t) * kSiteF4 + 13) * XB; dst += L.GO + 4 * L.GW; break;     // U_t of the input row (carry)
                    }
                    bulk_g2s(dst, src, bytes, &fullG[b]);
                }
                if (CLOV && mid && lane >= 32 - ROWS) {
                    const int r = lane - (32 - ROWS);
                    bulk_g2s(smem + L.off_C + b * L.C_BYTES + r * L.GO, p.clover + blk(xb, y0 + r % BY, z0 + r / BY, t) * kSiteF4 * XB, L.GO, &fullG[b]);
                }
            }
        };
        issue_rows(-1); issue_links(-1);
        issue_rows(0); issue_links(0);
        for (int k = -1; k + 2 <= lt; k++) {
            const uint32_t par = ((uint32_t)(k + 1) >> 1) & 1u;
            bar_wait(&freeI[(k + 1) & 1], par);   // the consumers are done with the rows of slice k (after its x hops)
            issue_rows(k + 2);
            bar_wait(&freeG[(k + 1) & 1], par);   // ... and with its links (end of the step)
            issue_links(k + 2);
        }
        return;
    }
    if (tid >= NC) return;

    // ---------------------------------------------------------------------- consumers
    int q = tid / NP;
    const int pair = tid - q * NP;
    const int r = q / XB, xin = q - r * XB;
    const int ty = r % BY, tz = r / BY;
    const int y = y0 + ty, z = z0 + tz;
    const float4 *S = reinterpret_cast<const float4 *>(smem);
    const int IB4 = L.I_BYTES / 16, G4 = L.G_BYTES / 16;
    const int oH = L.off_H / 16, oXH = L.off_XH / 16;
    const int e = xin * NP + pair;                    // this thread's element inside a row component
    const int rowlen = 12 * cs;
    // private halo slots: [y | z][component][thread], and for the edge sites of a row [side][row][component][pair]
    const Nbr hy = {oH + tid, 0, NC}, hz = {oH + 12 * NC + tid, 0, NC};
    const Nbr hxp = {oXH + ((ROWS + r) * 12) * NP + pair, 0, NP}, hxm = {oXH + (r * 12) * NP + pair, 0, NP};
    const bool edge_p = xin + 1 == XB, edge_m = xin == 0;
    const Nbr own = {r * rowlen + e, IB4, cs};
    const Nbr yp = ty + 1 < BY ? Nbr{(r + 1) * rowlen + e, IB4, cs} : hy;
    const Nbr ym = ty > 0 ? Nbr{(r - 1) * rowlen + e, IB4, cs} : hy;
    const Nbr zp = tz + 1 < BZ ? Nbr{(r + BY) * rowlen + e, IB4, cs} : hz;
    const Nbr zm = tz > 0 ? Nbr{(r - BY) * rowlen + e, IB4, cs} : hz;
    const Nbr xps = edge_p ? hxp : Nbr{r * rowlen + e + NP, IB4, cs};
    const Nbr xms = edge_m ? hxm : Nbr{r * rowlen + e - NP, IB4, cs};
    // where the halo neighbours live in global memory (slice 0; one slice further is st elements on)
    const size_t st = (size_t)nxb * Y * Z * 12 * cs;
    const float4 *gy = in + blk(xb, ty == 0 ? wrap(y - 1, Y) : wrap(y + 1, Y), z, 0) * 12 * cs + e;
    const float4 *gz = in + blk(xb, y, tz == 0 ? wrap(z - 1, Z) : wrap(z + 1, Z), 0) * 12 * cs + e;
    const float4 *gxp = in + blk(xbp, y, z, 0) * 12 * cs + pair;                      // site 0 of the next x-block
    const float4 *gxm = in + blk(xbm, y, z, 0) * 12 * cs + (XB - 1) * NP + pair;      // last site of the previous one
    // refill of a private slot for slice tn (every thread for itself)
    auto refill = [&](const Nbr &slot, const float4 *g, int tn, bool on) {
        if (on) {
            const float4 *src = g + st * tn;
#pragma unroll
            for (int c = 0; c < 12; c++) cp16(S + slot.o + c * slot.cs, src + (size_t)c * cs);
        }
    };
    auto refill_x = [&](int tn, bool active) {
        const int s = (p.out_parity + y + z + tn) & 1;
        refill(hxp, gxp, tn, active && edge_p && (!CB || s == 1));
        refill(hxm, gxm, tn, active && edge_m && (!CB || s == 0));
        cp_commit();
    };
    // links (float4 units): row r of the link buffer; windows are addressed through the base of a virtual 18-row site
    const int Gr = (int)(L.off_G / 16) + r * (int)(L.GROW / 16);
    const int g_own = Gr + xin;
    const int g_bx_same = CB ? Gr + 18 * XB + xin : g_own;
    const int g_bx_step = edge_m ? Gr + 23 * XB + XB - 1 : (CB ? Gr + 18 * XB + xin - 1 : g_own - 1);
    const int g_by = Gr + 28 * XB - 4 * XB + xin;
    const int g_bz = Gr + 33 * XB - 9 * XB + xin;
    const int g_bt = CB ? Gr + 38 * XB - 13 * XB + xin : g_own;

    CVec<2> acc[12];
    CVec<2> carry[6];      // (1 + gamma_t) U_t^+ psi of the slice before, as a half spinor
    HopOperands<2> A, B;

    // slice 0's halo neighbours: three groups in the order they are waited for (y, z, x)
    {
        const int tn = tw(0);
        refill(hy, gy, tn, true); cp_commit();
        refill(hz, gz, tn, true); cp_commit();
        refill_x(tn, true);
    }

#pragma unroll 1
    for (int k = -1; k < lt; k++) {
        const int t = tw(k);
        const uint32_t b = (uint32_t)(k + 1) & 1u;
        bar_wait(&fullI[b], ((uint32_t)(k + 1) >> 1) & 1u);
        bar_wait(&fullG[b], ((uint32_t)(k + 1) >> 1) & 1u);   // links of slice k, on their own barrier: the +t hop below waits for rows only
        const float4 *G = S + b * G4;
        const float4 *pc = S + L.off_C / 16 + b * (L.C_BYTES / 16) + r * (18 * XB) + xin;   // this site's clover blocks
        if (k >= 0) {
            if constexpr (EPI == 2) {
                // acc = -2 C in(x): the hops below add H, and the store scales by -1/2
                CVec<2> own_psi[12], cpsi[12];
#pragma unroll
                for (int c = 0; c < 12; c++) own_psi[c] = to_cvec(S[own.o + b * own.bs + c * own.cs]);
                clover_mul(pc, XB, own_psi, cpsi);
#pragma unroll
                for (int c = 0; c < 12; c++) acc[c] = rmul(-2.f, cpsi[c]);
            } else {
                zero_acc(acc);
            }
            hop_recon<2, 3, false>(carry, acc);
        }
        if (k + 1 < lt) {
            // -t hop of the next slice, first thing, so that the rows of this slice can be released after the x hops:
            // (1 + gamma_t) U_t(x, t)^+ psi(x, t), both at this thread's own position of slice k
            hop_load_s<3>(B, S + own.o + b * own.bs, own.cs, G + g_bt, XB);
            hop_half<2, 3, false>(B, carry);
        }
        if (k >= 0) {
            const int tn = tw(k + 1);
            const bool more = k + 1 < lt;
            // x neighbours of this step (checkerboarded lines alternate with t)
            Nbr xp = xps, xm = xms;
            int g_bx = g_bx_step;
            if (CB) {
                const int s = (p.out_parity + y + z + t) & 1;
                if (s) { xm = own; g_bx = g_bx_same; }
                else xp = own;
            }
            cp_wait<2>();                      // this thread's y slot holds slice k
            hop_load_s<1>(A, S + yp.o + b * yp.bs, yp.cs, G + g_own, XB);
            hop_load_s<1>(B, S + ym.o + b * ym.bs, ym.cs, G + g_by, XB);
            hop_compute<2, 1, true >(A, acc);
            refill(hy, gy, tn, more); cp_commit();
            cp_wait<2>();                      // z slot
            hop_load_s<2>(A, S + zp.o + b * zp.bs, zp.cs, G + g_own, XB);
            hop_compute<2, 1, false>(B, acc);
            hop_load_s<2>(B, S + zm.o + b * zm.bs, zm.cs, G + g_bz, XB);
            hop_compute<2, 2, true >(A, acc);
            refill(hz, gz, tn, more); cp_commit();
            cp_wait<2>();                      // x slot
            hop_load_s<0>(A, S + xp.o + b * xp.bs, xp.cs, G + g_own, XB);
            hop_compute<2, 2, false>(B, acc);
            hop_load_s<0>(B, S + xm.o + b * xm.bs, xm.cs, G + g_bx, XB);
            hop_compute<2, 0, true >(A, acc);
            refill_x(tn, more);
            hop_compute<2, 0, false>(B, acc);
            bar_arrive(&freeI[b]);             // rows of slice k are no longer read: slice k+2 may land
            bar_wait(&fullI[b ^ 1u], ((uint32_t)(k + 2) >> 1) & 1u);   // slice k+1
            hop_load_s<3>(A, S + own.o + (b ^ 1u) * own.bs, own.cs, G + g_own, XB);
            hop_compute<2, 3, true >(A, acc);
            float4 *o = out + (blk(xb, y, z, t) * 12 * XB + xin) * NP + pair;
            if constexpr (EPI == 1) {
                CVec<2> res[12];
                clover_mul(pc, XB, acc, res);
#pragma unroll
                for (int c = 0; c < 12; c++) __stcs(&o[(size_t)c * cs], from_cvec(res[c]));
            } else if constexpr (EPI == 2) {
#pragma unroll
                for (int c = 0; c < 12; c++) __stcs(&o[(size_t)c * cs], from_cvec(rmul(-0.5f, acc[c])));
            } else {
#pragma unroll
                for (int c = 0; c < 12; c++) __stcs(&o[(size_t)c * cs], from_cvec(acc[c]));
            }
        } else {
            bar_arrive(&freeI[b]);
        }
        bar_arrive(&freeG[b]);
    }
    cp_wait<0>();
}

}  // namespace

// ------------------------------------------------------------------ host side
bool sweep_supported(const FieldGeom &g) {
    if (g.N & 1) return false;                       // RHS pairs in FFMA2 lanes; bulk copies need 16-byte pieces
    if (g.Y < 2 || g.Z < 2 || (g.Y % BY) || (g.Z % BZ)) return false;
    const int np = threads_per_site(g.N);
    if (g.XB * np > 48) return false;                // 4 rows of consumers + the producer warp fit 224 threads
    const SweepSmem L(g.XB, np);
    return L.total <= 227u * 1024u;
}

SweepTiling default_sweep_tiling(const FieldGeom &g, int num_sms) {
    SweepTiling t = {g.T, 1, 1};
    const int nty = g.Y / BY, ntz = g.Z / BZ;
    // chunk: the tiles that run at the same time (one thread block per SM) should form a compact patch of the
    // (y,z) plane, so that most halo rows are another resident block's tile rows and come from L2
    long long best_n = 0;
    double best_shape = 1e30;
    for (int cy = 1; cy <= nty; cy++) {
        if (nty % cy) continue;
        for (int cz = 1; cz <= ntz; cz++) {
            if (ntz % cz) continue;
            const long long n = (long long)g.nxb * cy * cz;
            if (n > num_sms && !(cy == 1 && cz == 1)) continue;
            const double shape = 1.0 / (cy * BY) + 1.0 / (cz * BZ);
            if (n > best_n || (n == best_n && shape < best_shape)) { best_n = n; best_shape = shape; t.cy = cy; t.cz = cz; }
        }
    }
    // segment length: the whole t-line as long as that leaves two blocks per SM to balance the tail (every segment
    // pays two extra slice loads, measured slower whenever the line fits); shorter segments only for small lattices
    const long long tiles = (long long)g.nxb * nty * ntz;
    int pick = 0;
    for (int lt = g.T; lt >= 1; lt--) {
        if (g.T % lt) continue;
        if (tiles * (g.T / lt) >= 2ll * num_sms) { pick = lt; break; }
    }
    if (pick < 4) {
        pick = g.T;
        for (int lt = 4; lt <= g.T; lt++)
            if (g.T % lt == 0) { pick = lt; break; }
    }
    t.lt = pick;
    return t;
}

bool build_sweep_params(const FieldGeom &g, int out_parity, const SweepTiling &t, SweepParams &p) {
    if (!sweep_supported(g)) return false;
    if (t.lt < 1 || g.T % t.lt || t.cy < 1 || t.cz < 1) return false;
    const int nty = g.Y / BY, ntz = g.Z / BZ;
    if (nty % t.cy || ntz % t.cz) return false;
    const int np = threads_per_site(g.N);
    const long long grid = (long long)g.nxb * nty * ntz * (g.T / t.lt);
    if (grid >= (1ll << 31)) return false;
    p.Y = g.Y; p.Z = g.Z; p.T = g.T;
    p.XB = g.XB; p.nxb = g.nxb; p.NP = np;
    p.cb = g.cb; p.out_parity = out_parity;
    p.lt = t.lt; p.ntseg = g.T / t.lt;
    p.cy = t.cy; p.cz = t.cz;
    bool ok = true;
    ok &= make_fastdiv(g.nxb, grid, p.d_nxb);
    ok &= make_fastdiv(t.cy, grid, p.d_cy);
    ok &= make_fastdiv(t.cz, grid, p.d_cz);
    ok &= make_fastdiv(p.ntseg, grid, p.d_ntseg);
    ok &= make_fastdiv(nty / t.cy, grid, p.d_ncy);
    if (!ok) return false;
    p.gauge_out = p.gauge_in = nullptr;
    p.clover = nullptr;
    p.pf = 2;
    p.consumers = (unsigned)(ROWS * g.XB * np);
    p.threads = ((p.consumers + 31u) & ~31u) + 32u;
    p.grid = (unsigned)grid;
    p.smem_bytes = SweepSmem(g.XB, np).total;
    return true;
}

#define MRHS_SWEEP_LIST(F) F(8, 6) F(6, 6) F(4, 12) F(2, 24) F(16, 2) F(12, 2) F(0, 0)

mrhs_status_t sweep_prepare() {
    const int max_smem = 227 * 1024;
#define MRHS_CASE(XB, NP)                                                                                                     \
    MRHS_CUDA(cudaFuncSetAttribute(hop_sweep_kernel<XB, NP, false, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem)); \
    MRHS_CUDA(cudaFuncSetAttribute(hop_sweep_kernel<XB, NP, true, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem));  \
    MRHS_CUDA(cudaFuncSetAttribute(hop_sweep_kernel<XB, NP, true, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem));  \
    MRHS_CUDA(cudaFuncSetAttribute(hop_sweep_kernel<XB, NP, false, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem));
    MRHS_SWEEP_LIST(MRHS_CASE)
#undef MRHS_CASE
    return MRHS_OK;
}

namespace {
template <int XB, int NP>
void launch_sweep_t(const SweepParams &p, const void *d_in, void *d_out, cudaStream_t st) {
    if (p.cb && p.clover) hop_sweep_kernel<XB, NP, true, 1><<<p.grid, p.threads, p.smem_bytes, st>>>(p, (const float4 *)d_in, (float4 *)d_out);
    else if (p.cb)        hop_sweep_kernel<XB, NP, true, 0><<<p.grid, p.threads, p.smem_bytes, st>>>(p, (const float4 *)d_in, (float4 *)d_out);
    else if (p.clover)    hop_sweep_kernel<XB, NP, false, 2><<<p.grid, p.threads, p.smem_bytes, st>>>(p, (const float4 *)d_in, (float4 *)d_out);
    else                  hop_sweep_kernel<XB, NP, false, 0><<<p.grid, p.threads, p.smem_bytes, st>>>(p, (const float4 *)d_in, (float4 *)d_out);
}
}  // namespace

mrhs_status_t launch_sweep(const SweepParams &p, const void *d_in, void *d_out, cudaStream_t st) {
    switch (p.XB * 1000 + p.NP) {
        case 8006:  launch_sweep_t<8, 6>(p, d_in, d_out, st); break;     // N = 12
        case 6006:  launch_sweep_t<6, 6>(p, d_in, d_out, st); break;     // N = 12, 24^4 checkerboarded
        case 4012:  launch_sweep_t<4, 12>(p, d_in, d_out, st); break;    // N = 24
        case 2024:  launch_sweep_t<2, 24>(p, d_in, d_out, st); break;    // N = 48
        case 16002: launch_sweep_t<16, 2>(p, d_in, d_out, st); break;    // N = 4
        case 12002: launch_sweep_t<12, 2>(p, d_in, d_out, st); break;    // N = 4
        default:    launch_sweep_t<0, 0>(p, d_in, d_out, st); break;
    }
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

}  // namespace mrhs

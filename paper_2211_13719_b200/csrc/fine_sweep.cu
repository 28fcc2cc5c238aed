// fine_sweep.cu -- slice-sweep kernel of the fine-level hopping term:
//   out(x) = sum_mu (1-gamma_mu) U_mu(x) in(x+mu) + (1+gamma_mu) U_mu(x-mu)^+ in(x-mu)
// (reading S3) for N_rhs right-hand sides at once, D_hop and M_eooe from one body with
// different index maps ("different site ordering").
//
// A thread block owns a tile of XB x 2 x 2 sites in (x,y,z) and sweeps a segment of t.  Every operand of a
// step (one t-slice of the tile) is staged in shared memory once, by a producer warp, with TMA bulk copies that
// complete on mbarriers:
//   * the four tile rows (double buffered: the +t hop reads the next slice, which is the next centre slice);
//   * the eight halo rows in y and z (the rows of the neighbouring tiles; single buffered, released right after
//     the y / z hops so that they are refilled while the rest of the step runs);
//   * the links of the output sites and 640-byte windows of the backward links (double buffered), and for the
//     fused epilogues the packed clover blocks;
//   * only the x halo (one site on each side of the x-block) is fetched by the threads themselves, with 16-byte
//     cp.async into slots that only the fetching thread reads.
// The -t hop of slice s+1 is computed while slice s is the centre and carried in registers as a half spinor,
// so no slice is loaded twice along t.
//
// Work split: a "unit" is one site and one pair of right-hand sides (the two lanes of FFMA2 / FADD2, links are
// the broadcast scalar operand).  The two half-warps of a warp split a unit by the spin row of the projected
// half spinor: lanes 0-15 own h_0, lanes 16-31 own h_1 of the same sixteen units.  Each computes its row of
// (1 -+ gamma_mu) psi, the SU(3) product on it and its share of the reconstruction (9 complex accumulators instead
// of 12), and the halves meet in warp shuffles before the store.  The code is the same for both halves: which
// spin rows a lane reads is an address offset, and the two sign flips that depend on the spin row are the
// scalar operand e = +-1 of an FFMA2 that replaces an FADD2.  Twelve consumer warps per block (three per SM
// sub-partition) instead of six with twice the registers: balanced sub-partitions and enough warps to cover
// shared-memory latency without register double buffering.
#include "fine_sweep.cuh"
#include "async_copy.cuh"
#include "hop_math.cuh"

#include <algorithm>
#include <queue>
#include <vector>

namespace mrhs {

namespace {

constexpr int BY = kSweepBY, BZ = kSweepBZ, ROWS = kSweepRows;
static_assert(BY == 2 && BZ == 2, "every tile row has exactly one halo row in y and one in z");

// Byte sizes of the shared-memory regions for a layout block of XB sites and NP RHS pairs.
struct SweepSmem {
    uint32_t RB, GO, GW, GBK, GROW;         // tile row, own links of a row, one link window, backward links of a row (checkerboarded), all links of one row
    uint32_t I_BYTES, G_BYTES;              // per buffer (two buffers each)
    uint32_t H_BYTES, XH_BYTES;             // halo rows in y and z (ROWS each); x halo slots [side][row][component][pair]
    uint32_t C_BYTES;                       // packed clover blocks of the tile rows (fused epilogues), per buffer
    uint32_t off_G, off_H, off_XH, off_C, off_bar, total;
    __host__ __device__ SweepSmem(int XB, int NP, bool clov, bool cb) {
        RB = 12u * XB * NP * 16u;
        GO = 18u * XB * 16u;
        GW = 5u * XB * 16u;
        GBK = (uint32_t)kBackF4 * XB * 16u;
        // full lattice: the backward links are other sites' own links, three windows of them (x-block before, y-1, z-1);
        // checkerboarded: the packed backward links of the row (fine_sweep.cuh)
        GROW = cb ? GO + GBK : GO + 3u * GW;
        I_BYTES = ROWS * RB;
        G_BYTES = ROWS * GROW;
        H_BYTES = 2u * ROWS * RB;
        XH_BYTES = 2u * ROWS * 12u * NP * 16u;
        off_G = 2u * I_BYTES;
        off_H = off_G + 2u * G_BYTES;
        off_XH = off_H + H_BYTES;
        C_BYTES = clov ? ROWS * GO : 0u;
        off_C = off_XH + XH_BYTES;
        off_bar = off_C + 2u * C_BYTES;
        total = off_bar + 128u;
    }
};

__device__ __forceinline__ CVec<2> shfl_half(CVec<2> v) {
    CVec<2> r;
    r.re.v = __shfl_xor_sync(0xffffffffu, v.re.v, 16);
    r.im.v = __shfl_xor_sync(0xffffffffu, v.im.v, 16);
    return r;
}
__device__ __forceinline__ CVec<2> csel(bool take_a, CVec<2> a, CVec<2> b) {
    CVec<2> r;
    r.re.v = take_a ? a.re.v : b.re.v;
    r.im.v = take_a ? a.im.v : b.im.v;
    return r;
}

// Operands of one hop for this lane: its own spin row of the neighbour (ps), the partner row the projector
// combines it with (pp), and the link.
struct SplitOperands {
    float4 ps[3], pp[3];
    float u[18];
};

// nb: component 0 of the neighbour's element for this unit; os / op: offsets of colour 0 of the two spin rows; st: component
// stride; g: float4 0 of the link's site data
template <int MU, int LMU = MU>
__device__ __forceinline__ void split_load(SplitOperands &o, const float4 *nb, int os, int op, int st, const float4 *g, int XB) {
#pragma unroll
    for (int c = 0; c < 3; c++) {
        o.ps[c] = nb[os + c * st];
        o.pp[c] = nb[op + c * st];
    }
    load_link_s<LMU>(g, XB, o.u);
}

// This lane's row of the projected half spinor and of r = U h (FWD) or U^+ h.  Spin row s (e = +1 for s = 0, -1 for s = 1):
//   x: h_s = psi_s + S i psi_{3-s}     y: h_s = psi_s + e S psi_{3-s}     z: h_s = psi_s + e S i psi_{2+s}     t: h_s = psi_s - S psi_{2+s}
// with S = +1 for the forward hop (reading S2/S3, the rows of hop_half in hop_math.cuh).  d = +1: the operator as written;
// d = -1: its adjoint (gamma_5 D_hop gamma_5: S -> -S in projection and reconstruction, links unchanged); ed = e d.
// Every sign is the scalar operand of an FFMA2 (a * (+-1) is exact), so both variants cost the same.
template <int MU, bool FWD>
__device__ __forceinline__ void split_half(const SplitOperands &o, float d, float ed, CVec<2> (&r)[3]) {
    const float sg = (MU == 1 || MU == 2) ? (FWD ? ed : -ed) : (FWD ? d : -d);
    CVec<2> h[3];
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const CVec<2> a = to_cvec(o.ps[c]), b = to_cvec(o.pp[c]);
        if constexpr (MU == 0 || MU == 2) { h[c].re = sfnma(sg, b.im, a.re); h[c].im = sfma(sg, b.re, a.im); }
        else if constexpr (MU == 1) h[c] = rfma(sg, b, a);
        else h[c] = rfma(-sg, b, a);
    }
    const float (&u)[18] = o.u;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        if constexpr (FWD) {
            CVec<2> t = cmul(u[2 * (3 * c + 0)], u[2 * (3 * c + 0) + 1], h[0]);
            t = cfma(u[2 * (3 * c + 1)], u[2 * (3 * c + 1) + 1], h[1], t);
            r[c] = cfma(u[2 * (3 * c + 2)], u[2 * (3 * c + 2) + 1], h[2], t);
        } else {
            CVec<2> t = cmul_conj(u[2 * (0 + c)], u[2 * (0 + c) + 1], h[0]);
            t = cfma_conj(u[2 * (3 + c)], u[2 * (3 + c) + 1], h[1], t);
            r[c] = cfma_conj(u[2 * (6 + c)], u[2 * (6 + c) + 1], h[2], t);
        }
    }
}

// This lane's share of the reconstruction: up (output spin row s) += r; the lower rows get
//   x: out_{3-s} -= S i r     y: out_{3-s} += e S r     (accumulated in la)
//   z: out_{2+s} -= e S i r   t: out_{2+s} -= S r       (accumulated in lb)
// For the adjoint (d = -1) S changes sign.  lb is kept as d times its true value, so that the z and t updates do not depend
// on d (d d = 1) and the -t carry enters with +1; whoever reads lb multiplies it by d (one FFMA2 in place of an FADD2).
template <int MU, bool FWD>
__device__ __forceinline__ void split_recon(const CVec<2> (&r)[3], float d, float e, float ed, CVec<2> (&up)[3], CVec<2> (&la)[3], CVec<2> (&lb)[3]) {
    const float sg = MU == 1 ? (FWD ? ed : -ed) : MU == 2 ? (FWD ? e : -e) : (FWD ? d : -d);
#pragma unroll
    for (int c = 0; c < 3; c++) {
        up[c] = cadd(up[c], r[c]);
        if constexpr (MU == 0) { la[c].re = sfma(sg, r[c].im, la[c].re); la[c].im = sfnma(sg, r[c].re, la[c].im); }
        else if constexpr (MU == 1) la[c] = rfma(sg, r[c], la[c]);
        else if constexpr (MU == 2) { lb[c].re = sfma(sg, r[c].im, lb[c].re); lb[c].im = sfnma(sg, r[c].re, lb[c].im); }
        else lb[c] = FWD ? csub(lb[c], r[c]) : cadd(lb[c], r[c]);
    }
}

template <int MU, bool FWD>
__device__ __forceinline__ void split_hop(const SplitOperands &o, float d, float e, float ed, CVec<2> (&up)[3], CVec<2> (&la)[3], CVec<2> (&lb)[3]) {
    CVec<2> r[3];
    split_half<MU, FWD>(o, d, ed, r);
    split_recon<MU, FWD>(r, d, e, ed, up, la, lb);
}

// out = C v for ONE packed Hermitian 6x6 block (6 real diagonals + 15 complex lower-triangle entries, reading S7);
// pc: float4 0 of the block for this site (stride XB), broadcast reads from shared memory
__device__ __forceinline__ void clover_block_mul(const float4 *pc, int XB, const CVec<2> (&v)[6], CVec<2> (&out)[6]) {
    float a[36];
#pragma unroll
    for (int j = 0; j < 9; j++) {
        const float4 w = pc[j * XB];
        a[4 * j] = w.x; a[4 * j + 1] = w.y; a[4 * j + 2] = w.z; a[4 * j + 3] = w.w;
    }
#pragma unroll
    for (int i = 0; i < 6; i++) {
        CVec<2> t = rmul(a[i], v[i]);
#pragma unroll
        for (int j = 0; j < 6; j++) {
            if (j < i) t = cfma(a[6 + 2 * (i * (i - 1) / 2 + j)], a[6 + 2 * (i * (i - 1) / 2 + j) + 1], v[j], t);
            else if (j > i) t = cfma_conj(a[6 + 2 * (j * (j - 1) / 2 + i)], a[6 + 2 * (j * (j - 1) / 2 + i) + 1], v[j], t);
        }
        out[i] = t;
    }
}

// EPI, what happens to the hopping sum H before it is stored (the clover blocks of the output sites come in with the links):
//   0: out = H                                  D_hop, M_eooe
//   1: out = C H                                 M_ooee M_eooe, the first two steps of the Schur sequence (row a7), checkerboarded
//   2: out = C in - H / 2                        the full Wilson-clover matrix M (reading S6), full lattice: the centre
//                                                slice in shared memory holds in(x) itself
//   3: out = C aux - H / 4                       second launch of the even-odd preconditioned (Schur complement) operator
//                                                C_e - H_eo C_o^-1 H_oe / 4 (NEXT-2): checkerboarded, aux = the operator's
//                                                input on the output sites, read from global memory
template <int XB_, int NP_, bool CB, int EPI>
__global__ void __launch_bounds__(kSweepMaxThreads, 1)
hop_sweep_kernel(const SweepParams p, const float4 *__restrict__ in, float4 *__restrict__ out) {
    constexpr bool CLOV = EPI != 0;
    static_assert(EPI == 0 || ((EPI == 1 || EPI == 3) && CB) || (EPI == 2 && !CB), "fused epilogues: C H and C aux - H/4 on checkerboarded fields, C in - H/2 on the full lattice");
    const int XB = XB_ ? XB_ : p.XB;
    const int NP = NP_ ? NP_ : p.NP;
    const int cs = XB * NP;                       // units (site, RHS pair) per tile row = elements of one row component
    const int WPR = (cs + 15) >> 4;               // consumer warps per tile row: sixteen units x two spin rows each
    const int NWC = ROWS * WPR;
    const SweepSmem L(XB, NP, CLOV, CB);
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + L.off_bar);
    uint64_t *fullI = bars, *freeI = bars + 2, *fullG = bars + 4, *freeG = bars + 6, *fullH = bars + 8, *freeH = bars + 10;

    const int tid = threadIdx.x, wid = tid >> 5, lane = tid & 31;
    const int Y = p.Y, Z = p.Z, T = p.T, nxb = p.nxb;

    // block -> (x-block, tile, t-segment)
    int xb_i, y0, z0, t0, lt;
    sweep_block_coords(p, blockIdx.x, xb_i, y0, z0, t0, lt);
    const uint32_t xb = (uint32_t)xb_i;

    if (tid == 0) {
        for (int i = 0; i < 2; i++) {
            mbar_init(&fullI[i], 1); mbar_init(&freeI[i], NWC);
            mbar_init(&fullG[i], 2); mbar_init(&freeG[i], NWC);
            mbar_init(&fullH[i], 1); mbar_init(&freeH[i], NWC);
        }
        mbar_fence_init();
    }
    __syncthreads();

    auto tw = [&](int j) { int t = (t0 + j) % T; return t < 0 ? t + T : t; };
    auto blk = [&](int xbb, int y, int z, int t) -> size_t { return (size_t)xbb + (size_t)nxb * (y + (size_t)Y * (z + (size_t)Z * t)); };
    auto wrap = [](int v, int n) { return v < 0 ? v + n : (v >= n ? v - n : v); };
    const int xbm = xb == 0 ? nxb - 1 : (int)xb - 1, xbp = (int)xb + 1 == nxb ? 0 : (int)xb + 1;

    if (wid >= NWC) {
        // ------------------------------------------------------------------ producer warps
        warpgroup_reg_dec<kSweepProducerRegs>();
        // Four warps, each with its own wait / issue loop so that a late release of one region never delays the copies
        // into another: warp NWC the tile rows, NWC + 1 the halo rows, NWC + 2 and NWC + 3 the links of two tile rows each.
        // slice j of the segment (j = -1 .. lt): the tile rows; for 0 <= j < lt also the halo rows and the links; for j = -1 the t-links
        const int role = wid - NWC;
        auto halo_yz = [&](int h, int &yy, int &zz) {      // h < ROWS: y halo of tile row h; else z halo of tile row h - ROWS
            const int r = h % ROWS, ty = r % BY, tz = r / BY;
            yy = y0 + ty; zz = z0 + tz;
            if (h < ROWS) yy = ty == 0 ? wrap(y0 - 1, Y) : wrap(y0 + BY, Y);
            else zz = tz == 0 ? wrap(z0 - 1, Z) : wrap(z0 + BZ, Z);
        };
        if (role == 0) {
            auto issue_rows = [&](int j) {
                const int t = tw(j);
                const uint32_t b = (uint32_t)(j + 1) & 1u;
                if (lane == 0) mbar_expect_tx(&fullI[b], L.I_BYTES);
                __syncwarp();
                if (lane < ROWS) bulk_g2s(smem + b * L.I_BYTES + lane * L.RB, in + blk(xb, y0 + lane % BY, z0 + lane / BY, t) * 12 * cs, L.RB, &fullI[b]);
                // ask for the rows and links of a later slice to be brought into L2 now, so that their copy hits L2
                const int jp = j + p.pf;
                if (p.pf > 0 && jp <= lt && lane >= ROWS && lane < 3 * ROWS) {
                    const int q = lane - ROWS, rr = q % ROWS, tp = tw(jp);
                    const size_t bb = blk(xb, y0 + rr % BY, z0 + rr / BY, tp);
                    if (q < ROWS) bulk_prefetch_l2(in + bb * 12 * cs, L.RB);
                    else if (jp < lt) {
                        bulk_prefetch_l2(p.gauge_out + bb * kSiteF4 * XB, L.GO);
                        if (CB) bulk_prefetch_l2(p.gauge_back + bb * kBackF4 * XB, L.GBK);
                    }
                }
            };
            issue_rows(-1);
            issue_rows(0);
            for (int k = -1; k + 2 <= lt; k++) {
                mbar_wait(&freeI[(k + 1) & 1], ((uint32_t)(k + 1) >> 1) & 1u);   // the consumers are done with the rows of slice k
                issue_rows(k + 2);
            }
        } else if (role == 1) {
            auto issue_halo = [&](int j, int d) {     // d = 0: the y halo rows of slice j, d = 1: the z halo rows
                const int t = tw(j);
                if (lane == 0) mbar_expect_tx(&fullH[d], ROWS * L.RB);
                __syncwarp();
                if (lane < ROWS) {
                    int yy, zz;
                    halo_yz(d * ROWS + lane, yy, zz);
                    bulk_g2s(smem + L.off_H + (d * ROWS + lane) * L.RB, in + blk(xb, yy, zz, t) * 12 * cs, L.RB, &fullH[d]);
                }
                const int jp = j + p.pf;
                if (p.pf > 0 && jp < lt && lane >= ROWS && lane < 2 * ROWS) {
                    int yy, zz;
                    halo_yz(d * ROWS + lane - ROWS, yy, zz);
                    bulk_prefetch_l2(in + blk(xb, yy, zz, tw(jp)) * 12 * cs, L.RB);
                }
            };
            issue_halo(0, 0);
            issue_halo(0, 1);
            for (int k = 0; k + 1 < lt; k++) {
                mbar_wait(&freeH[0], (uint32_t)k & 1u); issue_halo(k + 1, 0);   // the consumers are done with the y hops of slice k
                mbar_wait(&freeH[1], (uint32_t)k & 1u); issue_halo(k + 1, 1);   // ... and with its z hops
            }
        } else {
            // two link warps, tile rows [0, ROWS/2) and [ROWS/2, ROWS): each announces its own bytes on the common barrier
            const int r_lo = (role - 2) * (ROWS / 2);
            auto issue_links = [&](int j) {
                const int t = tw(j);
                const uint32_t b = (uint32_t)(j + 1) & 1u;
                const bool mid = j >= 0 && j < lt;
                unsigned char *Gb = smem + L.off_G + b * L.G_BYTES;
                if (mid || j == -1) {
                    if constexpr (CB) {
                        // per row: the own links and the packed backward links (one contiguous copy each); for slice -1 only the
                        // t-links of the input row, which the carry of the first step needs
                        if (lane == 0) mbar_expect_tx(&fullG[b], mid ? (ROWS / 2) * (L.GO + L.GBK + (CLOV ? L.GO : 0u)) : (ROWS / 2) * L.GW);
                        __syncwarp();
                        if (lane < ROWS) {
                            const int r = r_lo + (lane >> 1), w = lane & 1;
                            const size_t bb = blk(xb, y0 + r % BY, z0 + r / BY, t);
                            unsigned char *dst = Gb + r * L.GROW;
                            if (mid && w == 0) bulk_g2s(dst, p.gauge_out + bb * kSiteF4 * XB, L.GO, &fullG[b]);
                            else if (mid) bulk_g2s(dst + L.GO, p.gauge_back + bb * kBackF4 * XB, L.GBK, &fullG[b]);
                            else if (w == 1) bulk_g2s(dst + L.GO + kBackT * XB * 16, p.gauge_back + (bb * kBackF4 + kBackT) * XB, L.GW, &fullG[b]);
                        }
                    } else {
                        // per row: the own links (U_x and U_t of the input row are own links too) and three windows of other rows'
                        // links; for slice -1 only the own links
                        if (lane == 0) mbar_expect_tx(&fullG[b], mid ? (ROWS / 2) * (L.GO + 3 * L.GW + (CLOV ? L.GO : 0u)) : (ROWS / 2) * L.GO);
                        __syncwarp();
                        if (lane < (ROWS / 2) * 4) {
                            const int r = r_lo + (lane >> 2), w = lane & 3;
                            const int y = y0 + r % BY, z = z0 + r / BY;
                            unsigned char *dst = Gb + r * L.GROW;
                            if (w == 0) bulk_g2s(dst, p.gauge_out + blk(xb, y, z, t) * kSiteF4 * XB, L.GO, &fullG[b]);                                     // own links
                            else if (!mid) {}
                            else if (w == 1) bulk_g2s(dst + L.GO, p.gauge_in + blk(xbm, y, z, t) * kSiteF4 * XB, L.GW, &fullG[b]);                        // U_x in the x-block before
                            else if (w == 2) bulk_g2s(dst + L.GO + L.GW, p.gauge_in + (blk(xb, wrap(y - 1, Y), z, t) * kSiteF4 + 4) * XB, L.GW, &fullG[b]);      // U_y at y-1
                            else bulk_g2s(dst + L.GO + 2 * L.GW, p.gauge_in + (blk(xb, y, wrap(z - 1, Z), t) * kSiteF4 + 9) * XB, L.GW, &fullG[b]);              // U_z at z-1
                        }
                    }
                    if (CLOV && mid && lane >= 32 - ROWS / 2) {
                        const int r = r_lo + lane - (32 - ROWS / 2);
                        bulk_g2s(smem + L.off_C + b * L.C_BYTES + r * L.GO, p.clover + blk(xb, y0 + r % BY, z0 + r / BY, t) * kSiteF4 * XB, L.GO, &fullG[b]);
                    }
                }
            };
            issue_links(-1);
            issue_links(0);
            for (int k = -1; k + 2 < lt; k++) {
                mbar_wait(&freeG[(k + 1) & 1], ((uint32_t)(k + 1) >> 1) & 1u);   // the consumers are done with the links of slice k (end of the step)
                issue_links(k + 2);
            }
        }
        return;
    }

    // ---------------------------------------------------------------------- consumers
    warpgroup_reg_inc<kSweepConsumerRegs>();
    const int s = lane >> 4;                          // spin row of the half spinor this lane owns
    const float d = p.dagger ? -1.f : 1.f;            // -1: the adjoint operator (projector signs exchanged)
    const float e = s ? -1.f : 1.f;                   // sign of this lane's spin row in the y and z projectors
    const float ed = e * d;
    const int r = wid / WPR;                          // tile row
    const int u0 = (wid - r * WPR) * 16 + (lane & 15);
    const bool live = u0 < cs;                        // lanes past the end of a row repeat unit 0 and store nothing
    const int u = live ? u0 : 0;                      // unit = element inside a row component
    const int xin = u / NP, pair = u - xin * NP;
    const int ty = r % BY, tz = r / BY;
    const int y = y0 + ty, z = z0 + tz;
    const float4 *S = reinterpret_cast<const float4 *>(smem);
    const int IB4 = L.I_BYTES / 16, G4 = L.G_BYTES / 16;
    const int rowlen = 12 * cs;
    const int oHy = (int)(L.off_H / 16) + r * rowlen + u, oHz = oHy + ROWS * rowlen;
    const int oXH = L.off_XH / 16;
    // spin rows this lane reads: its own (s) and the partner row of the projector: 3 - s for x and y, 2 + s for z and t
    const int rs = 3 * s, ra = 3 * (3 - s), rb = 3 * (2 + s);     // component index of colour 0 of those rows
    const int os = rs * cs, oa = ra * cs, ob = rb * cs;            // ... and its offset inside a tile row
    // neighbour positions, float4 index of component 0 of this unit: o for buffer 0, bs to add for buffer 1
    const int own = r * rowlen + u;
    const int yp_o = ty == 0 ? own + rowlen : oHy, yp_bs = ty == 0 ? IB4 : 0;
    const int ym_o = ty == 0 ? oHy : own - rowlen, ym_bs = ty == 0 ? 0 : IB4;
    const int zp_o = tz == 0 ? own + BY * rowlen : oHz, zp_bs = tz == 0 ? IB4 : 0;
    const int zm_o = tz == 0 ? oHz : own - BY * rowlen, zm_bs = tz == 0 ? 0 : IB4;
    const bool edge_p = xin + 1 == XB, edge_m = xin == 0;
    const int hxp = oXH + ((ROWS + r) * 12) * NP + pair, hxm = oXH + (r * 12) * NP + pair;
    // links (float4 units), row r of the link buffer: the own links, then
    //   checkerboarded: the packed backward links of this row's sites (the link of the hop from x-mu sits at site x; the t-links of
    //   the input row follow from float4 kBackT on)
    //   full lattice: windows of other sites' own links (last site of the x-block before, row y-1, row z-1), addressed through the
    //   base of a virtual 18-row site
    const int Gr = (int)(L.off_G / 16) + r * (int)(L.GROW / 16);
    const int g_own = Gr + xin;
    const int g_bx_same = CB ? Gr + 18 * XB + xin : g_own;
    const int g_bx_step = CB ? g_bx_same : (edge_m ? Gr + 18 * XB + XB - 1 : g_own - 1);
    const int g_by = CB ? g_bx_same : Gr + 23 * XB - 4 * XB + xin;
    const int g_bz = CB ? g_bx_same : Gr + 28 * XB - 9 * XB + xin;
    const int g_bt = CB ? Gr + (18 + kBackT) * XB + xin : g_own;
    constexpr int LT = CB ? 0 : 3;      // where the t-link starts inside its site data: float4 0 of the packed t-links, or link 3 of the own links

    CVec<2> up[3], la[3], lb[3];   // output spin row s; rows 3 - s (from the x and y hops) and 2 + s (from the z and t hops)
    // this lane's row of U_t^+ (1 + gamma_t) psi of the slice before the centre slice.  The own rows of a slice are read from
    // shared memory ONCE, when the slice is the +t neighbour, and stay in registers until its links have arrived: both t hops
    CVec<2> c1[3];
    SplitOperands A;
    const float4 *Sown = S + own;
    // this unit's output element and x halo sources of the current slice, advanced slice by slice
    const int tfirst = tw(0);
    float4 *o = out + blk(xb, y, z, tfirst) * 12 * cs + u;
    const float4 *gxp = in + blk(xbp, y, z, tfirst) * 12 * cs + pair;                      // site 0 of the next x-block
    const float4 *gxm = in + blk(xbm, y, z, tfirst) * 12 * cs + (XB - 1) * NP + pair;      // last site of the previous one
    const size_t st = (size_t)nxb * Y * Z * 12 * cs;                                       // one slice further
    int t = tfirst;                                                                        // the centre slice
    // refill of this lane's part of the x halo slots from slice pointers gp / gm: the two spin rows the x hops read
    auto refill_x = [&](const float4 *gp, const float4 *gm, int tn, bool active) {
        const int sn = (p.out_parity + y + z + tn) & 1;
        if (active && live) {
            if (edge_p && (!CB || sn == 1)) {
#pragma unroll
                for (int c = 0; c < 3; c++) {
                    cp_async16(S + hxp + (rs + c) * NP, gp + (size_t)(rs + c) * cs);
                    cp_async16(S + hxp + (ra + c) * NP, gp + (size_t)(ra + c) * cs);
                }
            }
            if (edge_m && (!CB || sn == 0)) {
#pragma unroll
                for (int c = 0; c < 3; c++) {
                    cp_async16(S + hxm + (rs + c) * NP, gm + (size_t)(rs + c) * cs);
                    cp_async16(S + hxm + (ra + c) * NP, gm + (size_t)(ra + c) * cs);
                }
            }
        }
        cp_async_commit();
    };
    refill_x(gxp, gxm, t, true);

    // prologue (slice -1 in buffer 0, slice 0 in buffer 1): the carry of the first step, and the own rows of slice 0 in registers
    mbar_wait(&fullI[0], 0);
    mbar_wait(&fullG[0], 0);
    split_load<3, LT>(A, Sown, os, ob, cs, S + g_bt, XB);
    split_half<3, false>(A, d, ed, c1);
    __syncwarp();
    if (lane == 0) { mbar_arrive(&freeI[0]); mbar_arrive(&freeG[0]); }
    mbar_wait(&fullI[1], 0);
#pragma unroll
    for (int c = 0; c < 3; c++) { A.ps[c] = Sown[IB4 + os + c * cs]; A.pp[c] = Sown[IB4 + ob + c * cs]; }

#pragma unroll 1
    for (int k = 0; k < lt; k++) {
        const uint32_t b = (uint32_t)(k + 1) & 1u;
        const int bo = b ? IB4 : 0;
        const bool more = k + 1 < lt;
        int tn = t + 1;
        if (tn == T) tn = 0;
        mbar_wait(&fullG[b], ((uint32_t)(k + 1) >> 1) & 1u);    // the rows of slice k were waited for as the +t slice of the step before
        const float4 *G = S + b * G4;
        const float4 *Sb = S + bo;
#pragma unroll
        for (int c = 0; c < 3; c++) { up[c] = c1[c]; lb[c] = c1[c]; la[c] = czero<2>(); }    // the -t hop (S = -1): up += r, out_{2+s} += d r (lb holds d times its value)
        if (more) {
            // A still holds the own rows of this slice (loaded as the +t neighbour of the step before): the -t hop of the next slice
            load_link_s<LT>(G + g_bt, XB, A.u);
            split_half<3, false>(A, d, ed, c1);
        }
        // y hops
        mbar_wait(&fullH[0], (uint32_t)k & 1u);
        split_load<1>(A, yp_bs ? Sb + yp_o : S + yp_o, os, oa, cs, G + g_own, XB);
        split_hop<1, true>(A, d, e, ed, up, la, lb);
        split_load<1>(A, ym_bs ? Sb + ym_o : S + ym_o, os, oa, cs, G + g_by, XB);
        split_hop<1, false>(A, d, e, ed, up, la, lb);
        __syncwarp();
        if (lane == 0) mbar_arrive(&freeH[0]);
        // z hops
        mbar_wait(&fullH[1], (uint32_t)k & 1u);
        split_load<2>(A, zp_bs ? Sb + zp_o : S + zp_o, os, ob, cs, G + g_own, XB);
        split_hop<2, true>(A, d, e, ed, up, la, lb);
        split_load<2>(A, zm_bs ? Sb + zm_o : S + zm_o, os, ob, cs, G + g_bz, XB);
        split_hop<2, false>(A, d, e, ed, up, la, lb);
        __syncwarp();
        if (lane == 0) mbar_arrive(&freeH[1]);
        // x hops (checkerboarded lines alternate with t: one neighbour has this unit's own index, the other is one site on)
        {
            const float4 *xp = edge_p ? S + hxp : Sb + own + NP, *xm = edge_m ? S + hxm : Sb + own - NP;
            int xp_st = edge_p ? NP : cs, xm_st = edge_m ? NP : cs;
            int g_bx = g_bx_step;
            if (CB) {
                if ((p.out_parity + y + z + t) & 1) { xm = Sb + own; xm_st = cs; g_bx = g_bx_same; }
                else { xp = Sb + own; xp_st = cs; }
            }
            cp_async_wait<0>();                // this lane's x halo slots hold slice k
            split_load<0>(A, xp, rs * xp_st, ra * xp_st, xp_st, G + g_own, XB);
            split_hop<0, true>(A, d, e, ed, up, la, lb);
            split_load<0>(A, xm, rs * xm_st, ra * xm_st, xm_st, G + g_bx, XB);
            split_hop<0, false>(A, d, e, ed, up, la, lb);
        }
        gxp += st; gxm += st;
        if (tn == 0) { gxp -= st * T; gxm -= st * T; }
        refill_x(gxp, gxm, tn, more);
        if constexpr (EPI != 2) {
            __syncwarp();
            if (lane == 0) mbar_arrive(&freeI[b]);       // rows of slice k are no longer read: slice k+2 may land
        }
        // the next slice at this unit's own position: the +t hop of this slice and the -t hop of the slice after the next
        mbar_wait(&fullI[b ^ 1u], ((uint32_t)(k + 2) >> 1) & 1u);
        {
            const float4 *Sn = S + (IB4 - bo) + own;
#pragma unroll
            for (int c = 0; c < 3; c++) { A.ps[c] = Sn[os + c * cs]; A.pp[c] = Sn[ob + c * cs]; }
            load_link_s<3>(G + g_own, XB, A.u);
            split_hop<3, true>(A, d, e, ed, up, la, lb);      // A.ps / A.pp stay live: the next step's -t carry is made from them
        }
        if constexpr (EPI == 0) {
            // lane s holds out_s (up), its share of out_{3-s} (la) and the partner's missing share of out_{2+s} (lb)
#pragma unroll
            for (int c = 0; c < 3; c++) la[c] = rfma(d, shfl_half(lb[c]), la[c]);
            if (live) {
#pragma unroll
                for (int c = 0; c < 3; c++) {
                    __stcs(&o[(size_t)(rs + c) * cs], from_cvec(up[c]));
                    __stcs(&o[(size_t)(ra + c) * cs], from_cvec(la[c]));
                }
            }
        } else {
            // gather one chirality per lane: lane s gets spin rows 2s and 2s+1 of H
            CVec<2> H[6];
#pragma unroll
            for (int c = 0; c < 3; c++) {
                const CVec<2> pu = shfl_half(up[c]), pla = shfl_half(la[c]), plb = shfl_half(lb[c]);
                H[c] = csel(s != 0, rfma(d, plb, la[c]), up[c]);       // s = 1: out_2 = lb(lane s=0) + la;  s = 0: out_0
                H[3 + c] = csel(s != 0, rfma(d, lb[c], pla), pu);      // s = 1: out_3 = la(lane s=0) + lb;  s = 0: out_1 (the partner's up)
            }
            const float4 *pc = S + L.off_C / 16 + b * (L.C_BYTES / 16) + r * (18 * XB) + 9 * s * XB + xin;   // this site's block of chirality s
            CVec<2> res[6];
            if constexpr (EPI == 1) {
                clover_block_mul(pc, XB, H, res);
            } else {
                CVec<2> v[6];
                if constexpr (EPI == 2) {
#pragma unroll
                    for (int i = 0; i < 6; i++) v[i] = to_cvec(Sb[own + (6 * s + i) * cs]);
                } else {
                    const float4 *ax = p.aux + (o - out);       // the same element of the auxiliary field
#pragma unroll
                    for (int i = 0; i < 6; i++) v[i] = to_cvec(__ldg(ax + (size_t)(6 * s + i) * cs));
                }
                clover_block_mul(pc, XB, v, res);
#pragma unroll
                for (int i = 0; i < 6; i++) res[i] = rfma(EPI == 2 ? -0.5f : -0.25f, H[i], res[i]);
                if constexpr (EPI == 2) {
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&freeI[b]);
                }
            }
            if (live) {
#pragma unroll
                for (int i = 0; i < 6; i++) __stcs(&o[(size_t)(6 * s + i) * cs], from_cvec(res[i]));
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&freeG[b]);
        o += st;
        if (tn == 0) o -= st * T;
        t = tn;
    }
    cp_async_wait<0>();
}

}  // namespace

namespace {
// one thread per float of the packed backward-link array (layout: fine_sweep.cuh)
__global__ void pack_back_kernel(FieldGeom g, const float *__restrict__ src, float *__restrict__ dst, long long total) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int k = (int)(idx & 3);
    long long q = idx >> 2;
    const int xin = (int)(q % g.XB); q /= g.XB;
    const int j = (int)(q % kBackF4);
    long long b = q / kBackF4;
    const int xb = (int)(b % g.nxb); b /= g.nxb;
    const int y = (int)(b % g.Y); b /= g.Y;
    const int z = (int)(b % g.Z);
    const int t = (int)(b / g.Z);
    const int xe = xb * g.XB + xin;
    auto lex = [&](int x, int yy, int zz, int tt) { return x + (long long)g.X * (yy + (long long)g.Y * (zz + (long long)g.Z * tt)); };
    float v = 0.f;
    if (j < kBackT) {
        const int f = 4 * j + k;                       // floats 0..53: U_mu(x - mu), mu = 0, 1, 2
        if (f < 54) {
            const int mu = f / 18, e = f % 18;
            int c[4] = {x_of(g, xe, y, z, t), y, z, t};
            const int ext[4] = {g.X, g.Y, g.Z, g.T};
            c[mu] = c[mu] == 0 ? ext[mu] - 1 : c[mu] - 1;
            v = src[lex(c[0], c[1], c[2], c[3]) * 72 + 18 * mu + e];
        }
    } else {
        const int f = 4 * (j - kBackT) + k;            // floats 56..73: U_t of the other parity's site with the same index
        if (f < 18) {
            FieldGeom o = g;
            o.parity = 1 - g.parity;
            v = src[lex(x_of(o, xe, y, z, t), y, z, t) * 72 + 54 + f];
        }
    }
    dst[idx] = v;
}

}  // namespace

mrhs_status_t pack_back_links(const FieldGeom &g, const float *d_gauge_canonical, float4 *d_dst, cudaStream_t st) {
    if (!g.cb) { set_error("pack_back_links: checkerboarded geometry expected"); return MRHS_ERR_INVALID_ARG; }
    const long long total = g.nblocks() * kBackF4 * g.XB * 4;
    pack_back_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(g, d_gauge_canonical, (float *)d_dst, total);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

// ------------------------------------------------------------------ host side
bool sweep_supported(const FieldGeom &g) {
    if (g.N & 1) return false;                       // RHS pairs in FFMA2 lanes; bulk copies need 16-byte pieces
    if (g.Y < 2 || g.Z < 2 || (g.Y % BY) || (g.Z % BZ)) return false;
    const int np = threads_per_site(g.N);
    if (g.XB * np > 48) return false;                // three consumer warps per tile row, twelve per block, plus the producer warps
    const SweepSmem L(g.XB, np, true, g.cb != 0);
    return L.total <= 227u * 1024u;
}

SweepTiling default_sweep_tiling(const FieldGeom &g, int num_sms) {
    SweepTiling t = {g.T, 1, 1};
    const int nty = g.Y / BY, ntz = g.Z / BZ;
    // Thread blocks are dispatched in index order, one per SM, so the tiles that run at the same time are a window of
    // num_sms consecutive blocks.  Tiles are ordered x-blocks fastest, then cy tiles in y, then ALL tiles in z (a strip of the
    // (y,z) plane), then the next strip: the window is then always a compact cy x (num_sms / nxb / cy) patch sliding along
    // z, whose halo rows are mostly another resident block's tile rows (L2 hits).  A chunk of exactly num_sms tiles would
    // drift against the dispatch window (148 SMs, 144-tile chunks) and leave ragged patches: measured 11.56 -> 10.91 GB of DRAM
    // reads per D_hop at 48^4, N = 12.  cy: the divisor of the y tile count closest to a square window.
    t.cz = ntz;
    {
        const double per_xy = (double)num_sms / g.nxb;          // (y,z) tiles in the window
        double best = 1e30;
        for (int cy = 1; cy <= nty; cy++) {
            if (nty % cy) continue;
            const double wz = per_xy / cy;                        // window extent in z, in tiles
            const double shape = 1.0 / (cy * BY) + 1.0 / ((wz < 1 ? 1 : wz) * BZ);
            if (shape < best) { best = shape; t.cy = cy; }
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

namespace {
// Time at which the last of `workers` SMs finishes when each takes the next block of the list as soon as it is free: n_whole
// blocks of cost c_whole, then n_short of cost c_short (costs in slice steps).
double sweep_makespan(long long n_whole, double c_whole, long long n_short, double c_short, int workers) {
    // after the whole blocks: n_whole % workers SMs have done one more than the others
    std::priority_queue<double, std::vector<double>, std::greater<double>> free_at;
    const long long q = n_whole / workers, r = n_whole % workers;
    for (int i = 0; i < workers; i++) free_at.push((q + (i < r ? 1 : 0)) * c_whole);
    double end = (q + (r ? 1 : 0)) * c_whole;
    for (long long i = 0; i < n_short; i++) {
        const double t = free_at.top() + c_short;
        free_at.pop();
        free_at.push(t);
        if (t > end) end = t;
    }
    return end;
}
}  // namespace

bool build_sweep_params(const FieldGeom &g, int out_parity, const SweepTiling &t, int num_sms, SweepParams &p) {
    if (!sweep_supported(g)) return false;
    if (t.lt < 1 || g.T % t.lt || t.cy < 1 || t.cz < 1) return false;
    const int nty = g.Y / BY, ntz = g.Z / BZ;
    if (nty % t.cy || ntz % t.cz) return false;
    const int np = threads_per_site(g.N);
    long long grid = (long long)g.nxb * nty * ntz * (g.T / t.lt);
    if (grid >= (1ll << 31)) return false;
    // Whole-line sweeps: the grid is rarely a multiple of the SM count, and a last wave of a few whole-line blocks keeps most SMs
    // idle for a full sweep (48^4, N = 12: 3456 tiles on 148 SMs = 23.35 waves).  Cut the last tail_tiles tiles into tail_seg
    // segments each; every segment costs about three extra slice steps (two extra slices, pipeline fill).  Pick the pair with
    // the shortest simulated schedule.
    p.n_whole = (unsigned)grid; p.tail_tiles = 0; p.tail_seg = 1;
    if (t.lt == g.T && num_sms > 0 && grid > num_sms) {
        const double extra = 3.0;
        double best = sweep_makespan(grid, g.T + extra, 0, 0.0, num_sms) * 0.995;     // a split has to win by more than the model's noise
        const long long max_tail = std::min<long long>(grid, 3ll * num_sms), step = std::max(1, num_sms / 37);
        for (int ts = 2; ts <= 8; ts++) {
            if (g.T % ts || g.T / ts < 6) continue;
            for (long long tt = step; tt <= max_tail; tt += step) {
                const double m = sweep_makespan(grid - tt, g.T + extra, tt * ts, g.T / ts + extra, num_sms);
                if (m < best) { best = m; p.tail_tiles = (int)tt; p.tail_seg = ts; }
            }
        }
        p.n_whole = (unsigned)(grid - p.tail_tiles);
        grid = (long long)p.n_whole + (long long)p.tail_tiles * p.tail_seg;
    }
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
    p.gauge_out = p.gauge_in = p.gauge_back = nullptr;
    p.clover = nullptr;
    p.aux = nullptr;
    p.dagger = 0;
    p.pf = 0;   // bulk L2 prefetch of later slices: measured to add DRAM traffic (early lines are evicted before use) and no speed
    const int wpr = (g.XB * np + 15) / 16;
    p.threads = (unsigned)(ROWS * wpr + kSweepProducerWarps) * 32u;
    p.grid = (unsigned)grid;
    p.smem_bytes = SweepSmem(g.XB, np, false, g.cb != 0).total;
    p.smem_bytes_clover = SweepSmem(g.XB, np, true, g.cb != 0).total;
    return true;
}

#define MRHS_SWEEP_LIST(F) F(8, 6) F(6, 6) F(4, 12) F(2, 24) F(16, 2) F(12, 2) F(0, 0)

mrhs_status_t sweep_prepare() {
    const int max_smem = 227 * 1024;
#define MRHS_CASE(XB, NP)                                                                                                     \
    MRHS_CUDA(cudaFuncSetAttribute(hop_sweep_kernel<XB, NP, false, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem)); \
    MRHS_CUDA(cudaFuncSetAttribute(hop_sweep_kernel<XB, NP, true, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem));  \
    MRHS_CUDA(cudaFuncSetAttribute(hop_sweep_kernel<XB, NP, true, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem));  \
    MRHS_CUDA(cudaFuncSetAttribute(hop_sweep_kernel<XB, NP, false, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem)); \
    MRHS_CUDA(cudaFuncSetAttribute(hop_sweep_kernel<XB, NP, true, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem));
    MRHS_SWEEP_LIST(MRHS_CASE)
#undef MRHS_CASE
    return MRHS_OK;
}

namespace {
template <int XB, int NP>
void launch_sweep_t(const SweepParams &p, const void *d_in, void *d_out, cudaStream_t st) {
    if (p.cb && p.clover && p.aux) hop_sweep_kernel<XB, NP, true, 3><<<p.grid, p.threads, p.smem_bytes_clover, st>>>(p, (const float4 *)d_in, (float4 *)d_out);
    else if (p.cb && p.clover) hop_sweep_kernel<XB, NP, true, 1><<<p.grid, p.threads, p.smem_bytes_clover, st>>>(p, (const float4 *)d_in, (float4 *)d_out);
    else if (p.cb)        hop_sweep_kernel<XB, NP, true, 0><<<p.grid, p.threads, p.smem_bytes, st>>>(p, (const float4 *)d_in, (float4 *)d_out);
    else if (p.clover)    hop_sweep_kernel<XB, NP, false, 2><<<p.grid, p.threads, p.smem_bytes_clover, st>>>(p, (const float4 *)d_in, (float4 *)d_out);
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

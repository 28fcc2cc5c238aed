// hop_math.cuh -- per-hop arithmetic of the fine-level hopping term, shared by the gather kernel
// (fine_hop.cu) and the slice-sweep kernel (fine_sweep.cu):
//   (1 - gamma_mu) U_mu(x) psi(x+mu)   and   (1 + gamma_mu) U_mu(x-mu)^+ psi(x-mu)
// (reading S3) in the Hermitian chiral basis of reading S2: spin projection to a
// two-component half spinor, SU(3) multiply on the half spinor, reconstruction.
#pragma once
#include "common.cuh"

namespace mrhs {
namespace {

template <int R> __device__ __forceinline__ CVec<R> czero();
template <> __device__ __forceinline__ CVec<1> czero<1>() { return {{0.f}, {0.f}}; }
template <> __device__ __forceinline__ CVec<2> czero<2>() { return {{0ull}, {0ull}}; }

__device__ __forceinline__ float2 ldg_nc(const float2 *p) { return __ldg(p); }
__device__ __forceinline__ float4 ldg_nc(const float4 *p) { return __ldg(p); }

// The 9 complex entries of link MU of one site.  Site data is [18][xin] float4 = 36 complex
// entries e = 9*mu + 3*row + col, two per float4; g points at float4 0 of the site, stride XB.
template <int MU>
__device__ __forceinline__ void load_link(const float4 *__restrict__ g, int XB, float (&u)[18]) {
    constexpr int e0 = 9 * MU;
    if constexpr ((e0 & 1) == 0) {
#pragma unroll
        for (int j = 0; j < 4; j++) {
            float4 v = __ldg(g + (size_t)(e0 / 2 + j) * XB);
            u[4 * j + 0] = v.x; u[4 * j + 1] = v.y; u[4 * j + 2] = v.z; u[4 * j + 3] = v.w;
        }
        float2 w = __ldg(reinterpret_cast<const float2 *>(g + (size_t)(e0 / 2 + 4) * XB));
        u[16] = w.x; u[17] = w.y;
    } else {
        float2 w = __ldg(reinterpret_cast<const float2 *>(g + (size_t)((e0 - 1) / 2) * XB) + 1);
        u[0] = w.x; u[1] = w.y;
#pragma unroll
        for (int j = 0; j < 4; j++) {
            float4 v = __ldg(g + (size_t)((e0 + 1) / 2 + j) * XB);
            u[2 + 4 * j + 0] = v.x; u[2 + 4 * j + 1] = v.y; u[2 + 4 * j + 2] = v.z; u[2 + 4 * j + 3] = v.w;
        }
    }
}

// Same, from shared memory (plain loads).  The 9 complex entries of link MU of one site.  Site data is [18][xin] float4 = 36 complex
// entries e = 9*mu + 3*row + col, two per float4; g points at float4 0 of the site, stride XB.
template <int MU>
__device__ __forceinline__ void load_link_s(const float4 *__restrict__ g, int XB, float (&u)[18]) {
    constexpr int e0 = 9 * MU;
    if constexpr ((e0 & 1) == 0) {
#pragma unroll
        for (int j = 0; j < 4; j++) {
            float4 v = *(g + (size_t)(e0 / 2 + j) * XB);
            u[4 * j + 0] = v.x; u[4 * j + 1] = v.y; u[4 * j + 2] = v.z; u[4 * j + 3] = v.w;
        }
        float2 w = *(reinterpret_cast<const float2 *>(g + (size_t)(e0 / 2 + 4) * XB));
        u[16] = w.x; u[17] = w.y;
    } else {
        float2 w = *(reinterpret_cast<const float2 *>(g + (size_t)((e0 - 1) / 2) * XB) + 1);
        u[0] = w.x; u[1] = w.y;
#pragma unroll
        for (int j = 0; j < 4; j++) {
            float4 v = *(g + (size_t)((e0 + 1) / 2 + j) * XB);
            u[2 + 4 * j + 0] = v.x; u[2 + 4 * j + 1] = v.y; u[2 + 4 * j + 2] = v.z; u[2 + 4 * j + 3] = v.w;
        }
    }
}

// Operands of one hop as loaded: the neighbour's 12 components for this thread's RHS and the 18 reals
// of the link.  Keeping load and arithmetic apart lets the kernel body put the loads of a later hop
// in front of the arithmetic of the current one (software pipelining in registers).
template <int R> struct HopOperands {
    typename Elem<R>::type psi[12];
    float u[18];
};

// nb: component 0 of the neighbour's element for this thread; cs: component stride (elements).
// g: the link's site data (own site for forward hops, the neighbour's for backward hops).
template <int R, int MU>
__device__ __forceinline__ void hop_load(HopOperands<R> &o, const typename Elem<R>::type *__restrict__ nb, size_t cs,
                                         const float4 *__restrict__ g, int XB) {
#pragma unroll
    for (int c = 0; c < 12; c++) o.psi[c] = ldg_nc(nb + c * cs);
    load_link<MU>(g, XB, o.u);
}

// operands of one hop from shared memory: nb -> component 0 of the neighbour's element (component stride cs
// elements), g -> float4 0 of the link's site data (stride XB)
template <int MU>
__device__ __forceinline__ void hop_load_s(HopOperands<2> &o, const float4 *nb, int cs, const float4 *g, int XB) {
#pragma unroll
    for (int c = 0; c < 12; c++) o.psi[c] = nb[c * cs];
    load_link_s<MU>(g, XB, o.u);
}

// One of the eight hops in two stages.  FWD: (1 - gamma_MU) U_MU(x) psi(x+MU); else (1 + gamma_MU) U_MU(x-MU)^+ psi(x-MU).
// hop_half: spin projection to a half spinor and colour multiply, r = U h or U^+ h (6 complex numbers);
// hop_recon: acc += the four spin components rebuilt from r.  hop_compute does both.
// dg = +1: the operator as written; dg = -1: its adjoint D_hop^+ = gamma_5 D_hop gamma_5 (gamma_5 = diag(1,1,-1,-1), reading S2;
// SURVEY.md Sec. 8(f) NEXT-2), i.e. the same links with the projector signs exchanged.  The sign rides as the scalar operand of
// an FMA that replaces the add (same instruction count, and a * (+-1) is exact).
template <int R, int MU, bool FWD>
__device__ __forceinline__ void hop_half(const HopOperands<R> &o, CVec<R> (&r)[6], float dg) {
    CVec<R> psi[12];
#pragma unroll
    for (int c = 0; c < 12; c++) psi[c] = to_cvec(o.psi[c]);
    const float (&u)[18] = o.u;
    const float sg = FWD ? dg : -dg;      // S of the projector (1 - S gamma_MU)

    // spin projection: h = upper two spin components of (1 - S gamma_MU) psi
    CVec<R> h[6];
#pragma unroll
    for (int c = 0; c < 3; c++) {
        if constexpr (MU == 0) {          // h0 = psi0 + S i psi3 ; h1 = psi1 + S i psi2
            h[c]     = {sfnma(sg, psi[9 + c].im, psi[c].re),     sfma(sg, psi[9 + c].re, psi[c].im)};
            h[3 + c] = {sfnma(sg, psi[6 + c].im, psi[3 + c].re), sfma(sg, psi[6 + c].re, psi[3 + c].im)};
        } else if constexpr (MU == 1) {   // h0 = psi0 + S psi3 ; h1 = psi1 - S psi2
            h[c]     = rfma(sg, psi[9 + c], psi[c]);
            h[3 + c] = rfma(-sg, psi[6 + c], psi[3 + c]);
        } else if constexpr (MU == 2) {   // h0 = psi0 + S i psi2 ; h1 = psi1 - S i psi3
            h[c]     = {sfnma(sg, psi[6 + c].im, psi[c].re),    sfma(sg, psi[6 + c].re, psi[c].im)};
            h[3 + c] = {sfma(sg, psi[9 + c].im, psi[3 + c].re), sfnma(sg, psi[9 + c].re, psi[3 + c].im)};
        } else {                          // h0 = psi0 - S psi2 ; h1 = psi1 - S psi3
            h[c]     = rfma(-sg, psi[6 + c], psi[c]);
            h[3 + c] = rfma(-sg, psi[9 + c], psi[3 + c]);
        }
    }

    // colour multiply: r = U h (FWD) or U^+ h
#pragma unroll
    for (int s = 0; s < 2; s++) {
#pragma unroll
        for (int c = 0; c < 3; c++) {
            if constexpr (FWD) {
                CVec<R> t = cmul(u[2 * (3 * c + 0)], u[2 * (3 * c + 0) + 1], h[3 * s + 0]);
                t = cfma(u[2 * (3 * c + 1)], u[2 * (3 * c + 1) + 1], h[3 * s + 1], t);
                r[3 * s + c] = cfma(u[2 * (3 * c + 2)], u[2 * (3 * c + 2) + 1], h[3 * s + 2], t);
            } else {
                CVec<R> t = cmul_conj(u[2 * (0 + c)], u[2 * (0 + c) + 1], h[3 * s + 0]);
                t = cfma_conj(u[2 * (3 + c)], u[2 * (3 + c) + 1], h[3 * s + 1], t);
                r[3 * s + c] = cfma_conj(u[2 * (6 + c)], u[2 * (6 + c) + 1], h[3 * s + 2], t);
            }
        }
    }

}

template <int R, int MU, bool FWD>
__device__ __forceinline__ void hop_recon(const CVec<R> (&r)[6], CVec<R> (&acc)[12], float dg) {
    // reconstruction: upper components get r, lower ones -S i sigma_MU r (spatial) or -S r (time)
    const float sg = FWD ? dg : -dg;
#pragma unroll
    for (int c = 0; c < 3; c++) {
        acc[c] = cadd(acc[c], r[c]);
        acc[3 + c] = cadd(acc[3 + c], r[3 + c]);
        if constexpr (MU == 0) {          // out2 += -S i r1 ; out3 += -S i r0
            acc[6 + c] = {sfma(sg, r[3 + c].im, acc[6 + c].re), sfnma(sg, r[3 + c].re, acc[6 + c].im)};
            acc[9 + c] = {sfma(sg, r[c].im, acc[9 + c].re),     sfnma(sg, r[c].re, acc[9 + c].im)};
        } else if constexpr (MU == 1) {   // out2 += -S r1 ; out3 += S r0
            acc[6 + c] = rfma(-sg, r[3 + c], acc[6 + c]);
            acc[9 + c] = rfma(sg, r[c], acc[9 + c]);
        } else if constexpr (MU == 2) {   // out2 += -S i r0 ; out3 += S i r1
            acc[6 + c] = {sfma(sg, r[c].im, acc[6 + c].re),      sfnma(sg, r[c].re, acc[6 + c].im)};
            acc[9 + c] = {sfnma(sg, r[3 + c].im, acc[9 + c].re), sfma(sg, r[3 + c].re, acc[9 + c].im)};
        } else {                          // out2 += -S r0 ; out3 += -S r1
            acc[6 + c] = rfma(-sg, r[c], acc[6 + c]);
            acc[9 + c] = rfma(-sg, r[3 + c], acc[9 + c]);
        }
    }
}

template <int R, int MU, bool FWD>
__device__ __forceinline__ void hop_compute(const HopOperands<R> &o, CVec<R> (&acc)[12], float dg) {
    CVec<R> r[6];
    hop_half<R, MU, FWD>(o, r, dg);
    hop_recon<R, MU, FWD>(r, acc, dg);
}

}  // namespace
}  // namespace mrhs

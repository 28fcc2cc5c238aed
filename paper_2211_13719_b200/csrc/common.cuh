// common.cuh -- shared host/device helpers of the sm_100a MRHS stencil library:
// error plumbing, exact small-integer division by runtime constants, and the
// packed-fp32 (FFMA2 / FADD2) arithmetic the stencil kernels are written in.
#pragma once
#include <cuda_runtime.h>
#include <cstdarg>
#include <cstdint>
#include <cstdio>

#include "../../include/mrhs.h"

namespace mrhs {

// ------------------------------------------------------------------ errors
void set_error(const char *fmt, ...);
mrhs_status_t cuda_fail(cudaError_t e, const char *what, const char *file, int line);

#define MRHS_CUDA(call)                                                                   \
    do {                                                                                  \
        cudaError_t e_ = (call);                                                          \
        if (e_ != cudaSuccess) return ::mrhs::cuda_fail(e_, #call, __FILE__, __LINE__);  \
    } while (0)

#define MRHS_REQUIRE(cond, ...)                                                           \
    do {                                                                                  \
        if (!(cond)) {                                                                    \
            ::mrhs::set_error(__VA_ARGS__);                                               \
            return MRHS_ERR_INVALID_ARG;                                                  \
        }                                                                                 \
    } while (0)

// --------------------------------------------------- division by a runtime constant
// q = n / d for 0 <= n < 2^32 / d  (exact there: m = floor(2^32/d) + 1, error term n*(m*d - 2^32) < 2^32).
// Every numerator in this library is a tile, block or thread index, far below that bound;
// the host checks the bound when it builds the divider.
struct FastDiv {
    uint32_t mul;
    uint32_t div;
    __host__ __device__ __forceinline__ uint32_t quot(uint32_t n) const {
#ifdef __CUDA_ARCH__
        return div == 1 ? n : __umulhi(n, mul);
#else
        return div == 1 ? n : (uint32_t)(((uint64_t)n * mul) >> 32);     // the same multiply as on the device (host-side plan checks)
#endif
    }
    // n -> (n / d, n % d)
    __host__ __device__ __forceinline__ void divmod(uint32_t n, uint32_t &q, uint32_t &r) const {
        q = quot(n);
        r = n - q * div;
    }
};

inline bool make_fastdiv(uint32_t d, uint64_t max_numerator, FastDiv &out) {
    if (d == 0) return false;
    out.div = d;
    out.mul = d == 1 ? 0u : (uint32_t)((1ull << 32) / d + 1);
    return max_numerator * (uint64_t)d < (1ull << 32);
}

// ------------------------------------------------------------ packed fp32 arithmetic
// Vec<2> holds the same real quantity for two right-hand sides in one 64-bit register
// pair, so one FFMA2 / FADD2 serves both; the scalar operand of sfma()/sfnma() is a link
// or clover entry shared by all RHS (PAPER.md:23 (i)) and becomes the broadcast ".F32"
// operand of FFMA2.  Vec<1> is the plain scalar path (N_rhs odd, i.e. N_rhs = 1).
template <int R> struct Vec;

template <> struct Vec<1> {
    float v;
};
template <> struct Vec<2> {
    unsigned long long v;
};

#ifdef __CUDACC__
__device__ __forceinline__ unsigned long long pack2(float a, float b) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ void unpack2(unsigned long long p, float &a, float &b) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(p));
}

__device__ __forceinline__ Vec<1> vadd(Vec<1> a, Vec<1> b) { return {a.v + b.v}; }
__device__ __forceinline__ Vec<1> vsub(Vec<1> a, Vec<1> b) { return {a.v - b.v}; }
__device__ __forceinline__ Vec<1> smul(float s, Vec<1> a) { return {s * a.v}; }
__device__ __forceinline__ Vec<1> sfma(float s, Vec<1> a, Vec<1> c) { return {fmaf(s, a.v, c.v)}; }
__device__ __forceinline__ Vec<1> sfnma(float s, Vec<1> a, Vec<1> c) { return {fmaf(-s, a.v, c.v)}; }
__device__ __forceinline__ Vec<1> vzero1() { return {0.f}; }

__device__ __forceinline__ Vec<2> vadd(Vec<2> a, Vec<2> b) {
    Vec<2> r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ Vec<2> vsub(Vec<2> a, Vec<2> b) {
    Vec<2> r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ Vec<2> smul(float s, Vec<2> a) {
    Vec<2> r;
    unsigned long long ss = pack2(s, s);
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(ss), "l"(a.v));
    return r;
}
__device__ __forceinline__ Vec<2> sfma(float s, Vec<2> a, Vec<2> c) {
    Vec<2> r;
    unsigned long long ss = pack2(s, s);
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(ss), "l"(a.v), "l"(c.v));
    return r;
}
__device__ __forceinline__ Vec<2> sfnma(float s, Vec<2> a, Vec<2> c) {
    Vec<2> r;
    unsigned long long ss = pack2(-s, -s);
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(ss), "l"(a.v), "l"(c.v));
    return r;
}

// A complex quantity for R right-hand sides.
template <int R> struct CVec {
    Vec<R> re, im;
};

template <int R> __device__ __forceinline__ CVec<R> cadd(CVec<R> a, CVec<R> b) {
    return {vadd(a.re, b.re), vadd(a.im, b.im)};
}
template <int R> __device__ __forceinline__ CVec<R> csub(CVec<R> a, CVec<R> b) {
    return {vsub(a.re, b.re), vsub(a.im, b.im)};
}
// a + i b
template <int R> __device__ __forceinline__ CVec<R> cadd_i(CVec<R> a, CVec<R> b) {
    return {vsub(a.re, b.im), vadd(a.im, b.re)};
}
// a - i b
template <int R> __device__ __forceinline__ CVec<R> csub_i(CVec<R> a, CVec<R> b) {
    return {vadd(a.re, b.im), vsub(a.im, b.re)};
}
// u * a          (u = ur + i ui, a scalar shared by all RHS)
template <int R> __device__ __forceinline__ CVec<R> cmul(float ur, float ui, CVec<R> a) {
    CVec<R> r;
    r.re = sfnma(ui, a.im, smul(ur, a.re));
    r.im = sfma(ui, a.re, smul(ur, a.im));
    return r;
}
// c + u * a
template <int R> __device__ __forceinline__ CVec<R> cfma(float ur, float ui, CVec<R> a, CVec<R> c) {
    CVec<R> r;
    r.re = sfnma(ui, a.im, sfma(ur, a.re, c.re));
    r.im = sfma(ui, a.re, sfma(ur, a.im, c.im));
    return r;
}
// conj(u) * a
template <int R> __device__ __forceinline__ CVec<R> cmul_conj(float ur, float ui, CVec<R> a) {
    CVec<R> r;
    r.re = sfma(ui, a.im, smul(ur, a.re));
    r.im = sfnma(ui, a.re, smul(ur, a.im));
    return r;
}
// c + conj(u) * a
template <int R> __device__ __forceinline__ CVec<R> cfma_conj(float ur, float ui, CVec<R> a, CVec<R> c) {
    CVec<R> r;
    r.re = sfma(ui, a.im, sfma(ur, a.re, c.re));
    r.im = sfnma(ui, a.re, sfma(ur, a.im, c.im));
    return r;
}
// c + s * a with s real
template <int R> __device__ __forceinline__ CVec<R> rfma(float s, CVec<R> a, CVec<R> c) {
    return {sfma(s, a.re, c.re), sfma(s, a.im, c.im)};
}
template <int R> __device__ __forceinline__ CVec<R> rmul(float s, CVec<R> a) {
    return {smul(s, a.re), smul(s, a.im)};
}

// ---- field element access.  One "element" is one spin-colour component of one site for
// the R right-hand sides a thread owns: R = 2 -> float4 (re0 re1 im0 im1), R = 1 -> float2.
template <int R> struct Elem;
template <> struct Elem<1> { typedef float2 type; };
template <> struct Elem<2> { typedef float4 type; };

__device__ __forceinline__ CVec<1> to_cvec(float2 e) { return {{e.x}, {e.y}}; }
__device__ __forceinline__ CVec<2> to_cvec(float4 e) { return {{pack2(e.x, e.y)}, {pack2(e.z, e.w)}}; }
__device__ __forceinline__ float2 from_cvec(CVec<1> c) { return make_float2(c.re.v, c.im.v); }
__device__ __forceinline__ float4 from_cvec(CVec<2> c) {
    float4 e;
    unpack2(c.re.v, e.x, e.y);
    unpack2(c.im.v, e.z, e.w);
    return e;
}
#endif  // __CUDACC__

}  // namespace mrhs

// layout.cu -- canonical <-> native conversion kernels and the layout entry points of
// include/mrhs.h.  Pure data movement, bit-exact; never on
// the timed path (no layout transforms inside the solver).
#include "layout.cuh"

namespace mrhs {

namespace {

// One thread per complex element, enumerated in NATIVE order (block, comp, site in block, rhs).
template <bool IMPORT>
__global__ void fine_convert_kernel(FieldGeom g, const float2 *__restrict__ src_c, float *__restrict__ nat,
                                    float2 *__restrict__ dst_c, long long total) {
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    int r = (int)(idx % g.N);
    long long q = idx / g.N;
    int xin = (int)(q % g.XB); q /= g.XB;
    int comp = (int)(q % g.ncomp);
    long long b = q / g.ncomp;
    int xb = (int)(b % g.nxb); b /= g.nxb;
    int y = (int)(b % g.Y); b /= g.Y;
    int z = (int)(b % g.Z);
    int t = (int)(b / g.Z);
    int xe = xb * g.XB + xin;
    int x = x_of(g, xe, y, z, t);
    long long lex = x + (long long)g.X * (y + (long long)g.Y * (z + (long long)g.Z * t));
    long long cs = g.cb ? (lex >> 1) : lex;
    long long cidx = (cs * g.ncomp + comp) * g.N + r;
    long long noff = native_offset(g, xe, y, z, t, comp);
    int ere = rhs_elem(g.N, r, 0), eim = rhs_elem(g.N, r, 1);
    if (IMPORT) {
        float2 v = src_c[cidx];
        nat[noff + ere] = v.x;
        nat[noff + eim] = v.y;
    } else {
        dst_c[cidx] = make_float2(nat[noff + ere], nat[noff + eim]);
    }
}

// Coarse vectors: native v[lex][nb][e(r)], canonical v[lex][nb][r] complex.
template <bool IMPORT>
__global__ void coarse_convert_kernel(int N, const float2 *__restrict__ src_c, float *__restrict__ nat,
                                      float2 *__restrict__ dst_c, long long total) {
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    int r = (int)(idx % N);
    long long grp = idx / N;   // (site, comp)
    long long noff = grp * 2ll * N;
    int ere = rhs_elem(N, r, 0), eim = rhs_elem(N, r, 1);
    if (IMPORT) {
        float2 v = src_c[idx];
        nat[noff + ere] = v.x;
        nat[noff + eim] = v.y;
    } else {
        dst_c[idx] = make_float2(nat[noff + ere], nat[noff + eim]);
    }
}

// full native <-> even/odd native.  One thread per (site of the full field, comp, rhs-float).
template <bool SPLIT>
__global__ void cb_kernel(FieldGeom gf, FieldGeom ge, FieldGeom go, float *__restrict__ full,
                          float *__restrict__ even, float *__restrict__ odd, long long total) {
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    int e = (int)(idx % (2 * gf.N));
    long long q = idx / (2 * gf.N);
    int xin = (int)(q % gf.XB); q /= gf.XB;
    int comp = (int)(q % gf.ncomp);
    long long b = q / gf.ncomp;
    int xb = (int)(b % gf.nxb); b /= gf.nxb;
    int y = (int)(b % gf.Y); b /= gf.Y;
    int z = (int)(b % gf.Z);
    int t = (int)(b / gf.Z);
    int x = xb * gf.XB + xin;
    int p = (x + y + z + t) & 1;
    const FieldGeom &gc = p ? go : ge;
    long long coff = native_offset(gc, x >> 1, y, z, t, comp) + e;
    float *cbp = p ? odd : even;
    if (SPLIT) cbp[coff] = full[idx];
    else full[idx] = cbp[coff];
}

// Coarse vectors, full native [lex][nb][2N floats] <-> even/odd native [lex >> 1][nb][2N floats].  One thread per float of the full field.
template <bool SPLIT>
__global__ void coarse_cb_kernel(int X, int Y, int Z, long long per_site, float *__restrict__ full, float *__restrict__ even,
                                 float *__restrict__ odd, long long total) {
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const long long lex = idx / per_site, e = idx - lex * per_site;
    long long s = lex;
    const int x = (int)(s % X); s /= X;
    const int y = (int)(s % Y); s /= Y;
    const int z = (int)(s % Z);
    const int t = (int)(s / Z);
    float *cbp = ((x + y + z + t) & 1) ? odd : even;
    const long long coff = (lex >> 1) * per_site + e;
    if (SPLIT) cbp[coff] = full[idx];
    else full[idx] = cbp[coff];
}

bool valid_fine_dims(const int dims[4]) {
    for (int i = 0; i < 4; i++)
        if (dims[i] < 2 || (dims[i] & 1)) return false;
    return true;
}
bool valid_coarse_dims(const int dims[4]) {
    for (int i = 0; i < 4; i++)
        if (dims[i] < 2) return false;
    return true;
}
bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// kind: 0 = decide by ncomp (12 -> fine layout, anything else -> coarse layout), 1 = coarse layout whatever ncomp is
template <bool IMPORT>
mrhs_status_t convert(const int dims[4], int ncomp, int nrhs, int parity, const void *src, void *dst,
                      void *stream, int kind = 0) {
    MRHS_REQUIRE(dims && src && dst, "field convert: NULL argument");
    MRHS_REQUIRE(nrhs >= 1 && ncomp >= 1, "field convert: nrhs and ncomp must be positive");
    MRHS_REQUIRE(parity >= 0 && parity <= 2, "field convert: parity must be 0, 1 or 2");
    MRHS_REQUIRE(aligned16(src) && aligned16(dst), "field convert: buffers must be 16-byte aligned");
    MRHS_REQUIRE(src != dst, "field convert: in-place conversion is not supported");
    cudaStream_t st = (cudaStream_t)stream;
    const int threads = 256;
    if (ncomp == 12 && kind == 0) {
        MRHS_REQUIRE(valid_fine_dims(dims), "field convert: fine extents must be even and >= 2");
        FieldGeom g = make_geom(dims, ncomp, nrhs, parity);
        long long total = g.nsites * ncomp * nrhs;
        long long blocks = (total + threads - 1) / threads;
        MRHS_REQUIRE(blocks < (1ll << 31), "field convert: field too large");
        if (IMPORT)
            fine_convert_kernel<true><<<(unsigned)blocks, threads, 0, st>>>(g, (const float2 *)src, (float *)dst, nullptr, total);
        else
            fine_convert_kernel<false><<<(unsigned)blocks, threads, 0, st>>>(g, nullptr, (float *)const_cast<void *>(src), (float2 *)dst, total);
    } else {
        MRHS_REQUIRE(valid_coarse_dims(dims), "field convert: coarse extents must be >= 2");
        // a checkerboarded coarse field holds the sites of one parity ordered by lex (index lex >> 1): same element order
        MRHS_REQUIRE(parity == MRHS_FULL || valid_fine_dims(dims), "field convert: checkerboarded coarse fields need even extents");
        long long total = (long long)dims[0] * dims[1] * dims[2] * dims[3] * ncomp * nrhs / (parity == MRHS_FULL ? 1 : 2);
        long long blocks = (total + threads - 1) / threads;
        MRHS_REQUIRE(blocks < (1ll << 31), "field convert: field too large");
        if (IMPORT)
            coarse_convert_kernel<true><<<(unsigned)blocks, threads, 0, st>>>(nrhs, (const float2 *)src, (float *)dst, nullptr, total);
        else
            coarse_convert_kernel<false><<<(unsigned)blocks, threads, 0, st>>>(nrhs, nullptr, (float *)const_cast<void *>(src), (float2 *)dst, total);
    }
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

template <bool SPLIT>
mrhs_status_t cb_convert(const int dims[4], int ncomp, int nrhs, void *full, void *even, void *odd, void *stream, int kind = 0) {
    MRHS_REQUIRE(dims && full && even && odd, "cb split/merge: NULL argument");
    MRHS_REQUIRE(nrhs >= 1 && ncomp >= 1, "cb split/merge: nrhs and ncomp must be positive");
    if (ncomp != 12 || kind == 1) {
        MRHS_REQUIRE(valid_fine_dims(dims), "cb split/merge: extents must be even and >= 2");
        MRHS_REQUIRE(aligned16(full) && aligned16(even) && aligned16(odd), "cb split/merge: buffers must be 16-byte aligned");
        MRHS_REQUIRE(full != even && full != odd && even != odd, "cb split/merge: buffers must be distinct");
        const long long per_site = 2ll * ncomp * nrhs;
        const long long total = (long long)dims[0] * dims[1] * dims[2] * dims[3] * per_site;
        const long long blocks = (total + 255) / 256;
        MRHS_REQUIRE(blocks < (1ll << 31), "cb split/merge: field too large");
        coarse_cb_kernel<SPLIT><<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(dims[0], dims[1], dims[2], per_site, (float *)full, (float *)even,
                                                                                   (float *)odd, total);
        MRHS_CUDA(cudaGetLastError());
        return MRHS_OK;
    }
    MRHS_REQUIRE(valid_fine_dims(dims), "cb split/merge: extents must be even and >= 2");
    MRHS_REQUIRE(aligned16(full) && aligned16(even) && aligned16(odd), "cb split/merge: buffers must be 16-byte aligned");
    MRHS_REQUIRE(full != even && full != odd && even != odd, "cb split/merge: buffers must be distinct");
    FieldGeom gf = make_geom(dims, ncomp, nrhs, MRHS_FULL);
    FieldGeom ge = make_geom(dims, ncomp, nrhs, MRHS_EVEN);
    FieldGeom go = make_geom(dims, ncomp, nrhs, MRHS_ODD);
    long long total = gf.nfloats();
    const int threads = 256;
    long long blocks = (total + threads - 1) / threads;
    MRHS_REQUIRE(blocks < (1ll << 31), "cb split/merge: field too large");
    cb_kernel<SPLIT><<<(unsigned)blocks, threads, 0, (cudaStream_t)stream>>>(gf, ge, go, (float *)full, (float *)even, (float *)odd, total);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

}  // namespace

}  // namespace mrhs

using namespace mrhs;

extern "C" {

int mrhs_xblock(int x_eff, int nrhs) {
    if (x_eff < 1 || nrhs < 1) return 0;
    return xblock_host(x_eff, nrhs);
}

size_t mrhs_field_bytes(const int dims[4], int ncomp, int nrhs, int checkerboarded) {
    if (!dims || ncomp < 1 || nrhs < 1) return 0;
    for (int i = 0; i < 4; i++)
        if (dims[i] < 2) return 0;
    size_t v = (size_t)dims[0] * dims[1] * dims[2] * dims[3];
    if (checkerboarded) {
        if (!valid_fine_dims(dims)) return 0;
        v /= 2;
    }
    return v * (size_t)ncomp * (size_t)nrhs * 8u;
}

mrhs_status_t mrhs_field_import(const int dims[4], int ncomp, int nrhs, int parity, const void *d_canonical,
                                void *d_native, void *cuda_stream) {
    return convert<true>(dims, ncomp, nrhs, parity, d_canonical, d_native, cuda_stream);
}

mrhs_status_t mrhs_field_export(const int dims[4], int ncomp, int nrhs, int parity, const void *d_native,
                                void *d_canonical, void *cuda_stream) {
    return convert<false>(dims, ncomp, nrhs, parity, d_native, d_canonical, cuda_stream);
}

mrhs_status_t mrhs_coarse_field_import(const int cdims[4], int nbasis, int nrhs, int parity, const void *d_canonical,
                                       void *d_native, void *cuda_stream) {
    return convert<true>(cdims, nbasis, nrhs, parity, d_canonical, d_native, cuda_stream, 1);
}

mrhs_status_t mrhs_coarse_field_export(const int cdims[4], int nbasis, int nrhs, int parity, const void *d_native,
                                       void *d_canonical, void *cuda_stream) {
    return convert<false>(cdims, nbasis, nrhs, parity, d_native, d_canonical, cuda_stream, 1);
}

mrhs_status_t mrhs_coarse_cb_split(const int cdims[4], int nbasis, int nrhs, const void *d_full, void *d_even, void *d_odd,
                                   void *cuda_stream) {
    return cb_convert<true>(cdims, nbasis, nrhs, const_cast<void *>(d_full), d_even, d_odd, cuda_stream, 1);
}

mrhs_status_t mrhs_coarse_cb_merge(const int cdims[4], int nbasis, int nrhs, const void *d_even, const void *d_odd,
                                   void *d_full, void *cuda_stream) {
    return cb_convert<false>(cdims, nbasis, nrhs, d_full, const_cast<void *>(d_even), const_cast<void *>(d_odd), cuda_stream, 1);
}

mrhs_status_t mrhs_cb_split(const int dims[4], int ncomp, int nrhs, const void *d_full, void *d_even, void *d_odd,
                            void *cuda_stream) {
    return cb_convert<true>(dims, ncomp, nrhs, const_cast<void *>(d_full), d_even, d_odd, cuda_stream);
}

mrhs_status_t mrhs_cb_merge(const int dims[4], int ncomp, int nrhs, const void *d_even, const void *d_odd,
                            void *d_full, void *cuda_stream) {
    return cb_convert<false>(dims, ncomp, nrhs, d_full, const_cast<void *>(d_even), const_cast<void *>(d_odd), cuda_stream);
}

}  // extern "C"

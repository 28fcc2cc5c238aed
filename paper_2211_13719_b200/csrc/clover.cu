// clover.cu -- the site-diagonal clover term.
//   M_ooee(x) = (4 + m) - (c_sw/2) sum_{mu<nu} sigma_munu F_munu(x)        (readings S5-S7)
// "precomputed" once per gauge field and applied as two 6x6 Hermitian chiral
// blocks per site (PAPER.md:47 compact clover) to N_rhs right-hand sides at once.
//
// In the chiral basis of reading S2, sigma_jk = -eps_jkl sigma_l on both chiralities and
// sigma_kt = diag(+sigma_k, -sigma_k), so with the Hermitian 3x3 colour matrices
//   B_x = +-F_xt - F_yz,  B_y = +-F_yt + F_xz,  B_z = +-F_zt - F_xy   (+ for chirality 0)
// the block of chirality ch is (4+m) 1 - (c_sw/2) [[B_z, B_x - i B_y], [B_x + i B_y, -B_z]].
//
// Packed block (36 floats): 6 real diagonal entries, then the 15 strictly-lower entries in
// row-major order (i(i-1)/2 + j), re then im.  Two blocks per site = 72 floats = 18 float4.
#include "fine_hop.cuh"

namespace mrhs {

namespace {

struct M3 {
    double re[9], im[9];
};

__device__ M3 load_link_c(const float2 *__restrict__ U, long long lex, int mu) {
    M3 m;
    const float2 *p = U + (lex * 4 + mu) * 9;
    for (int k = 0; k < 9; k++) { m.re[k] = p[k].x; m.im[k] = p[k].y; }
    return m;
}
__device__ M3 adj(const M3 &a) {
    M3 r;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) { r.re[3 * i + j] = a.re[3 * j + i]; r.im[3 * i + j] = -a.im[3 * j + i]; }
    return r;
}
__device__ M3 mul(const M3 &a, const M3 &b) {
    M3 r;
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            double sr = 0, si = 0;
            for (int k = 0; k < 3; k++) {
                sr += a.re[3 * i + k] * b.re[3 * k + j] - a.im[3 * i + k] * b.im[3 * k + j];
                si += a.re[3 * i + k] * b.im[3 * k + j] + a.im[3 * i + k] * b.re[3 * k + j];
            }
            r.re[3 * i + j] = sr; r.im[3 * i + j] = si;
        }
    return r;
}

struct Lat {
    int X, Y, Z, T;
};
__device__ long long shift(const Lat &L, long long lex, int mu, int d) {
    int c[4];
    c[0] = (int)(lex % L.X); lex /= L.X;
    c[1] = (int)(lex % L.Y); lex /= L.Y;
    c[2] = (int)(lex % L.Z);
    c[3] = (int)(lex / L.Z);
    const int ext[4] = {L.X, L.Y, L.Z, L.T};
    c[mu] = (c[mu] + d + ext[mu]) % ext[mu];
    return c[0] + (long long)L.X * (c[1] + (long long)L.Y * (c[2] + (long long)L.Z * c[3]));
}

// F_munu(x) = (Q - Q^+) / (8 i), Q = sum of the four plaquette leaves in the mu-nu plane that
// start and end at x, all with the same orientation (reading S5).
__device__ M3 field_strength(const Lat &L, const float2 *__restrict__ U, long long x, int mu, int nu) {
    const long long xpm = shift(L, x, mu, 1), xpn = shift(L, x, nu, 1);
    const long long xmm = shift(L, x, mu, -1), xmn = shift(L, x, nu, -1);
    const long long xmmpn = shift(L, xmm, nu, 1), xmmmn = shift(L, xmm, nu, -1), xmnpm = shift(L, xmn, mu, 1);
    M3 q[4];
    // U_mu(x) U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+
    q[0] = mul(mul(load_link_c(U, x, mu), load_link_c(U, xpm, nu)),
               mul(adj(load_link_c(U, xpn, mu)), adj(load_link_c(U, x, nu))));
    // U_nu(x) U_mu(x-mu+nu)^+ U_nu(x-mu)^+ U_mu(x-mu)
    q[1] = mul(mul(load_link_c(U, x, nu), adj(load_link_c(U, xmmpn, mu))),
               mul(adj(load_link_c(U, xmm, nu)), load_link_c(U, xmm, mu)));
    // U_mu(x-mu)^+ U_nu(x-mu-nu)^+ U_mu(x-mu-nu) U_nu(x-nu)
    q[2] = mul(mul(adj(load_link_c(U, xmm, mu)), adj(load_link_c(U, xmmmn, nu))),
               mul(load_link_c(U, xmmmn, mu), load_link_c(U, xmn, nu)));
    // U_nu(x-nu)^+ U_mu(x-nu) U_nu(x-nu+mu) U_mu(x)^+
    q[3] = mul(mul(adj(load_link_c(U, xmn, nu)), load_link_c(U, xmn, mu)),
               mul(load_link_c(U, xmnpm, nu), adj(load_link_c(U, x, mu))));
    M3 Q;
    for (int k = 0; k < 9; k++) {
        Q.re[k] = q[0].re[k] + q[1].re[k] + q[2].re[k] + q[3].re[k];
        Q.im[k] = q[0].im[k] + q[1].im[k] + q[2].im[k] + q[3].im[k];
    }
    M3 F;   // (Q - Q^+)/(8i): (a + i b)/i = b - i a
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            double dr = Q.re[3 * i + j] - Q.re[3 * j + i];
            double di = Q.im[3 * i + j] + Q.im[3 * j + i];
            F.re[3 * i + j] = di * 0.125;
            F.im[3 * i + j] = -dr * 0.125;
        }
    return F;
}

__global__ void build_clover_kernel(Lat L, double diag, double half_csw, const float2 *__restrict__ U,
                                    float *__restrict__ packed, long long nsites) {
    long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= nsites) return;
    const M3 Fxy = field_strength(L, U, x, 0, 1), Fxz = field_strength(L, U, x, 0, 2);
    const M3 Fyz = field_strength(L, U, x, 1, 2), Fxt = field_strength(L, U, x, 0, 3);
    const M3 Fyt = field_strength(L, U, x, 1, 3), Fzt = field_strength(L, U, x, 2, 3);
    for (int ch = 0; ch < 2; ch++) {
        const double s = ch == 0 ? 1.0 : -1.0;
        double blk_re[36], blk_im[36];   // 6x6, index 3*spin + colour
        for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++) {
                const int k = 3 * a + b;
                const double bx_re = s * Fxt.re[k] - Fyz.re[k], bx_im = s * Fxt.im[k] - Fyz.im[k];
                const double by_re = s * Fyt.re[k] + Fxz.re[k], by_im = s * Fyt.im[k] + Fxz.im[k];
                const double bz_re = s * Fzt.re[k] - Fxy.re[k], bz_im = s * Fzt.im[k] - Fxy.im[k];
                const double dd = (a == b) ? diag : 0.0;
                // [0][0] = B_z ; [1][1] = -B_z ; [0][1] = B_x - i B_y ; [1][0] = B_x + i B_y
                blk_re[6 * a + b] = dd - half_csw * bz_re;               blk_im[6 * a + b] = -half_csw * bz_im;
                blk_re[6 * (3 + a) + 3 + b] = dd + half_csw * bz_re;     blk_im[6 * (3 + a) + 3 + b] = half_csw * bz_im;
                blk_re[6 * a + 3 + b] = -half_csw * (bx_re + by_im);     blk_im[6 * a + 3 + b] = -half_csw * (bx_im - by_re);
                blk_re[6 * (3 + a) + b] = -half_csw * (bx_re - by_im);   blk_im[6 * (3 + a) + b] = -half_csw * (bx_im + by_re);
            }
        float *o = packed + x * 72 + 36 * ch;
        for (int i = 0; i < 6; i++) o[i] = (float)blk_re[7 * i];
        for (int i = 1; i < 6; i++)
            for (int j = 0; j < i; j++) {
                const int idx = i * (i - 1) / 2 + j;
                o[6 + 2 * idx] = (float)blk_re[6 * i + j];
                o[6 + 2 * idx + 1] = (float)blk_im[6 * i + j];
            }
    }
}

// canonical [site][2][6][6] complex <-> packed [site][72]; one thread per (site, chirality)
__global__ void pack_blocks_kernel(const float2 *__restrict__ blocks, float *__restrict__ packed, long long n2) {
    long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= n2) return;
    const float2 *b = blocks + g * 36;
    float *o = packed + g * 36;
    for (int i = 0; i < 6; i++) o[i] = b[7 * i].x;
    for (int i = 1; i < 6; i++)
        for (int j = 0; j < i; j++) {
            const int idx = i * (i - 1) / 2 + j;
            o[6 + 2 * idx] = b[6 * i + j].x;
            o[6 + 2 * idx + 1] = b[6 * i + j].y;
        }
}
__global__ void unpack_blocks_kernel(const float *__restrict__ packed, float2 *__restrict__ blocks, long long n2) {
    long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= n2) return;
    float2 *b = blocks + g * 36;
    const float *o = packed + g * 36;
    for (int i = 0; i < 6; i++) b[7 * i] = make_float2(o[i], 0.f);
    for (int i = 1; i < 6; i++)
        for (int j = 0; j < i; j++) {
            const int idx = i * (i - 1) / 2 + j;
            b[6 * i + j] = make_float2(o[6 + 2 * idx], o[6 + 2 * idx + 1]);
            b[6 * j + i] = make_float2(o[6 + 2 * idx], -o[6 + 2 * idx + 1]);
        }
}

// packed Hermitian 6x6 blocks -> packed inverse blocks (the inverse of a Hermitian matrix is Hermitian, so the same
// packing holds it).  One thread per (site, chirality); Gauss-Jordan with partial pivoting in fp64.  Setup, untimed.
__global__ void invert_blocks_kernel(const float *__restrict__ packed, float *__restrict__ inv, long long n2) {
    long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= n2) return;
    const float *o = packed + g * 36;
    double ar[6][12], ai[6][12];   // [A | 1] -> [1 | A^-1]
    for (int i = 0; i < 6; i++)
        for (int j = 0; j < 12; j++) { ar[i][j] = (j == 6 + i) ? 1.0 : 0.0; ai[i][j] = 0.0; }
    for (int i = 0; i < 6; i++) ar[i][i] = o[i];
    for (int i = 1; i < 6; i++)
        for (int j = 0; j < i; j++) {
            const int idx = i * (i - 1) / 2 + j;
            ar[i][j] = o[6 + 2 * idx]; ai[i][j] = o[6 + 2 * idx + 1];
            ar[j][i] = o[6 + 2 * idx]; ai[j][i] = -(double)o[6 + 2 * idx + 1];
        }
    for (int c = 0; c < 6; c++) {
        int piv = c;
        double best = ar[c][c] * ar[c][c] + ai[c][c] * ai[c][c];
        for (int r = c + 1; r < 6; r++) {
            const double m = ar[r][c] * ar[r][c] + ai[r][c] * ai[r][c];
            if (m > best) { best = m; piv = r; }
        }
        if (piv != c)
            for (int j = 0; j < 12; j++) {
                double t = ar[c][j]; ar[c][j] = ar[piv][j]; ar[piv][j] = t;
                t = ai[c][j]; ai[c][j] = ai[piv][j]; ai[piv][j] = t;
            }
        const double pr = ar[c][c] / best, pi = -ai[c][c] / best;   // 1 / pivot
        for (int j = 0; j < 12; j++) {
            const double xr = ar[c][j], xi = ai[c][j];
            ar[c][j] = xr * pr - xi * pi; ai[c][j] = xr * pi + xi * pr;
        }
        for (int r = 0; r < 6; r++) {
            if (r == c) continue;
            const double fr = ar[r][c], fi = ai[r][c];
            for (int j = 0; j < 12; j++) {
                ar[r][j] -= fr * ar[c][j] - fi * ai[c][j];
                ai[r][j] -= fr * ai[c][j] + fi * ar[c][j];
            }
        }
    }
    float *q = inv + g * 36;
    for (int i = 0; i < 6; i++) q[i] = (float)ar[i][6 + i];
    for (int i = 1; i < 6; i++)
        for (int j = 0; j < i; j++) {
            const int idx = i * (i - 1) / 2 + j;   // Hermitian part of the computed inverse
            q[6 + 2 * idx] = (float)(0.5 * (ar[i][6 + j] + ar[j][6 + i]));
            q[6 + 2 * idx + 1] = (float)(0.5 * (ai[i][6 + j] - ai[j][6 + i]));
        }
}

// ------------------------------------------------------------------ M_ooee apply
// One thread = one site and R right-hand sides; the 72 packed floats of the site are fetched
// once and reused by every RHS.  One chirality at a time keeps the live set at 6 + 6 elements.
// MODE 0: out = C in.  MODE 1: out = C in + scale * out (out holds a hopping sum: scale -1/2 gives the full Wilson-clover
// matrix of reading S6, -1/4 the Schur complement; gather-kernel paths).  MODE 2: out = C out, in place (in is not read; a
// thread reads the six components of a chirality before it writes them, and no other thread touches them).
template <int R, int MODE>
__global__ void __launch_bounds__(256)
mooee_kernel(int XB, int NP, long long nthreads, float scale, const float4 *__restrict__ clov,
             const typename Elem<R>::type *in, typename Elem<R>::type *out) {
    typedef typename Elem<R>::type E;
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= nthreads) return;
    const int CS = XB * NP;
    const long long b = g / CS;
    const int rem = (int)(g - b * CS);
    const int xin = rem / NP;
    const E *pi = in + (size_t)b * 12 * CS + rem;
    E *po = out + (size_t)b * 12 * CS + rem;
    const float4 *pc = clov + (size_t)b * kSiteF4 * XB + xin;
#pragma unroll
    for (int ch = 0; ch < 2; ch++) {
        CVec<R> psi[6];
#pragma unroll
        for (int c = 0; c < 6; c++) psi[c] = to_cvec(MODE == 2 ? po[(size_t)(6 * ch + c) * CS] : __ldg(pi + (size_t)(6 * ch + c) * CS));
        float a[36];
#pragma unroll
        for (int j = 0; j < 9; j++) {
            float4 v = __ldg(pc + (size_t)(9 * ch + j) * XB);
            a[4 * j] = v.x; a[4 * j + 1] = v.y; a[4 * j + 2] = v.z; a[4 * j + 3] = v.w;
        }
#pragma unroll
        for (int i = 0; i < 6; i++) {
            CVec<R> r = rmul(a[i], psi[i]);
#pragma unroll
            for (int j = 0; j < 6; j++) {
                if (j < i) {
                    const int idx = i * (i - 1) / 2 + j;
                    r = cfma(a[6 + 2 * idx], a[6 + 2 * idx + 1], psi[j], r);
                } else if (j > i) {
                    const int idx = j * (j - 1) / 2 + i;
                    r = cfma_conj(a[6 + 2 * idx], a[6 + 2 * idx + 1], psi[j], r);
                }
            }
            if constexpr (MODE == 1) r = rfma(scale, to_cvec(po[(size_t)(6 * ch + i) * CS]), r);
            po[(size_t)(6 * ch + i) * CS] = from_cvec(r);
        }
    }
}

}  // namespace

mrhs_status_t build_clover(const int dims[4], float mass, float csw, const float2 *d_gauge, float *d_packed, cudaStream_t st) {
    Lat L = {dims[0], dims[1], dims[2], dims[3]};
    long long n = (long long)dims[0] * dims[1] * dims[2] * dims[3];
    long long blocks = (n + 63) / 64;
    build_clover_kernel<<<(unsigned)blocks, 64, 0, st>>>(L, 4.0 + (double)mass, 0.5 * (double)csw, d_gauge, d_packed, n);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

mrhs_status_t pack_clover_blocks(long long nsites, const float2 *d_blocks, float *d_packed, cudaStream_t st) {
    long long n2 = nsites * 2, blocks = (n2 + 127) / 128;
    pack_blocks_kernel<<<(unsigned)blocks, 128, 0, st>>>(d_blocks, d_packed, n2);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

mrhs_status_t invert_clover_blocks(long long nsites, const float *d_packed, float *d_packed_inv, cudaStream_t st) {
    long long n2 = nsites * 2, blocks = (n2 + 63) / 64;
    invert_blocks_kernel<<<(unsigned)blocks, 64, 0, st>>>(d_packed, d_packed_inv, n2);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

mrhs_status_t unpack_clover_blocks(long long nsites, const float *d_packed, float2 *d_blocks, cudaStream_t st) {
    long long n2 = nsites * 2, blocks = (n2 + 127) / 128;
    unpack_blocks_kernel<<<(unsigned)blocks, 128, 0, st>>>(d_packed, d_blocks, n2);
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

mrhs_status_t launch_mooee(const FieldGeom &g, const float4 *d_clover, const void *d_in, void *d_out, cudaStream_t st, float axpy_scale) {
    const int np = threads_per_site(g.N);
    const long long nthreads = g.nsites * np;
    const unsigned blocks = (unsigned)((nthreads + 255) / 256);
    const int mode = d_in == d_out ? 2 : (axpy_scale != 0.f ? 1 : 0);
#define MRHS_MOOEE(R, E, MODE) mooee_kernel<R, MODE><<<blocks, 256, 0, st>>>(g.XB, np, nthreads, axpy_scale, d_clover, (const E *)d_in, (E *)d_out)
    if (g.N & 1) {
        if (mode == 2) MRHS_MOOEE(1, float2, 2); else if (mode == 1) MRHS_MOOEE(1, float2, 1); else MRHS_MOOEE(1, float2, 0);
    } else {
        if (mode == 2) MRHS_MOOEE(2, float4, 2); else if (mode == 1) MRHS_MOOEE(2, float4, 1); else MRHS_MOOEE(2, float4, 0);
    }
#undef MRHS_MOOEE
    MRHS_CUDA(cudaGetLastError());
    return MRHS_OK;
}

}  // namespace mrhs

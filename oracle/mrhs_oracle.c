/*
 * mrhs_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU restatement of the operators of arxiv 2211.13719
 * ("MRHS multigrid solver for Wilson-clover fermions"): the fine-level hopping
 * term D_hop on the full lattice and M_eooe between checkerboarded lattices
 * (Sec. 4), the precomputed site-diagonal clover term M_ooee
 * (Sec. 4) and the coarse-level stencil with nbasis spinor
 * elements per site (PAPER.md:61 Sec. 5, :75 Sec. 6), each applied to N_rhs
 * right-hand sides held in an extra innermost index (Sec. 2).
 *
 * The paper prints no formula.  Every definition below is the textbook form
 * adopted in SURVEY.md Sec. 8(c), readings S1-S9, listed again in DESIGN.md.
 * The code is the definition written out: loops over sites, directions, spin,
 * colour and RHS with full 4x4 gamma matrices; no spin-projection trick, no
 * blocking, no packing, no reordering.  It shares no source, header, table or
 * helper with the CUDA path (paper_2211_13719_b200/csrc) and neither includes
 * the other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this file's shared object.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): gamma algebra; free-field plane
 * wave closed form; gamma5-hermiticity; gauge covariance; D_hop = sum of both
 * M_eooe; RHS-column independence; clover blocks Hermitian / block diagonal /
 * trace / pure gauge / uniform abelian flux closed form / covariance; coarse
 * apply = per-site numpy matmul and = brute-force Galerkin R M P.
 * Versus the paper's own code (not available here): parity unpinned.
 *
 * Canonical layouts (C order, last index fastest), SURVEY.md Sec. 8(b):
 *   site lex = x + X*(y + Y*(z + Z*t)), all extents even, periodic (S1);
 *   spinor  psi[lex][spin 4][colour 3][rhs N];
 *   checkerboarded spinor of parity p: sites with (x+y+z+t)%2 == p, index lex>>1;
 *   gauge   U[lex][mu 4][row 3][col 3], U_mu(x) links x -> x+mu;
 *   clover  C[lex][chirality 2][6][6], block index 3*(spin%2)+colour;
 *   coarse  A[lex][p 9][row nb][col nb], p=0 self, 1..4 = +x..+t, 5..8 = -x..-t;
 *   coarse vector v[lex][nb][rhs N].
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double _Complex dc;

/* ------------------------------------------------------------------ threads */

void orc_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int orc_get_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------ gamma algebra */

/* S2: Hermitian chiral basis.  gamma_k = [[0, -i sigma_k], [i sigma_k, 0]],
 * k = x,y,z; gamma_t = [[0, 1], [1, 0]]; gamma_5 = gamma_x gamma_y gamma_z gamma_t.
 * mu = 0..3 -> x,y,z,t; mu = 4 -> gamma_5 (computed as the product). */
static void pauli(int k, dc s[2][2])
{
    s[0][0] = s[0][1] = s[1][0] = s[1][1] = 0.0;
    if (k == 0) { s[0][1] = 1.0; s[1][0] = 1.0; }
    if (k == 1) { s[0][1] = -I;  s[1][0] = I;   }
    if (k == 2) { s[0][0] = 1.0; s[1][1] = -1.0; }
}

static void mat4_mul(const dc a[4][4], const dc b[4][4], dc c[4][4])
{
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) {
            dc s = 0.0;
            for (int k = 0; k < 4; k++) s += a[i][k] * b[k][j];
            c[i][j] = s;
        }
}

static void gamma_mat(int mu, dc g[4][4])
{
    memset(g, 0, 16 * sizeof(dc));
    if (mu >= 0 && mu < 3) {
        dc s[2][2];
        pauli(mu, s);
        for (int a = 0; a < 2; a++)
            for (int b = 0; b < 2; b++) {
                g[a][2 + b] = -I * s[a][b];
                g[2 + a][b] = I * s[a][b];
            }
    } else if (mu == 3) {
        g[0][2] = g[1][3] = g[2][0] = g[3][1] = 1.0;
    } else {
        dc gx[4][4], gy[4][4], gz[4][4], gt[4][4], t1[4][4], t2[4][4];
        gamma_mat(0, gx); gamma_mat(1, gy); gamma_mat(2, gz); gamma_mat(3, gt);
        mat4_mul(gx, gy, t1); mat4_mul(t1, gz, t2); mat4_mul(t2, gt, g);
    }
}

void orc_gamma(int mu, dc *g16) { gamma_mat(mu, (dc (*)[4])g16); }

/* S6: sigma_munu = (i/2) [gamma_mu, gamma_nu]. */
static void sigma_mat(int mu, int nu, dc s[4][4])
{
    dc a[4][4], b[4][4], ab[4][4], ba[4][4];
    gamma_mat(mu, a); gamma_mat(nu, b);
    mat4_mul(a, b, ab); mat4_mul(b, a, ba);
    for (int i = 0; i < 4; i++)
        for (int j = 0; j < 4; j++) s[i][j] = 0.5 * I * (ab[i][j] - ba[i][j]);
}

void orc_sigma(int mu, int nu, dc *s16) { sigma_mat(mu, nu, (dc (*)[4])s16); }

/* ---------------------------------------------------------------- lattice */

static long lex_of(const int d[4], const int c[4])
{
    return c[0] + (long)d[0] * (c[1] + (long)d[1] * (c[2] + (long)d[2] * c[3]));
}

static void coords_of(const int d[4], long lex, int c[4])
{
    c[0] = (int)(lex % d[0]); lex /= d[0];
    c[1] = (int)(lex % d[1]); lex /= d[1];
    c[2] = (int)(lex % d[2]); lex /= d[2];
    c[3] = (int)lex;
}

/* periodic neighbour (S1): site x + sign * mu_hat */
static long neighbour(const int d[4], long lex, int mu, int sign)
{
    int c[4];
    coords_of(d, lex, c);
    c[mu] = (c[mu] + sign + d[mu]) % d[mu];
    return lex_of(d, c);
}

static int parity_of(const int d[4], long lex)
{
    int c[4];
    coords_of(d, lex, c);
    return (c[0] + c[1] + c[2] + c[3]) & 1;
}

long orc_neighbour(const int dims[4], long lex, int mu, int sign) { return neighbour(dims, lex, mu, sign); }
int orc_parity(const int dims[4], long lex) { return parity_of(dims, lex); }

/* ------------------------------------------------------------- fine hopping */

/* S3, one site: out[s][c][r] = sum over the directions enabled in dirmask of
 *   bit mu     : sum_{s'} (1 - gamma_mu)[s][s'] sum_{c'} U_mu(x)[c][c']          psi(x+mu)[s'][c'][r]
 *   bit 4 + mu : sum_{s'} (1 + gamma_mu)[s][s'] sum_{c'} conj(U_mu(x-mu)[c'][c]) psi(x-mu)[s'][c'][r]
 * Bare sum: no -1/2, no mass.  ufwd[mu] -> U_mu(x) (3x3), ubwd[mu] -> U_mu(x-mu),
 * pfwd[mu] -> psi(x+mu), pbwd[mu] -> psi(x-mu), each [4][3][N].  If x+mu and x-mu
 * coincide (extent 2) both terms are still summed (S17). */
static void dhop_site(int N, const dc *const ufwd[4], const dc *const ubwd[4],
                      const dc *const pfwd[4], const dc *const pbwd[4], int dirmask, dc *out)
{
    for (int i = 0; i < 12 * N; i++) out[i] = 0.0;
    for (int mu = 0; mu < 4; mu++) {
        dc g[4][4];
        gamma_mat(mu, g);
        for (int dir = 0; dir < 2; dir++) {          /* 0: forward hop, 1: backward hop */
            if (!(dirmask & (1 << (4 * dir + mu)))) continue;
            const dc *u = dir ? ubwd[mu] : ufwd[mu];
            const dc *p = dir ? pbwd[mu] : pfwd[mu];
            double sg = dir ? 1.0 : -1.0;
            for (int r = 0; r < N; r++) {
                dc w[4][3];                           /* colour-rotated neighbour spinor */
                for (int s = 0; s < 4; s++)
                    for (int c = 0; c < 3; c++) {
                        dc acc = 0.0;
                        for (int k = 0; k < 3; k++) {
                            dc link = dir ? conj(u[3 * k + c]) : u[3 * c + k];
                            acc += link * p[(s * 3 + k) * N + r];
                        }
                        w[s][c] = acc;
                    }
                for (int s = 0; s < 4; s++)
                    for (int c = 0; c < 3; c++) {
                        dc acc = 0.0;
                        for (int k = 0; k < 4; k++) {
                            dc proj = (s == k ? 1.0 : 0.0) + sg * g[s][k];
                            acc += proj * w[k][c];
                        }
                        out[(s * 3 + c) * N + r] += acc;
                    }
            }
        }
    }
}

/* Packed single-site entry for sampled parity checks (48^4): links[8][3][3] =
 * U_mu(x) for mu=0..3 then U_mu(x-mu) for mu=0..3; nbrs[8][4][3][N] = psi(x+mu)
 * for mu=0..3 then psi(x-mu).  nsites independent sites are processed. */
void orc_dhop_sites(long nsites, int N, const dc *links, const dc *nbrs, int dirmask, dc *out)
{
#pragma omp parallel for schedule(static)
    for (long i = 0; i < nsites; i++) {
        const dc *uf[4], *ub[4], *pf[4], *pb[4];
        for (int mu = 0; mu < 4; mu++) {
            uf[mu] = links + (i * 8 + mu) * 9;
            ub[mu] = links + (i * 8 + 4 + mu) * 9;
            pf[mu] = nbrs + (i * 8 + mu) * 12 * (long)N;
            pb[mu] = nbrs + (i * 8 + 4 + mu) * 12 * (long)N;
        }
        dhop_site(N, uf, ub, pf, pb, dirmask, out + i * 12 * (long)N);
    }
}

/* S3: D_hop on the full lattice.  dirmask = 0xFF for the operator;
 * sub-masks expose single directed hops for the Galerkin self-check (S9). */
void orc_dhop(const int dims[4], int N, const dc *U, const dc *psi, dc *out, int dirmask)
{
    long V = (long)dims[0] * dims[1] * dims[2] * dims[3];
#pragma omp parallel for schedule(static)
    for (long x = 0; x < V; x++) {
        const dc *uf[4], *ub[4], *pf[4], *pb[4];
        for (int mu = 0; mu < 4; mu++) {
            long xp = neighbour(dims, x, mu, +1), xm = neighbour(dims, x, mu, -1);
            uf[mu] = U + (x * 4 + mu) * 9;
            ub[mu] = U + (xm * 4 + mu) * 9;
            pf[mu] = psi + xp * 12 * (long)N;
            pb[mu] = psi + xm * 12 * (long)N;
        }
        dhop_site(N, uf, ub, pf, pb, dirmask, out + x * 12 * (long)N);
    }
}

/* S4: M_eooe.  Same sum at the V/2 sites of parity out_parity,
 * reading the checkerboarded field psi_cb of parity 1 - out_parity.  Both fields
 * are indexed lex >> 1. */
void orc_meooe(const int dims[4], int N, const dc *U, const dc *psi_cb, dc *out_cb, int out_parity)
{
    long V = (long)dims[0] * dims[1] * dims[2] * dims[3];
#pragma omp parallel for schedule(static)
    for (long x = 0; x < V; x++) {
        if (parity_of(dims, x) != out_parity) continue;
        const dc *uf[4], *ub[4], *pf[4], *pb[4];
        for (int mu = 0; mu < 4; mu++) {
            long xp = neighbour(dims, x, mu, +1), xm = neighbour(dims, x, mu, -1);
            uf[mu] = U + (x * 4 + mu) * 9;
            ub[mu] = U + (xm * 4 + mu) * 9;
            pf[mu] = psi_cb + (xp >> 1) * 12 * (long)N;
            pb[mu] = psi_cb + (xm >> 1) * 12 * (long)N;
        }
        dhop_site(N, uf, ub, pf, pb, 0xFF, out_cb + (x >> 1) * 12 * (long)N);
    }
}

/* ------------------------------------------------------------------ clover */

static void su3_mul(const dc *a, const dc *b, dc *c)          /* c = a b */
{
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            dc s = 0.0;
            for (int k = 0; k < 3; k++) s += a[3 * i + k] * b[3 * k + j];
            c[3 * i + j] = s;
        }
}

static void su3_dag(const dc *a, dc *c)                       /* c = a^dagger */
{
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) c[3 * i + j] = conj(a[3 * j + i]);
}

/* product of four 3x3 matrices, each optionally daggered */
static void leaf(const dc *a, int da, const dc *b, int db, const dc *c, int dcg, const dc *d, int dd, dc *out)
{
    dc ta[9], tb[9], tc[9], td[9], t1[9], t2[9];
    if (da) su3_dag(a, ta); else memcpy(ta, a, sizeof ta);
    if (db) su3_dag(b, tb); else memcpy(tb, b, sizeof tb);
    if (dcg) su3_dag(c, tc); else memcpy(tc, c, sizeof tc);
    if (dd) su3_dag(d, td); else memcpy(td, d, sizeof td);
    su3_mul(ta, tb, t1); su3_mul(t1, tc, t2); su3_mul(t2, td, out);
}

static const dc *link_at(const dc *U, long x, int mu) { return U + (x * 4 + mu) * 9; }

/* S5: F_munu(x) = (Q - Q^dagger) / (8 i), Q = sum of the four plaquette leaves in
 * the mu-nu plane that start and end at x, all with the same orientation. */
static void field_strength(const int d[4], const dc *U, long x, int mu, int nu, dc *F)
{
    long xpm = neighbour(d, x, mu, +1), xpn = neighbour(d, x, nu, +1);
    long xmm = neighbour(d, x, mu, -1), xmn = neighbour(d, x, nu, -1);
    long xmm_pn = neighbour(d, xmm, nu, +1);
    long xmm_mn = neighbour(d, xmm, nu, -1);
    long xmn_pm = neighbour(d, xmn, mu, +1);
    dc Q[9], L[9];
    /* U_mu(x) U_nu(x+mu) U_mu(x+nu)^+ U_nu(x)^+ */
    leaf(link_at(U, x, mu), 0, link_at(U, xpm, nu), 0, link_at(U, xpn, mu), 1, link_at(U, x, nu), 1, Q);
    /* U_nu(x) U_mu(x-mu+nu)^+ U_nu(x-mu)^+ U_mu(x-mu) */
    leaf(link_at(U, x, nu), 0, link_at(U, xmm_pn, mu), 1, link_at(U, xmm, nu), 1, link_at(U, xmm, mu), 0, L);
    for (int i = 0; i < 9; i++) Q[i] += L[i];
    /* U_mu(x-mu)^+ U_nu(x-mu-nu)^+ U_mu(x-mu-nu) U_nu(x-nu) */
    leaf(link_at(U, xmm, mu), 1, link_at(U, xmm_mn, nu), 1, link_at(U, xmm_mn, mu), 0, link_at(U, xmn, nu), 0, L);
    for (int i = 0; i < 9; i++) Q[i] += L[i];
    /* U_nu(x-nu)^+ U_mu(x-nu) U_nu(x-nu+mu) U_mu(x)^+ */
    leaf(link_at(U, xmn, nu), 1, link_at(U, xmn, mu), 0, link_at(U, xmn_pm, nu), 0, link_at(U, x, mu), 1, L);
    for (int i = 0; i < 9; i++) Q[i] += L[i];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) F[3 * i + j] = (Q[3 * i + j] - conj(Q[3 * j + i])) / (8.0 * I);
}

void orc_field_strength(const int dims[4], const dc *U, long lex, int mu, int nu, dc *F9)
{
    field_strength(dims, U, lex, mu, nu, F9);
}

/* S6: the full 12x12 site matrix, row/col index 3*spin + colour:
 * M_ooee(x) = (4 + m) 1 - (c_sw/2) sum_{mu<nu} sigma_munu (x) F_munu(x). */
void orc_clover_site_matrix(const int dims[4], const dc *U, double mass, double csw, long lex, dc *M144)
{
    for (int i = 0; i < 144; i++) M144[i] = 0.0;
    for (int i = 0; i < 12; i++) M144[13 * i] = 4.0 + mass;
    for (int mu = 0; mu < 4; mu++)
        for (int nu = mu + 1; nu < 4; nu++) {
            dc S[4][4], F[9];
            sigma_mat(mu, nu, S);
            field_strength(dims, U, lex, mu, nu, F);
            for (int s = 0; s < 4; s++)
                for (int sp = 0; sp < 4; sp++)
                    for (int c = 0; c < 3; c++)
                        for (int cp = 0; cp < 3; cp++)
                            M144[(3 * s + c) * 12 + 3 * sp + cp] -= 0.5 * csw * S[s][sp] * F[3 * c + cp];
        }
}

/* S7: cut the two chiral 6x6 blocks out of the 12x12 site matrix.  C[lex][2][6][6].
 * Returns through *offdiag_max the largest |entry| found outside the two blocks
 * (a pin asserts it is zero). */
void orc_clover_blocks(const int dims[4], const dc *U, double mass, double csw, dc *C, double *offdiag_max)
{
    long V = (long)dims[0] * dims[1] * dims[2] * dims[3];
    double worst = 0.0;
#pragma omp parallel for schedule(static) reduction(max : worst)
    for (long x = 0; x < V; x++) {
        dc M[144];
        orc_clover_site_matrix(dims, U, mass, csw, x, M);
        for (int i = 0; i < 12; i++)
            for (int j = 0; j < 12; j++) {
                int bi = i / 6, bj = j / 6;
                if (bi == bj) C[((x * 2 + bi) * 6 + i % 6) * 6 + j % 6] = M[12 * i + j];
                else if (cabs(M[12 * i + j]) > worst) worst = cabs(M[12 * i + j]);
            }
    }
    if (offdiag_max) *offdiag_max = worst;
}

/* M_ooee apply: out(x) = C(x) psi(x), block b acts on spins
 * {2b, 2b+1}.  nsites is V (full field) or V/2 (one parity; C then holds the
 * blocks of that parity's sites in the same lex>>1 order). */
void orc_mooee(long nsites, int N, const dc *C, const dc *psi, dc *out)
{
#pragma omp parallel for schedule(static)
    for (long x = 0; x < nsites; x++)
        for (int b = 0; b < 2; b++)
            for (int i = 0; i < 6; i++)
                for (int r = 0; r < N; r++) {
                    dc acc = 0.0;
                    for (int j = 0; j < 6; j++)
                        acc += C[((x * 2 + b) * 6 + i) * 6 + j] * psi[(x * 12 + 6 * b + j) * (long)N + r];
                    out[(x * 12 + 6 * b + i) * (long)N + r] = acc;
                }
}

/* ------------------------------------------------------------------ coarse */

/* S8, one site: out[i][r] = sum_{p=0..8} sum_j A_p[i][j] v(x+delta_p)[j][r].
 * A9 -> [9][nb][nb]; nbr[p] -> v(x + delta_p) [nb][N]. */
static void coarse_site(int nb, int N, const dc *A9, const dc *const nbr[9], int pmask, dc *out)
{
    for (int i = 0; i < nb * N; i++) out[i] = 0.0;
    for (int p = 0; p < 9; p++) {
        if (!(pmask & (1 << p))) continue;
        const dc *A = A9 + (long)p * nb * nb;
        for (int i = 0; i < nb; i++)
            for (int j = 0; j < nb; j++)
                for (int r = 0; r < N; r++) out[i * N + r] += A[i * nb + j] * nbr[p][j * N + r];
    }
}

/* delta_0 = 0, delta_{1..4} = +mu, delta_{5..8} = -mu, periodic. */
void orc_coarse_apply(const int cdims[4], int nb, int N, const dc *A, const dc *v, dc *out, int pmask)
{
    long V = (long)cdims[0] * cdims[1] * cdims[2] * cdims[3];
#pragma omp parallel for schedule(static)
    for (long x = 0; x < V; x++) {
        const dc *nbr[9];
        nbr[0] = v + x * nb * (long)N;
        for (int mu = 0; mu < 4; mu++) {
            nbr[1 + mu] = v + neighbour(cdims, x, mu, +1) * nb * (long)N;
            nbr[5 + mu] = v + neighbour(cdims, x, mu, -1) * nb * (long)N;
        }
        coarse_site(nb, N, A + x * 9 * (long)nb * nb, nbr, pmask, out + x * nb * (long)N);
    }
}

/* Coarse M_eooe ("M_eooe" on the coarse levels): the 8-point hopping term of S8 at
 * the coarse sites x of parity out_parity only, reading v at sites of the other parity:
 *   out(x) = sum_{p=1..8} A_p(x) v(x + delta_p),   parity(x) = (x+y+z+t) mod 2.
 * v_cb [V/2][nb][N] holds the sites of parity 1 - out_parity, out [V/2][nb][N] those of parity out_parity, both ordered by
 * increasing lex (index lex >> 1; all coarse extents even).  A is the full-lattice link field [V][9][nb][nb]. */
void orc_coarse_meooe(const int cdims[4], int nb, int N, const dc *A, const dc *v_cb, dc *out, int out_parity)
{
    long V = (long)cdims[0] * cdims[1] * cdims[2] * cdims[3];
#pragma omp parallel for schedule(static)
    for (long x = 0; x < V; x++) {
        if (parity_of(cdims, x) != out_parity) continue;
        const dc *nbr[9];
        nbr[0] = NULL;                               /* the self term is not part of M_eooe */
        for (int mu = 0; mu < 4; mu++) {
            nbr[1 + mu] = v_cb + (neighbour(cdims, x, mu, +1) >> 1) * nb * (long)N;
            nbr[5 + mu] = v_cb + (neighbour(cdims, x, mu, -1) >> 1) * nb * (long)N;
        }
        coarse_site(nb, N, A + x * 9 * (long)nb * nb, nbr, 0x1FE, out + (x >> 1) * nb * (long)N);
    }
}

/* Packed per-site entry: A[nsites][9][nb][nb], nbrs[nsites][9][nb][N]. */
void orc_coarse_sites(long nsites, int nb, int N, const dc *A, const dc *nbrs, dc *out)
{
#pragma omp parallel for schedule(static)
    for (long i = 0; i < nsites; i++) {
        const dc *nbr[9];
        for (int p = 0; p < 9; p++) nbr[p] = nbrs + (i * 9 + p) * nb * (long)N;
        coarse_site(nb, N, A + i * 9 * (long)nb * nb, nbr, 0x1FF, out + i * nb * (long)N);
    }
}

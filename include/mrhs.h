/*
 * mrhs.h -- C ABI of the B200-native MRHS Wilson-clover stencil library.
 *
 * One data-parallel hot path of arxiv 2211.13719 ("MRHS multigrid solver for
 * Wilson-clover fermions"): the Wilson-clover stencil operators applied to
 * N_rhs right-hand sides at once, with the RHS index innermost so that each
 * gauge link, clover block or coarse link matrix fetched from HBM serves every
 * RHS (PAPER.md:23 benefit (i), "RHS index in the fifth dimension").
 * The paper prints no formula; the definitions implemented are the readings
 * S1-S8 of SURVEY.md Sec. 8(c), restated in DESIGN.md.
 *
 * Conventions common to every entry point
 *  - "d_" pointers are DEVICE pointers, "h_" pointers are HOST pointers.
 *  - All field data is single precision complex (two fp32).
 *  - Return value: MRHS_OK or an error code; never throws, never aborts.
 *    mrhs_last_error() returns a thread-local message for the last failure.
 *  - Applies enqueue work on the handle's stream and return without
 *    synchronising.  Asynchronous faults surface at the caller's next sync.
 *  - Handles are not thread-safe.  The current device at create time is the
 *    handle's device.  One GPU, periodic boundaries handled in-kernel, no
 *    communication (BASELINE.json north_star).
 *  - create copies/repacks gauge, clover and coarse links into device memory
 *    OWNED by the handle; the caller may free its buffers after create returns
 *    (create synchronises the stream before returning).  Field buffers are
 *    caller-owned, 16-byte aligned, and d_in must not alias d_out.
 *
 * Canonical layouts (C order, last index fastest):
 *   site    lex = x + X*(y + Y*(z + Z*t)), extents even and >= 2, periodic
 *   spinor  psi[lex][spin 4][colour 3][rhs N]   complex64 (re,im interleaved)
 *   checkerboarded spinor of parity p: the V/2 sites with (x+y+z+t)%2 == p in
 *           increasing lex order (index lex >> 1)
 *   gauge   U[lex][mu 4][row 3][col 3], mu = x,y,z,t; U_mu(x) links x -> x+mu
 *   clover  C[lex][chirality 2][6][6], block index 3*(spin%2)+colour
 *   coarse links  A[lex][p 9][row nb][col nb]; p=0 self, 1..4 = +x..+t, 5..8 = -x..-t
 *   coarse vector v[lex][nb][rhs N]
 *
 * Native layouts (what the timed applies read and write).
 * Fine fields (ncomp == 12):
 *   x-lines are cut in blocks of XB = mrhs_xblock(X_eff, N) sites (largest divisor of X_eff
 *   with XB <= 16 and XB * threads-per-site <= 48), X_eff = X
 *   for a full field and X/2 for a checkerboarded one (site xh of a parity-p
 *   line has x = 2*xh + ((p+y+z+t)&1)).  Block b = xb + (X_eff/XB)*(y + Y*(z + Z*t)).
 *   float index = ((b*12 + comp)*XB + x_in)*2N + e, comp = 3*spin + colour, with
 *     N even: e = 4*(r/2) + (r&1) + 2*im   (RHS pairs stored re0 re1 im0 im1)
 *     N odd : e = 2*r + im
 *   i.e. the RHS index is fastest, then the site inside the block, then the
 *   spin-colour component, so that a warp reads 512 contiguous bytes per load.
 * Coarse fields (ncomp == nbasis): v[lex][nb][rhs] with the same RHS-pair
 *   element order e as above (site-contiguous, fetched by bulk copies).
 * The helpers below convert; the applies never do.
 */
#ifndef MRHS_H
#define MRHS_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mrhs_wilson mrhs_wilson_t;       /* opaque: owns packed gauge + clover */
typedef struct mrhs_coarse mrhs_coarse_t;       /* opaque: owns packed coarse links */
typedef struct mrhs_transfer mrhs_transfer_t;   /* opaque: owns the repacked multigrid basis vectors */

typedef enum {
    MRHS_OK = 0,
    MRHS_ERR_INVALID_ARG = 1,   /* NULL pointer, odd or < 2 extent, bad parity, misalignment, overlapping in and out buffers */
    MRHS_ERR_UNSUPPORTED = 2,   /* N_rhs or nbasis without a compiled specialisation */
    MRHS_ERR_ALLOC = 3,         /* device or host allocation failed */
    MRHS_ERR_CUDA = 4           /* a CUDA runtime call or kernel launch failed */
} mrhs_status_t;

/* Parity arguments: 0 = even sites, 1 = odd sites, 2 = full lattice. */
#define MRHS_EVEN 0
#define MRHS_ODD 1
#define MRHS_FULL 2

/* ------------------------------------------------------------------ fine level */

/* Build a fine-level handle for lattice dims = {X,Y,Z,T} and N_rhs = nrhs
 * (1..128; UNSUPPORTED above).
 *   d_gauge : device, canonical gauge field, required.
 *   d_clover: device, canonical clover blocks, or NULL.  NULL => the blocks
 *             M_ooee(x) = (4+mass) - (csw/2) sum_{mu<nu} sigma_munu F_munu(x)
 *             (readings S5-S7) are built on the device from d_gauge, mass, csw.
 *             When given, mass and csw are not used by mrhs_mooee.
 *   cuda_stream: a cudaStream_t (NULL = default stream); every later apply on
 *             this handle is enqueued on it.
 * PAPER.md:43 (D_hop, M_eooe), PAPER.md:47,:53 (precomputed clover term). */
mrhs_status_t mrhs_wilson_create(mrhs_wilson_t **out, const int dims[4], int nrhs,
                                 float mass, float csw,
                                 const void *d_gauge, const void *d_clover,
                                 void *cuda_stream);

/* D_hop on the full lattice (reading S3):
 *   out(x) = sum_mu (1-gamma_mu) U_mu(x) in(x+mu) + (1+gamma_mu) U_mu(x-mu)^+ in(x-mu)
 * bare sum (no -1/2, no mass), 1320 flops per site per RHS.
 * d_in, d_out: native full-lattice fields, mrhs_field_bytes(dims,12,nrhs,0) each. */
mrhs_status_t mrhs_dhop(mrhs_wilson_t *h, const void *d_in, void *d_out);

/* M_eooe (reading S4): the same sum evaluated at the V/2 sites of
 * parity out_parity (0 or 1), reading the checkerboarded field of the other
 * parity.  d_in, d_out: native checkerboarded fields. */
mrhs_status_t mrhs_meooe(mrhs_wilson_t *h, const void *d_in, void *d_out, int out_parity);

/* M_ooee (readings S6, S7): out(x) = C(x) in(x), two 6x6
 * Hermitian chiral blocks per site, includes the (4+mass) diagonal.
 * parity 0/1: checkerboarded fields of that parity; 2: full-lattice fields. */
mrhs_status_t mrhs_mooee(mrhs_wilson_t *h, const void *d_in, void *d_out, int parity);

/* M_ooee^-1 ("precomputed"): out(x) = C(x)^-1 in(x).  The inverse
 * blocks are computed once at create (fp64 Gauss-Jordan per 6x6 block, stored fp32 in the same packed
 * Hermitian form), so the apply is the same kernel with the same cost as mrhs_mooee.  A singular
 * user-supplied block gives non-finite entries in its inverse (not checked). */
mrhs_status_t mrhs_mooee_inv(mrhs_wilson_t *h, const void *d_in, void *d_out, int parity);

/* The full Wilson-clover matrix on full-lattice fields (reading S6):
 *   out = M in = M_ooee in - (1/2) D_hop in.
 * With the sweep kernel ONE launch (the clover term of in(x) is formed from the slice in shared
 * memory and the eight hops are added to it: no intermediate field, no separate axpy); with the
 * gather kernel two launches (D_hop, then out = C in - out / 2). */
mrhs_status_t mrhs_wilson_apply(mrhs_wilson_t *h, const void *d_in, void *d_out);

/* Fused out = M_ooee(out_parity) M_eooe(in): the hopping term onto parity out_parity followed by
 * the clover term of those sites (the first two steps of the Schur
 * sequence below).  With the sweep kernel (even N_rhs) this is ONE
 * launch: the clover blocks are applied to the hop result in registers before it is stored, so the
 * intermediate field never goes through HBM.  With the gather kernel it is two launches.
 * d_in: native field of parity 1 - out_parity; d_out: native field of parity out_parity. */
mrhs_status_t mrhs_meooe_mooee(mrhs_wilson_t *h, const void *d_in, void *d_out, int out_parity);
/* The same with the inverse blocks: out = M_ooee(out_parity)^-1 M_eooe(in), the inner part of the
 * even-odd (Schur) preconditioned operator. */
mrhs_status_t mrhs_meooe_mooee_inv(mrhs_wilson_t *h, const void *d_in, void *d_out, int out_parity);

/* Schur-style sequence of config 5, back to back on the handle's
 * stream with no host synchronisation:
 *   tmp_o = M_eooe(in_e -> odd); tmp2_o = M_ooee(tmp_o); out_e = M_eooe(tmp2_o -> even).
 * With the sweep kernel the first two steps are one fused launch (mrhs_meooe_mooee) that writes
 * tmp2_o into d_tmp1 and leaves d_tmp0 untouched; with the gather kernel three launches.
 * d_in, d_out: even checkerboarded native fields; d_tmp0, d_tmp1: odd ones. */
mrhs_status_t mrhs_schur_sequence(mrhs_wilson_t *h, const void *d_in, void *d_tmp0,
                                  void *d_tmp1, void *d_out);

/* Adjoint operators (reading S3): D_hop^+ = gamma_5 D_hop gamma_5,
 *   (D_hop^+ in)(x) = sum_mu (1+gamma_mu) U_mu(x) in(x+mu) + (1-gamma_mu) U_mu(x-mu)^+ in(x-mu),
 * the same links with the projector signs exchanged; M_eooe^+ is the same sum at the sites of out_parity (it maps a field
 * of parity 1 - out_parity to one of parity out_parity, like mrhs_meooe); M^+ = M_ooee - D_hop^+ / 2 (the clover blocks are
 * Hermitian).  Same kernels, same cost, same argument rules as the plain calls. */
mrhs_status_t mrhs_dhop_dag(mrhs_wilson_t *h, const void *d_in, void *d_out);
mrhs_status_t mrhs_meooe_dag(mrhs_wilson_t *h, const void *d_in, void *d_out, int out_parity);
mrhs_status_t mrhs_wilson_apply_dag(mrhs_wilson_t *h, const void *d_in, void *d_out);

/* The even-odd preconditioned operator (Schur complement of M on the even sites; PAPER.md:43,
 * :53 "precomputed clover term"; reading S6 with M_eo = -M_eooe / 2):
 *   out = S in,  S = M_ee - M_eo M_oo^-1 M_oe = C_e - M_eooe(e<-o) C_o^-1 M_eooe(o<-e) / 4,    dagger != 0: S^+ (daggered hops).
 * d_in, d_out: native EVEN fields; d_tmp: native ODD scratch field (overwritten); all three distinct.  Sweep kernel: three
 * launches (C_o^-1 rides in the first hop's epilogue; plain hop; clover kernel forming C_e in - ... / 4); gather kernel: four. */
mrhs_status_t mrhs_schur_apply(mrhs_wilson_t *h, const void *d_in, void *d_tmp, void *d_out, int dagger);

/* Copy the handle's native clover blocks back in canonical form
 * d_clover_out[lex][2][6][6] complex64 (parity check of the device-side
 * construction, row a0). */
mrhs_status_t mrhs_wilson_export_clover(mrhs_wilson_t *h, void *d_clover_out);

/* Optional tuning knobs (defaults are chosen at create from the lattice, N_rhs
 * and the L2 size).  which: 0 = D_hop (full), 1 = M_eooe (checkerboarded).
 * tile = {by, bz, bt}: sites per thread-block tile in y,z,t (x extent is the
 * layout block XB); chunk = {cy, cz}: tiles per L2 sweep chunk in y and z.
 * Each must divide the lattice accordingly; INVALID_ARG otherwise. */
mrhs_status_t mrhs_wilson_set_tiling(mrhs_wilson_t *h, int which, const int tile[3], const int chunk[2]);
mrhs_status_t mrhs_wilson_get_tiling(mrhs_wilson_t *h, int which, int tile[3], int chunk[2]);
/* L2 prefetch distance of the hopping kernel, in thread-block tiles of its sweep order: a tile
 * asks the copy engine to bring the rows of the tile distance_tiles later into L2 (0 = off).
 * set_tiling resets it to the default (296 tiles: half of the tiles resident on 148 SMs at four per SM).
 * While the sweep kernel is selected for `which`, the call sets ITS prefetch distance instead, in t-slices
 * (default 0 = off: measured to add DRAM traffic and no speed; set_sweep keeps it).  The environment variable MRHS_DEBUG=1 makes create calls print
 * their launch geometry to stderr; nothing else in the library reads the environment. */
mrhs_status_t mrhs_wilson_set_prefetch(mrhs_wilson_t *h, int which, int distance_tiles);


/* The hopping term has two kernels computing the same map:
 *   MRHS_HOP_GATHER  every thread gathers its eight neighbours from global memory through L1/L2
 *                    (any N_rhs; the only kernel for odd N_rhs);
 *   MRHS_HOP_SWEEP   a thread block sweeps a t-segment of an XB x 2 x 2 tile with the current slice,
 *                    its halo and the links staged in shared memory by TMA bulk copies (even N_rhs;
 *                    the default where it measured faster: from N_rhs = 24 at 16^4 sites, 12 at 24^4, 4 at 32^4).
 * which: 0 = D_hop, 1 = M_eooe.  UNSUPPORTED if the sweep kernel is asked for with odd N_rhs.
 * set_sweep: lt = t-slices one thread block sweeps (divides T); chunk = {cy, cz}: tiles (of 2 x 2
 * sites in y,z) per concurrently scheduled patch; INVALID_ARG if they do not divide the lattice.
 * With lt = T the last tiles of the dispatch order are cut into shorter t-segments by the library so that the
 * last wave of thread blocks is balanced; results do not depend on any of these settings (bit-identical). */
#define MRHS_HOP_GATHER 0
#define MRHS_HOP_SWEEP 1
mrhs_status_t mrhs_wilson_set_hop_kernel(mrhs_wilson_t *h, int which, int kernel);
mrhs_status_t mrhs_wilson_get_hop_kernel(mrhs_wilson_t *h, int which, int *kernel);
mrhs_status_t mrhs_wilson_set_sweep(mrhs_wilson_t *h, int which, int lt, const int chunk[2]);
mrhs_status_t mrhs_wilson_get_sweep(mrhs_wilson_t *h, int which, int *lt, int chunk[2]);

mrhs_status_t mrhs_wilson_destroy(mrhs_wilson_t *h);

/* Launch plan of the sweep kernel for a lattice, computed on the host (no device needed; what a handle on a device with
 * num_sms multiprocessors would launch with its default settings).  parity: MRHS_FULL = D_hop, 0 / 1 = M_eooe with that
 * output parity.  plan[0..8] = {thread blocks, threads per block, tiles (XB x 2 x 2 sites each), whole-line blocks,
 * tail tiles, t-segments per tail tile, slices per whole block (lt), cy, cz}.  UNSUPPORTED if the sweep kernel cannot
 * run the geometry (odd N_rhs, shared memory).  mrhs_sweep_blocks: the tile segments that blocks first .. first + count - 1
 * of that plan sweep, coords[5 i ..] = {x-block, first y, first z, first t, slices}: the same index function the kernel
 * evaluates. */
mrhs_status_t mrhs_sweep_plan(const int dims[4], int nrhs, int parity, int num_sms, int plan[9]);
mrhs_status_t mrhs_sweep_blocks(const int dims[4], int nrhs, int parity, int num_sms, int first, int count, int *coords);

/* ---------------------------------------------------------------- coarse level */

/* Coarse-level handle (reading S8; PAPER.md:61 nbasis, PAPER.md:75 coarse hopping).
 *   cdims: coarse lattice extents (>= 2; need not be even), nbasis in {24, 40},
 *   nrhs in {1,2,4,8,12,16,24,32,48,64,96};
 *   d_links: device, canonical A[lex][9][nb][nb];
 *   math_mode: 0 = FP32 FMA; 1 = tensor cores, tf32 split precision (three kind::tf32 MMAs per K step on hi / lo parts made in
 *   the kernel); 2 = tensor cores, fp16 split precision (kind::f16 on hi + lo fp16 parts after an exact power-of-two scaling:
 *   the link field is split once here, one scale per site, and keeps its size; every apply first splits its input vector into
 *   a scratch image owned by the handle (2 nbasis (2 N_rhs rounded up to 16) fp16 per site), one scale per right-hand side
 *   taken from that RHS's largest magnitude over the field).  Modes 1 and 2 need even nrhs and are held to the same 1e-5
 *   tolerance per RHS (reading S15); in mode 2 an element smaller than 2^-17 of the largest element of its RHS (or, for the
 *   links, of its site) carries an absolute error of 2^-40 of that largest element instead of a relative one. */
mrhs_status_t mrhs_coarse_create(mrhs_coarse_t **out, const int cdims[4], int nbasis, int nrhs,
                                 const void *d_links, int math_mode, void *cuda_stream);

/* out_i(x) = sum_{p=0..8} sum_j A_p(x)_ij in_j(x + delta_p), periodic;
 * 72 nb^2 flops per site per RHS.  d_in, d_out: native coarse vectors. */
mrhs_status_t mrhs_coarse_apply(mrhs_coarse_t *h, const void *d_in, void *d_out);

/* The same apply restricted to a subset of the nine stencil points (
 * PAPER.md:75 benchmarks the coarse hopping term without the self term, reading S12):
 *   out(x) = sum over p with bit p of point_mask set of A_p(x) in(x + delta_p),
 * p = 0 self, 1..4 = +x..+t, 5..8 = -x..-t.  MRHS_COARSE_SELF is the stand-alone coarse clover
 * (self) term, MRHS_COARSE_HOP the 8-point coarse hopping term (M_eooe + M_oeeo on full-lattice
 * fields), MRHS_COARSE_ALL the 9-point operator.  Both math modes.  INVALID_ARG for an empty mask. */
#define MRHS_COARSE_SELF 0x001
#define MRHS_COARSE_HOP 0x1FE
#define MRHS_COARSE_ALL 0x1FF
mrhs_status_t mrhs_coarse_apply_points(mrhs_coarse_t *h, const void *d_in, void *d_out, int point_mask);

/* Coarse M_eooe (Sec. 6: "M_eooe" on both coarse levels): the 8-point coarse
 * hopping term at the coarse sites of parity out_parity, reading a field of the other parity,
 *   out(x) = sum_{p=1..8} A_p(x) in(x + delta_p),  parity(x) = (x+y+z+t) mod 2 = out_parity.
 * d_in: native checkerboarded coarse vector of parity 1 - out_parity, d_out: of parity out_parity (V/2 sites each, made by
 * mrhs_coarse_field_import / mrhs_coarse_cb_split); the link matrices are the handle's full-lattice field.  Both math
 * modes (same kernels with a parity site map).  64 nb^2 flops per output site per RHS.  INVALID_ARG: odd coarse extent,
 * bad parity, aliasing. */
mrhs_status_t mrhs_coarse_meooe(mrhs_coarse_t *h, const void *d_in, void *d_out, int out_parity);

mrhs_status_t mrhs_coarse_destroy(mrhs_coarse_t *h);

/* ------------------------------------------------- layout helpers (untimed) */

/* Layout block extent along x for a line of x_eff sites and N_rhs = nrhs. */
int mrhs_xblock(int x_eff, int nrhs);

/* Bytes of a native field: ncomp = 12 (fine) or nbasis (coarse);
 * checkerboarded != 0 => one parity (V/2 sites).  0 on invalid arguments. */
size_t mrhs_field_bytes(const int dims[4], int ncomp, int nrhs, int checkerboarded);

/* canonical -> native and back.  parity 0/1: checkerboarded field of that
 * parity (canonical side has V/2 sites in lex>>1 order); 2: full field.
 * Pure data movement, bit-exact round trip. */
mrhs_status_t mrhs_field_import(const int dims[4], int ncomp, int nrhs, int parity,
                                const void *d_canonical, void *d_native, void *cuda_stream);
mrhs_status_t mrhs_field_export(const int dims[4], int ncomp, int nrhs, int parity,
                                const void *d_native, void *d_canonical, void *cuda_stream);

/* full native <-> (even native, odd native). */
mrhs_status_t mrhs_cb_split(const int dims[4], int ncomp, int nrhs, const void *d_full,
                            void *d_even, void *d_odd, void *cuda_stream);
mrhs_status_t mrhs_cb_merge(const int dims[4], int ncomp, int nrhs, const void *d_even,
                            const void *d_odd, void *d_full, void *cuda_stream);

/* The four calls above choose the layout from ncomp: 12 = fine spinor (x-blocked, Sec. "Native layouts"), anything else =
 * coarse vector (site-contiguous [site][component][rhs]).  A coarse level whose vectors happen to have 12 components
 * (n_vec = 6) must say so: these entries always use the COARSE layout.  parity 0/1 = checkerboarded coarse field of that
 * parity (V/2 sites ordered by lex, index lex >> 1; needs even extents), 2 = full.  (NEXT-1.) */
mrhs_status_t mrhs_coarse_field_import(const int cdims[4], int nbasis, int nrhs, int parity,
                                       const void *d_canonical, void *d_native, void *cuda_stream);
mrhs_status_t mrhs_coarse_field_export(const int cdims[4], int nbasis, int nrhs, int parity,
                                       const void *d_native, void *d_canonical, void *cuda_stream);
mrhs_status_t mrhs_coarse_cb_split(const int cdims[4], int nbasis, int nrhs, const void *d_full,
                                   void *d_even, void *d_odd, void *cuda_stream);
mrhs_status_t mrhs_coarse_cb_merge(const int cdims[4], int nbasis, int nrhs, const void *d_even,
                                   const void *d_odd, void *d_full, void *cuda_stream);

/* ------------------------------------------- intergrid operators (projection / promotion) */

/* MRHS prolongation and restriction between the fine level and its first coarse level (SURVEY.md
 * Sec. 8(f) NEXT-3; reading S9).  n_vec basis vectors phi_k, nbasis = 2 n_vec, chirality
 * chi = 0 for spins {0,1}, 1 for spins {2,3}, coarse index j = chi n_vec + k, blocks of bdims fine sites:
 *   prolong:   fine(x)[s][c][r]  = sum_k phi_k(x)[s][c] coarse(B(x))[chi(s) n_vec + k][r]
 *   restrict:  coarse(B)[chi n_vec + k][r] = sum_{x in B, s in chi, c} conj(phi_k(x)[s][c]) fine(x)[s][c][r]
 * (restrict is the adjoint of prolong; the basis is used as given, orthonormalising it is the setup's job).
 * create: dims fine extents, bdims block extents (each divides the fine extent, coarse extent >= 2);
 *   d_basis: device, canonical [n_vec][site][4][3] complex64, copied and repacked (caller may free it).
 * prolong: d_coarse_in native coarse vector (ncomp = 2 n_vec, COARSE layout: mrhs_coarse_field_import, which is what
 *   mrhs_field_import does for ncomp != 12; with n_vec = 6 the explicit coarse entry is required) of the coarse lattice
 *   dims / bdims, d_fine_out native full-lattice fine field; restrict the other way.  Asynchronous on the stream.
 * UNSUPPORTED: aggregates whose index table and reduction scratch do not fit 100 KB of shared memory (> ~2000 sites). */
mrhs_status_t mrhs_transfer_create(mrhs_transfer_t **out, const int dims[4], const int bdims[4], int nvec,
                                   int nrhs, const void *d_basis, void *cuda_stream);
/* The same pair one level up (the operators between the intermediate and the coarsest level, nbasis 40
 * -> 60 in the paper's solve, where it reports its largest intergrid gains): the "fine" field is a coarse vector of nf
 * components per site (nf a multiple of 4; chirality chi(c) = 0 for c < nf / 2, else 1) on the lattice fdims, in the COARSE
 * native layout (mrhs_coarse_field_import); blocks of bdims of its sites:
 *   prolong:   out(x)[c][r] = sum_k phi_k(x)[c] coarse(B(x))[chi(c) n_vec + k][r]
 *   restrict:  coarse(B)[chi n_vec + k][r] = sum_{x in B, c in chi} conj(phi_k(x)[c]) in(x)[c][r]
 * d_basis: device, canonical [n_vec][site][nf] complex64, copied and repacked.  The handle is used with mrhs_prolong /
 * mrhs_restrict / mrhs_transfer_destroy like a fine-level one.  UNSUPPORTED (at restrict): more than 256 (chirality, basis
 * pair, RHS lane group) items per aggregate. */
mrhs_status_t mrhs_transfer_create_coarse(mrhs_transfer_t **out, const int fdims[4], const int bdims[4], int nf, int nvec,
                                          int nrhs, const void *d_basis, void *cuda_stream);
mrhs_status_t mrhs_prolong(mrhs_transfer_t *h, const void *d_coarse_in, void *d_fine_out);
mrhs_status_t mrhs_restrict(mrhs_transfer_t *h, const void *d_fine_in, void *d_coarse_out);
mrhs_status_t mrhs_transfer_destroy(mrhs_transfer_t *h);

/* ------------------------------------------- block reductions over the RHS index */

/* Simultaneous inner products:
 *   result[r] = sum over sites and components of conj(x[..., r]) y[..., r],   r = 0 .. nrhs-1.
 * d_x, d_y: two fields of the same geometry in NATIVE layout (fine: ncomp = 12, coarse: ncomp =
 * nbasis; parity 0/1 checkerboarded, 2 full).  d_result: device, nrhs complex128 (re, im doubles),
 * 16-byte aligned.  One pass over both fields, products and sums in fp64, fixed summation order
 * (bit-reproducible).  Asynchronous on cuda_stream (scratch is allocated stream-ordered). */
mrhs_status_t mrhs_inner_products(const int dims[4], int ncomp, int nrhs, int parity,
                                  const void *d_x, const void *d_y, void *d_result, void *cuda_stream);

/* The same operation for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): no cudaMalloc / cudaMallocAsync / cudaFree and no allocating library routine is called.  The per-block
 * partial sums live in a static __device__ array of the library (2 MiB = 131072 complex128 partial sums, held by every GPU
 * that loads the library until the process exits) instead of stream-ordered scratch.  Same arguments, same kernels, same
 * thread-block count and summation order as mrhs_inner_products: the results are bit-identical.
 *   Limit: (8 x SM count) x nrhs <= 131072, i.e. nrhs <= 110 on a 148-SM B200; beyond it MRHS_ERR_UNSUPPORTED with a message
 *   naming both numbers (nothing is launched).  The lattice size is not limited.
 *   Every call on a device shares the one array: calls that overlap on the GPU (different streams, no ordering between
 *   them) RACE on it; calls on one stream, or ordered by events, are safe.  The array keeps the last call's contents;
 *   nothing needs clearing, because a call writes every partial sum it later reads.
 *   The first call on a device looks the array's device address up (cudaGetSymbolAddress, no allocation) and caches it;
 *   make that first call outside a graph capture.  Asynchronous on cuda_stream. */
mrhs_status_t mrhs_inner_products_noalloc(const int dims[4], int ncomp, int nrhs, int parity,
                                          const void *d_x, const void *d_y, void *d_result, void *cuda_stream);

/* ------------------------------------------- host-buffer (end-to-end) entries */

/* One operator apply with HOST buffers in CANONICAL layout: host->device copy,
 * import, the same kernel the device entry launches, export, device->host copy,
 * then a stream synchronise.  op: 0 = D_hop, 1 = M_eooe, 2 = M_ooee, 3 = the Schur
 * sequence of mrhs_schur_sequence (even field in, even field out).
 * parity: out parity for op 1; field parity (0,1,2) for op 2; ignored for ops 0 and 3.
 * Staging buffers are owned by the handle and allocated on first use. */
mrhs_status_t mrhs_wilson_apply_host(mrhs_wilson_t *h, int op, int parity,
                                     const void *h_in, void *h_out);
mrhs_status_t mrhs_coarse_apply_host(mrhs_coarse_t *h, const void *h_in, void *h_out);
/* The same without the final synchronise: the call returns once its copies and kernels are enqueued, and
 * mrhs_*_host_wait blocks until every enqueued call of the handle has delivered its result.  h_in and h_out must stay
 * valid (and should be pinned, else the copies serialise) until then; results of different calls must not alias.
 * The handle cycles through three staging slots: the host->device copy of a call runs under the kernels and the
 * device->host copy of the call before (one copy stream per direction, events in between), so a sequence of calls
 * uses both directions of the link at once.  Calls are executed in the order they were made. */
mrhs_status_t mrhs_wilson_apply_host_async(mrhs_wilson_t *h, int op, int parity,
                                           const void *h_in, void *h_out);
mrhs_status_t mrhs_wilson_host_wait(mrhs_wilson_t *h);
mrhs_status_t mrhs_coarse_apply_host_async(mrhs_coarse_t *h, const void *h_in, void *h_out);
mrhs_status_t mrhs_coarse_host_wait(mrhs_coarse_t *h);

/* ------------------------------------------------------------------- errors */

const char *mrhs_last_error(void);   /* thread-local, valid until the next call */
const char *mrhs_version(void);      /* build string incl. target arch */

#ifdef __cplusplus
}
#endif
#endif /* MRHS_H */

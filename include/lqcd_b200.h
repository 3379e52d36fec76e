/*
 * lqcd_b200.h -- C ABI of the B200 (sm_100a) hot path of arXiv:2111.05012:
 * the Dirac-operator matrix-vector products of the multigrid-preconditioned solve.
 *
 * Citations are PAPER.md:<line> (the paper text) and SURVEY.md section 8 (the scope contract);
 * every reading of a point the paper leaves open is listed in DESIGN.md "Readings".
 *
 * Conventions (the paper fixes none of them):
 *   dims = {Lx, Ly, Lz, Lt}; mu = 0..3 <-> x, y, z, t (paper's mu = 1..4); sites 0-based;
 *   canonical site index  s = x + Lx (y + Ly (z + Lz t)),  V = Lx Ly Lz Lt;
 *   block b[4] divides dims; coarse dims Lc = dims / b (each >= 2); coarse site
 *   X = Xx + Lcx (Xy + Lcy (Xz + Lcz Xt)), Vc = prod Lc; N = 2 nvec coarse dofs per coarse site,
 *   coarse component  c = chi * nvec + i,  chi = alpha / 2 the chirality block of spin alpha.
 *   Gamma matrices: chiral basis of DESIGN.md (gamma5 = -g1 g2 g3 g4 = diag(-1,-1,+1,+1), Eq. 2,
 *   PAPER.md:54).  Complex numbers are interleaved (re, im).
 *
 * CANONICAL layouts (what the pack kernels read / unpack kernels write; x = fastest index last):
 *   spinor      psi[s][alpha][c]                 V*12 complex
 *   gauge       U[mu][s][a][b], (U psi)_a = sum_b U_ab psi_b     4*V*9 complex
 *   clover      F[s][chi][k][l], k = 3*(alpha%2)+c, Hermitian 6x6 blocks       V*2*36 complex
 *   null vecs   v[i][s][alpha][c]                nvec*V*12 complex
 *   coarse vec  x[X][chi][i]                     Vc*N complex
 *   coarse mat  A[X][d][row][col], d = 0 diag, 1+2mu forward, 2+2mu backward   Vc*9*N*N complex
 *
 * NATIVE layouts (what the mult kernels consume; sizes from lqcd_native_*_reals; R = real type,
 * a "vec16" is 16 bytes = 4 floats or 2 doubles; sites are grouped in chunks of 32: site s sits at
 * native position n(s), chunk = n / 32, lane = n % 32, nchunk = ceil(V / 32).  Site order: when
 * Lx % 4 == Ly % 4 == Lz % 2 == 0 a chunk is a 4 x 4 x 2 tile of sites (x, y, z), tiles in
 * lexicographic order, n = 32 (x/4 + (Lx/4) (y/4 + (Ly/4) (z/2 + (Lz/2) t))) + x%4 + 4 (y%4) + 16 (z%2)
 * -- every 128-byte line then belongs to one 4^4 domain; otherwise n(s) = s (canonical order).  The
 * native layouts are opaque to callers: pack / unpack are the only calls that speak them):
 *   spinor   [chunk][j][lane] vec16, j = 0..24/nv-1 over the 24 reals r = 2*(3 alpha + c) + reim
 *   gauge18  [chunk][mu][18 reals as 18/nv full vec16 rows of 32 lanes, then (f32 only) one row of
 *            32 float2 holding reals 16,17], reals r = 2*(3a+b)+reim
 *   gauge12  [chunk][mu][j][lane] vec16 over the 12 reals of rows a = 0,1; the third row is rebuilt
 *            in the kernel as conj(row0 x row1)
 *   clover   [chunk][j][lane] vec16 over 72 reals: per chi 6 real diagonal entries then the 15
 *            complex entries below the diagonal in row-major order (1,0),(2,0),(2,1),(3,0),...
 *            (only the Hermitian part of the canonical input is kept)
 *   null vecs [X][chi][i][l][k] complex, l = local site index inside the block (x fastest),
 *            k = 3*(alpha%2)+c -- one contiguous (|block|*6)-complex vector per (X, chi, i)
 *   coarse vec, coarse mat: identical to canonical.
 *
 * All pointers named *_dev / without suffix are DEVICE pointers owned by the caller and must be
 * 16-byte aligned; *_host are HOST pointers.  No call allocates device memory, none keeps state
 * beyond a thread-local error string and the tuning knobs below.  Every call enqueues its work on
 * `stream` (a cudaStream_t passed as void*; NULL = legacy default stream) and returns without
 * synchronising, except the *_host_* calls, which synchronise the stream before returning.
 *
 * Return value: 0 = LQCD_OK; negative = error and NOTHING was enqueued:
 *   LQCD_EINVAL (-1)        null pointer, misaligned pointer, non-positive dim, block not dividing
 *                           dims, coarse extent < 2, bc[mu] not in {+1,-1}, nvec < 1, out == in
 *   LQCD_EUNSUPPORTED (-2)  size outside a kernel's compiled range
 *   LQCD_ECUDA (-3)         the launch reported an error (text in lqcd_last_error())
 * There is no CPU fallback and no other GPU architecture.
 */
#ifndef LQCD_B200_H
#define LQCD_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LQCD_OK 0
#define LQCD_EINVAL (-1)
#define LQCD_EUNSUPPORTED (-2)
#define LQCD_ECUDA (-3)

/* flags */
#define LQCD_DAGGER 1u   /* apply gamma5 D gamma5 = D^dag (Eq. 2) / Gamma5c D_c Gamma5c */
#define LQCD_LINKS_12 2u /* U holds the 12-real compressed native gauge layout */
#define LQCD_DOMAIN_EVEN 4u /* lqcd_wilson_clover_dd_mult only: compute even domains, zero elsewhere */
#define LQCD_DOMAIN_ODD 8u  /* lqcd_wilson_clover_dd_mult only: compute odd domains, zero elsewhere */
#define LQCD_ACCUMULATE 16u /* lqcd_mr_domain_solve: z += M r on the selected domains, other sites untouched */
#define LQCD_SAP_INITIAL_GUESS 32u     /* lqcd_sap: x holds x0 on entry; start from r = b - D x0 instead of x = 0 */
#define LQCD_SAP_NO_FINAL_RESIDUAL 64u /* lqcd_sap: skip the last r = b - D x (r is then NOT the final residual) */

/* ---- diagnostics ------------------------------------------------------------------------- */
int lqcd_version(void);
/* Text of the last error on this thread ("" if none).  Owned by the library. */
const char* lqcd_last_error(void);
/* Number of kernel launches this library has enqueued so far (all threads). */
unsigned long long lqcd_launch_count(void);

/* ---- tuning knobs (process-wide; defaults chosen for B200; results never depend on them) --- */
/* Thread tile of the fine kernel: tile[mu] sites per CTA in direction mu, product <= 256,
 * each dividing dims[mu] at call time (otherwise the call falls back to the automatic choice).
 * tile = NULL or tile[0] = 0 restores the automatic choice. */
int lqcd_set_fine_tile(const int tile[4]);
/* Generic integer knob by name; returns LQCD_EINVAL for an unknown name. */
int lqcd_set_knob(const char* name, int value);

/* ---- native sizes, in reals of the precision in use -------------------------------------- */
size_t lqcd_native_spinor_reals(const int dims[4]);
size_t lqcd_native_gauge_reals(const int dims[4], unsigned flags /* LQCD_LINKS_12 or 0 */);
size_t lqcd_native_clover_reals(const int dims[4]);
size_t lqcd_native_nullvecs_reals(const int dims[4], const int block[4], int nvec);
size_t lqcd_native_coarse_vec_reals(const int cdims[4], int nvec);
size_t lqcd_native_coarse_mat_reals(const int cdims[4], int nvec);

/* ---- layout helpers: device -> device re-layout kernels (not on the timed path) ---------- */
int lqcd_pack_spinor_f32(float* dst_native, const float* src_canonical, const int dims[4], void* stream);
int lqcd_pack_spinor_f64(double* dst_native, const double* src_canonical, const int dims[4], void* stream);
int lqcd_unpack_spinor_f32(float* dst_canonical, const float* src_native, const int dims[4], void* stream);
int lqcd_unpack_spinor_f64(double* dst_canonical, const double* src_native, const int dims[4], void* stream);
/* flags: LQCD_LINKS_12 packs rows 0,1 only */
int lqcd_pack_gauge_f32(float* dst_native, const float* src_canonical, const int dims[4], unsigned flags,
                        void* stream);
int lqcd_pack_gauge_f64(double* dst_native, const double* src_canonical, const int dims[4], unsigned flags,
                        void* stream);
int lqcd_pack_clover_f32(float* dst_native, const float* src_canonical, const int dims[4], void* stream);
int lqcd_pack_clover_f64(double* dst_native, const double* src_canonical, const int dims[4], void* stream);
int lqcd_unpack_clover_f32(float* dst_canonical, const float* src_native, const int dims[4], void* stream);
int lqcd_unpack_clover_f64(double* dst_canonical, const double* src_native, const int dims[4], void* stream);
/* Packs ONE canonical null vector v_i[s][alpha][c] into slot i of the native array (so that a
 * 32-vector set never has to exist twice in HBM). */
int lqcd_pack_nullvec_f32(float* dst_native, const float* src_canonical_vi, int i, const int dims[4],
                          const int block[4], int nvec, void* stream);
int lqcd_pack_nullvec_f64(double* dst_native, const double* src_canonical_vi, int i, const int dims[4],
                          const int block[4], int nvec, void* stream);
int lqcd_unpack_nullvec_f32(float* dst_canonical_vi, const float* src_native, int i, const int dims[4],
                            const int block[4], int nvec, void* stream);
int lqcd_unpack_nullvec_f64(double* dst_canonical_vi, const double* src_native, int i, const int dims[4],
                            const int block[4], int nvec, void* stream);

/* ---- A1 / A2: fine Wilson-clover operator, Eq. 1, dagger Eq. 2 ---
 *   out(x) = in(x) + F(x) in(x)
 *            - kappa sum_mu [ (1 - g_mu) U_mu(x) beta+ in(x+mu) + (1 + g_mu) U_mu^dag(x-mu) beta- in(x-mu) ]
 * neighbours modulo dims (halo-free); beta+- = bc[mu] when the hop wraps around the lattice, else 1
 * (psi(x + L_mu mu) = bc[mu] psi(x); "periodic or anti-periodic").
 * out, in: native spinor; U: native gauge (18-real, or 12-real with LQCD_LINKS_12); clover: native
 * clover.  out must not alias in.  flags: LQCD_DAGGER, LQCD_LINKS_12. */
int lqcd_wilson_clover_mult_f32(float* out, const float* in, const float* U, const float* clover, float kappa,
                                const int dims[4], const int bc[4], unsigned flags, void* stream);
int lqcd_wilson_clover_mult_f64(double* out, const double* in, const double* U, const double* clover,
                                double kappa, const int dims[4], const int bc[4], unsigned flags, void* stream);

/* ---- F1: domain-decomposed operator D_SAP: "the Dirac matrix D_SAP [is defined] by turning off
 * the interaction across the domains" -- Eq. 1 with every hop whose two ends lie in different domains dropped.
 * domain[4] divides dims (the paper sets the SAP domain equal to the aggregation block); a direction spanned
 * by a single domain keeps all its hops, including the wrapping one with its boundary phase.
 * "Splitting the domains into even and odd groups, D_SAP^(e) and D_SAP^(o)": with LQCD_DOMAIN_EVEN (ODD) only
 * the sites of domains with (X_x+X_y+X_z+X_t) even (odd) are computed, out is set to ZERO on the others
 * (P_e D_SAP P_e).  Other flags and all argument rules as for lqcd_wilson_clover_mult. */
int lqcd_wilson_clover_dd_mult_f32(float* out, const float* in, const float* U, const float* clover, float kappa,
                                   const int dims[4], const int bc[4], const int domain[4], unsigned flags,
                                   void* stream);
int lqcd_wilson_clover_dd_mult_f64(double* out, const double* in, const double* U, const double* clover,
                                   double kappa, const int dims[4], const int bc[4], const int domain[4],
                                   unsigned flags, void* stream);

/* ---- A3: coarse operator, Eqs. 4, 7 ---------------------------------------
 *   out(X) = A[X][0] in(X) + sum_mu ( A[X][1+2mu] in(X+mu) + A[X][2+2mu] in(X-mu) ),
 * neighbours modulo cdims, always periodic (boundary phases live inside A).  LQCD_DAGGER applies
 * Gamma5c D_c Gamma5c, Gamma5c = diag(gamma5 sign of chi) (x) 1_nvec.  out must not alias in. */
int lqcd_coarse_mult_f32(float* out, const float* in, const float* A, const int cdims[4], int nvec,
                         unsigned flags, void* stream);
int lqcd_coarse_mult_f64(double* out, const double* in, const double* A, const int cdims[4], int nvec,
                         unsigned flags, void* stream);

/* A3 on HALF storage.  gamma5-hermiticity (Eq. 2) makes the blocks of Eq. 7
 * redundant:  A[X][2+2mu] = Gamma5c A[X-mu][1+2mu]^dag Gamma5c  for a Galerkin matrix, so the half layout
 * keeps A_0 and the four forward blocks only,
 *   Ah: complex[Vc][5][N][N],  Ah[X][0] = A[X][0],  Ah[X][1+mu] = A[X][1+2mu]
 * (lqcd_native_coarse_half_reals reals; lqcd_pack_coarse_half copies them out of the nine-block matrix, device to
 * device), and lqcd_coarse_mult_half applies
 *   out(X) = Ah[X][0] in(X) + sum_mu ( Ah[X][1+mu] in(X+mu) + Gamma5c Ah[X-mu][1+mu]^dag Gamma5c in(X-mu) ),
 * which IS lqcd_coarse_mult whenever A has the symmetry above (any Galerkin P^dag D P), at 5/9 of the matrix traffic:
 * every stored block is read once and serves both sites it couples.  ws_dev: caller-owned device scratch of
 * lqcd_coarse_half_workspace_bytes(cdims, nvec, sizeof(real)) bytes (four coarse vectors).  Two launches on `stream`,
 * fixed summation order (no atomics).  Flags, errors and aliasing rules as for lqcd_coarse_mult. */
size_t lqcd_native_coarse_half_reals(const int cdims[4], int nvec);
size_t lqcd_coarse_half_workspace_bytes(const int cdims[4], int nvec, int real_bytes);
int lqcd_pack_coarse_half_f32(float* Ah, const float* A, const int cdims[4], int nvec, void* stream);
int lqcd_pack_coarse_half_f64(double* Ah, const double* A, const int cdims[4], int nvec, void* stream);
int lqcd_coarse_mult_half_f32(float* out, const float* in, const float* Ah, const int cdims[4], int nvec,
                              unsigned flags, void* ws_dev, void* stream);
int lqcd_coarse_mult_half_f64(double* out, const double* in, const double* Ah, const int cdims[4], int nvec,
                              unsigned flags, void* ws_dev, void* stream);

/* lqcd_coarse_mult_half_f32 for callers that must not allocate device memory (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): the same two kernels, the same arithmetic and summation order --
 * the result is bit-identical with lqcd_coarse_mult_half_f32 -- but the four scratch vectors live in a file-scope
 * `static __device__` array inside the library instead of a caller-owned workspace.  The call itself calls no
 * cudaMalloc, cudaFree or any allocating routine; out, in and Ah are the caller's, as above.
 *   Limit: lqcd_coarse_half_workspace_bytes(cdims, nvec, 4) = Vc * 4 * 4 * nvec * 4 bytes must not exceed
 *     LQCD_NOALLOC_SCRATCH_BYTES (16 MiB: up to config 4's coarse lattice, 8^3 x 16 sites at nvec = 32, or 32 768
 *     sites at nvec = 8); a larger problem is refused with LQCD_EUNSUPPORTED and a message naming both sizes --
 *     nothing is launched.  Every GPU that loads the library holds these 16 MiB until the process exits.
 *   Sharing: every call on a device uses the SAME array.  Calls are safe back to back on one stream (stream order);
 *     two calls that can overlap on the GPU (different streams, or graphs replayed concurrently) RACE on it and give
 *     wrong results -- serialise them, or use the workspace form.  The array keeps the last call's contents; the
 *     kernels overwrite every element they later read, so nothing needs clearing between calls of any sizes.
 *   First call on a device: the array's device address is looked up once (cudaGetSymbolAddress, no allocation) and
 *     cached per device; make that first call outside a graph capture.  LQCD_ECUDA if the lookup fails.
 * Other errors, flags and aliasing rules as for lqcd_coarse_mult_half_f32. */
#define LQCD_NOALLOC_SCRATCH_BYTES (16u << 20)
int lqcd_coarse_mult_half_noalloc_f32(float* out, const float* in, const float* Ah, const int cdims[4], int nvec,
                                      unsigned flags, void* stream);

/* ---- A4: restriction, Eq. 5:  out_c[X][chi][i] = <v_i restricted to (X,chi) | in_f> -- */
int lqcd_restrict_f32(float* out_c, const float* in_f, const float* nullvecs, const int dims[4],
                      const int block[4], int nvec, void* stream);
int lqcd_restrict_f64(double* out_c, const double* in_f, const double* nullvecs, const int dims[4],
                      const int block[4], int nvec, void* stream);
/* Restriction of nrhs fine vectors at once (native spinors back to back -> coarse vectors back to back): the null
 * vectors, 97 % of a restriction's traffic, are streamed once per group of up to 9 vectors (as many slices of a 4^4
 * aggregate as fit in shared memory).  Used by the Galerkin assembly (the nine pieces of D of one column). */
int lqcd_restrict_mrhs_f32(float* out_c, const float* in_f, const float* nullvecs, const int dims[4],
                           const int block[4], int nvec, int nrhs, void* stream);
int lqcd_restrict_mrhs_f64(double* out_c, const double* in_f, const double* nullvecs, const int dims[4],
                           const int block[4], int nvec, int nrhs, void* stream);
/* ---- A5: prolongation, Eq. 6:  out_f(x,alpha,c) = sum_i v_i(x,alpha,c) in_c[X(x)][chi(alpha)][i];
 * overwrites out_f (no accumulate). */
int lqcd_prolong_f32(float* out_f, const float* in_c, const float* nullvecs, const int dims[4],
                     const int block[4], int nvec, void* stream);
int lqcd_prolong_f64(double* out_f, const double* in_c, const double* nullvecs, const int dims[4],
                     const int block[4], int nvec, void* stream);

/* Prolongation of nrhs coarse vectors at once (coarse vectors back to back -> native spinors back to back): the null
 * vectors are streamed once per group of up to 8 vectors. */
int lqcd_prolong_mrhs_f32(float* out_f, const float* in_c, const float* nullvecs, const int dims[4],
                          const int block[4], int nvec, int nrhs, void* stream);
int lqcd_prolong_mrhs_f64(double* out_f, const double* in_c, const double* nullvecs, const int dims[4],
                          const int block[4], int nvec, int nrhs, void* stream);

/* ---- F2: set-up of the operator fields on the device (not on the timed path) ------------------------------
 * Clover term from the links (formula: DESIGN.md reading Q1):
 *   F(x) = kappa csw sum_{mu<nu} sigma_{mu nu} (x) F_{mu nu}(x), sigma_{mu nu} = [g_mu, g_nu]/(2i),
 *   F_{mu nu} = (Q - Q^dag)/(8i), Q = the four plaquette leaves in the mu-nu plane (links periodic).
 * U: native 18-real gauge; clover: native clover (output). */
int lqcd_clover_from_links_f32(float* clover_native, const float* U_native18, float kappa, float csw,
                               const int dims[4], void* stream);
int lqcd_clover_from_links_f64(double* clover_native, const double* U_native18, double kappa, double csw,
                               const int dims[4], void* stream);

/* Block orthonormalisation of the null vectors, in place on the NATIVE null-vector array: within
 * every aggregate (X, chi) the nvec vectors are orthonormalised in index order (Gram-Schmidt, each vector projected
 * twice against its predecessors; the result is the unique Q of the QR factorisation with positive diagonal).
 * Requires |block| * 6 >= nvec.  Aggregate-local: any coarse extent >= 1.  A vector with nothing left after the
 * projections (zero or non-finite norm: e.g. a zero input vector) is written as ZERO, never Inf/NaN, and counted;
 * lqcd_orthonormalize_degenerate_count synchronises `stream`, returns the number of such (aggregate, vector) pairs of
 * the current device since the last query (0 = P has full rank everywhere) and resets it; < 0 on a CUDA error. */
int lqcd_orthonormalize_blocks_f32(float* nullvecs, const int dims[4], const int block[4], int nvec, void* stream);
int lqcd_orthonormalize_blocks_f64(double* nullvecs, const int dims[4], const int block[4], int nvec, void* stream);
long long lqcd_orthonormalize_degenerate_count(void* stream);
/* Galerkin coarse operator, Eq. 7: A[X][d][I][J] = <I| D_d |J> for the nine pieces of D (d = 0: the
 * site-diagonal term and the hops inside the aggregate; 1 + 2 mu / 2 + 2 mu: the forward / backward hops that leave
 * it), coarse-matrix layout as consumed by lqcd_coarse_mult.  U: native 18-real gauge; nullvecs: native, block-
 * orthonormal.  ws_dev: device scratch of lqcd_galerkin_workspace_bytes(dims, block, nvec, sizeof(real)) bytes.
 * Built column by column from the hot-path kernels: 2 nvec * 20 launches (one multi-vector restriction per column). */
size_t lqcd_galerkin_workspace_bytes(const int dims[4], const int block[4], int nvec, int real_bytes);
int lqcd_galerkin_coarse_f32(float* A, const float* U, const float* clover, const float* nullvecs, float kappa,
                             const int dims[4], const int bc[4], const int block[4], int nvec, void* ws_dev,
                             void* stream);
int lqcd_galerkin_coarse_f64(double* A, const double* U, const double* clover, const double* nullvecs, double kappa,
                             const int dims[4], const int bc[4], const int block[4], int nvec, void* ws_dev,
                             void* stream);

/* ---- F3: Richardson residual, blocked BLAS-1, inner-domain solver, SAP --------
 * Residual of one Richardson refinement "|x> + M_i(|b> - D|x>)" and of the SAP listing (PAPER.md:
 * 128-131) in one pass:  r = b - D x.  r must alias neither x nor b (b is read through the read-only data path;
 * LQCD_EINVAL otherwise).  flags: LQCD_LINKS_12 only. */
int lqcd_wilson_clover_residual_f32(float* r, const float* b, const float* x, const float* U, const float* clover,
                                    float kappa, const int dims[4], const int bc[4], unsigned flags, void* stream);
int lqcd_wilson_clover_residual_f64(double* r, const double* b, const double* x, const double* U,
                                    const double* clover, double kappa, const int dims[4], const int bc[4],
                                    unsigned flags, void* stream);

/* Blocked linear algebra ("a set of blocked version of linear algebraic functions such as dotc and axpy",
 * PAPER.md:155-157): the BLAS-1 operation restricted to each domain X (domain[4] divides dims; any number of
 * domains per direction, including 1), one number per domain, X in canonical coarse order.
 *   dotc:  out[X] = sum_{x in X} sum_{alpha,c} conj(a(x,alpha,c)) b(x,alpha,c)      out: Vc complex (re, im)
 *   caxpy: y(x) += coef[X(x)] a(x)                                                  coef: Vc complex
 * a, b, y: native spinors.  Fixed summation order (bit-reproducible). */
int lqcd_block_dotc_f32(float* out, const float* a, const float* b, const int dims[4], const int domain[4],
                        void* stream);
int lqcd_block_dotc_f64(double* out, const double* a, const double* b, const int dims[4], const int domain[4],
                        void* stream);
int lqcd_block_caxpy_f32(float* y, const float* coef, const float* a, const int dims[4], const int domain[4],
                         void* stream);
int lqcd_block_caxpy_f64(double* y, const double* coef, const double* a, const int dims[4], const int domain[4],
                         void* stream);

/* Inner-domain solver z = M_SAP^(g) r ~ (D_SAP^(g))^-1 r: "the MINRES algorithm with fixed number of iterations"
 * (PAPER.md:133).  D_SAP is not Hermitian, so this is the minimal-residual iteration of the SAP literature the paper
 * cites (reading Q17), run independently in every domain X of the selected group, from z = 0:
 *   rho = P_g r;  repeat niter times:  p = D_SAP^(g) rho;  alpha[X] = <p|rho>_X / <p|p>_X (0 if <p|p>_X = 0);
 *                                      z += alpha rho;  rho -= alpha p.
 * flags: LQCD_DOMAIN_EVEN / LQCD_DOMAIN_ODD select the group (neither: all domains); without LQCD_ACCUMULATE z is
 * overwritten (zero outside the group), with it z += M r on the group's sites and the others are left untouched.
 * U: native 18-real gauge.  z must not alias r.  When a domain's residual, links and clover term fit in the shared
 * memory of one SM (fp32: |domain| <= 256 sites, e.g. 4^4) all niter iterations run inside ONE kernel with the
 * operator read from HBM once; other sizes take a generic path that needs ws_dev, device scratch of
 * lqcd_mr_workspace_bytes(dims, domain, sizeof(real)) bytes (0 when the resident kernel applies; then ws_dev may be
 * NULL).  Both paths compute the same iteration; results agree to rounding. */
size_t lqcd_mr_workspace_bytes(const int dims[4], const int domain[4], int real_bytes);
int lqcd_mr_domain_solve_f32(float* z, const float* r, const float* U, const float* clover, float kappa,
                             const int dims[4], const int bc[4], const int domain[4], unsigned flags, int niter,
                             void* ws_dev, void* stream);
int lqcd_mr_domain_solve_f64(double* z, const double* r, const double* U, const double* clover, double kappa,
                             const int dims[4], const int bc[4], const int domain[4], unsigned flags, int niter,
                             void* ws_dev, void* stream);

/* Schwarz alternating procedure with fixed iterations, the listing of PAPER.md:127-131:
 *   |x> := 0, |r> := |b>;  for i = 1..n_sap:  |x> += M_SAP^(e)|r>;  |r> := |b> - D|x>;
 *                                             |x> += M_SAP^(o)|r>;  |r> := |b> - D|x>
 * with M_SAP^(e/o) = lqcd_mr_domain_solve with n_mr iterations (paper: n_sap = 4, n_mr = 6).
 * x: the result; r: caller-owned scratch spinor that receives the final residual b - D x; b: right-hand side; all
 * three distinct native spinors.  flags: LQCD_SAP_INITIAL_GUESS starts from the x passed in (|r> := |b> - D|x>
 * first): x0 + SAP(b - D x0), the Richardson refinement with M_2 = SAP in one call;
 * LQCD_SAP_NO_FINAL_RESIDUAL omits the last residual (saves one application of D when r is not needed; r then holds
 * no defined value).  The intermediate |r> := |b> - D|x> are evaluated only where the next half sweep reads them, on
 * the domains of its group (same arithmetic there; x and the final r do not depend on it).
 * ws_dev as for lqcd_mr_domain_solve.  2 n_sap solver launches + 2 n_sap residual launches on `stream`. */
int lqcd_sap_f32(float* x, float* r, const float* b, const float* U, const float* clover, float kappa,
                 const int dims[4], const int bc[4], const int domain[4], int n_sap, int n_mr, unsigned flags,
                 void* ws_dev, void* stream);
int lqcd_sap_f64(double* x, double* r, const double* b, const double* U, const double* clover, double kappa,
                 const int dims[4], const int bc[4], const int domain[4], int n_sap, int n_mr, unsigned flags,
                 void* ws_dev, void* stream);

/* SAP on nrhs right-hand sides at once (x, r, b: nrhs native spinors back to back each): the listing above for every
 * right-hand side; inside the shared-memory-resident inner-domain solver the right-hand sides are solved one after the
 * other on the resident links and clover term of the domain, which are read from HBM once per half sweep for all of
 * them.  Result k is bit-identical with lqcd_sap on (x_k, r_k, b_k). */
int lqcd_sap_mrhs_f32(float* x, float* r, const float* b, const float* U, const float* clover, float kappa,
                      const int dims[4], const int bc[4], const int domain[4], int nrhs, int n_sap, int n_mr,
                      unsigned flags, void* ws_dev, void* stream);
int lqcd_sap_mrhs_f64(double* x, double* r, const double* b, const double* U, const double* clover, double kappa,
                      const int dims[4], const int bc[4], const int domain[4], int nrhs, int n_sap, int n_mr,
                      unsigned flags, void* ws_dev, void* stream);

/* Coarse solver (1b) of PAPER.md:116 ("We employ the BiCGStab algorithm ... not necessarily performed with high
 * precision"): the BiCGStab recurrence of the listing PAPER.md:71 with M = 1 and x_0 = 0 for D_c x = b, with a FIXED
 * number of iterations instead of the listing's two "small enough" break points (reading Q18):
 *   r = rt = p = b;  repeat niter times:  v = D_c p;  alpha = <rt|r>/<rt|v>;  s = r - alpha v;  t = D_c s;
 *     omega = <t|s>/<t|t>;  x += alpha p + omega s;  r' = s - omega t;  beta = (alpha/omega) <rt|r'>/<rt|r>;
 *     p = r' + beta (p - omega v);  r = r'.        (a vanishing denominator sets its quotient to 0)
 * x, b: coarse vectors; r_out (may be NULL): receives the recurrence residual; A as for lqcd_coarse_mult.  All scalars
 * stay on the device (no host synchronisation); dot products have a fixed summation order.  ws_dev: device scratch of
 * lqcd_coarse_bicgstab_workspace_bytes(cdims, nvec, sizeof(real)) bytes.  7 launches per iteration. */
size_t lqcd_coarse_bicgstab_workspace_bytes(const int cdims[4], int nvec, int real_bytes);
int lqcd_coarse_bicgstab_f32(float* x, float* r_out, const float* b, const float* A, const int cdims[4], int nvec,
                             int niter, void* ws_dev, void* stream);
int lqcd_coarse_bicgstab_f64(double* x, double* r_out, const double* b, const double* A, const int cdims[4], int nvec,
                             int niter, void* ws_dev, void* stream);
/* The same solver on the HALF storage of the coarse matrix (Ah as for lqcd_coarse_mult_half): every application of D_c
 * moves 5/9 of the matrix bytes.  Same workspace size; same recurrences, so the result differs from the nine-block
 * solve only by the rounding of the operator applications. */
int lqcd_coarse_bicgstab_half_f32(float* x, float* r_out, const float* b, const float* Ah, const int cdims[4], int nvec,
                                  int niter, void* ws_dev, void* stream);
int lqcd_coarse_bicgstab_half_f64(double* x, double* r_out, const double* b, const double* Ah, const int cdims[4],
                                  int nvec, int niter, void* ws_dev, void* stream);

/* The same for nrhs right-hand sides at once (x, r_out, b: nrhs coarse vectors back to back): nrhs independent
 * recurrences -- every right-hand side has its own alpha, omega, beta -- that share the applications of D_c through
 * lqcd_coarse_mult_mrhs, i.e. ONE pass over A per application for up to 16 right-hand sides (tensor cores, fp32,
 * N = 64).  Result k is what lqcd_coarse_bicgstab gives for b_k, up to rounding. */
size_t lqcd_coarse_bicgstab_mrhs_workspace_bytes(const int cdims[4], int nvec, int nrhs, int real_bytes);
int lqcd_coarse_bicgstab_mrhs_f32(float* x, float* r_out, const float* b, const float* A, const int cdims[4], int nvec,
                                  int nrhs, int niter, void* ws_dev, void* stream);
int lqcd_coarse_bicgstab_mrhs_f64(double* x, double* r_out, const double* b, const double* A, const int cdims[4],
                                  int nvec, int nrhs, int niter, void* ws_dev, void* stream);

/* One V-cycle x = M b of the multigrid preconditioner, two Richardson refinements
 * "|x> + M_i(|b> - D|x>) -> |x>" from |x> = 0:
 *   (1) M_1 = prolong o BiCGStab(D_c, n_coarse iterations) o restrict     steps (1a)-(1c)
 *   (2) M_2 = SAP(n_sap, n_mr) with the aggregation block as SAP domain   ("We set the SAP domain to be the same as
 *                                                                          the domain of coarsening")
 * x, b: native spinors, distinct; U: native 18-real gauge; nullvecs: native, block-orthonormal; A: coarse matrix.
 * Everything is enqueued on `stream`, device-resident, no host synchronisation or copy.  ws_dev: device scratch of
 * lqcd_mg_workspace_bytes(dims, block, nvec, sizeof(real)) bytes. */
size_t lqcd_mg_workspace_bytes(const int dims[4], const int block[4], int nvec, int real_bytes);
int lqcd_mg_vcycle_f32(float* x, const float* b, const float* U, const float* clover, float kappa, const int dims[4],
                       const int bc[4], const int block[4], int nvec, const float* nullvecs, const float* A,
                       int n_coarse, int n_sap, int n_mr, void* ws_dev, void* stream);
int lqcd_mg_vcycle_f64(double* x, const double* b, const double* U, const double* clover, double kappa,
                       const int dims[4], const int bc[4], const int block[4], int nvec, const double* nullvecs,
                       const double* A, int n_coarse, int n_sap, int n_mr, void* ws_dev, void* stream);
/* The same V-cycle with the coarse matrix in half storage (its coarse solve is lqcd_coarse_bicgstab_half). */
int lqcd_mg_vcycle_half_f32(float* x, const float* b, const float* U, const float* clover, float kappa,
                            const int dims[4], const int bc[4], const int block[4], int nvec, const float* nullvecs,
                            const float* Ah, int n_coarse, int n_sap, int n_mr, void* ws_dev, void* stream);
int lqcd_mg_vcycle_half_f64(double* x, const double* b, const double* U, const double* clover, double kappa,
                            const int dims[4], const int bc[4], const int block[4], int nvec, const double* nullvecs,
                            const double* Ah, int n_coarse, int n_sap, int n_mr, void* ws_dev, void* stream);

/* The V-cycle on nrhs right-hand sides at once (x, b: nrhs native spinors back to back): the restrictions, the coarse
 * solves (lqcd_coarse_bicgstab_mrhs, i.e. D_c on the tensor cores) and the prolongations are shared by all right-hand
 * sides -- one pass over the null vectors / over A per group --, the smoother is lqcd_sap_mrhs.
 * Result k is what lqcd_mg_vcycle gives for b_k, up to rounding.  ws_dev: lqcd_mg_mrhs_workspace_bytes(...) bytes. */
size_t lqcd_mg_mrhs_workspace_bytes(const int dims[4], const int block[4], int nvec, int nrhs, int real_bytes);
int lqcd_mg_vcycle_mrhs_f32(float* x, const float* b, const float* U, const float* clover, float kappa,
                            const int dims[4], const int bc[4], const int block[4], int nvec, const float* nullvecs,
                            const float* A, int nrhs, int n_coarse, int n_sap, int n_mr, void* ws_dev, void* stream);
int lqcd_mg_vcycle_mrhs_f64(double* x, const double* b, const double* U, const double* clover, double kappa,
                            const int dims[4], const int bc[4], const int block[4], int nvec, const double* nullvecs,
                            const double* A, int nrhs, int n_coarse, int n_sap, int n_mr, void* ws_dev, void* stream);

/* ---- F4: the coarse operator on K right-hand sides at once (many right-hand sides are "a typical
 * situation") ----------------------------------------------------------------------------------------------------
 *   out_k = D_c in_k,  k = 0 .. nrhs-1     (Eqs. 4, 7; the definition of lqcd_coarse_mult, K times)
 * in, out: nrhs coarse vectors back to back, [k][X][chi][i]; A as for lqcd_coarse_mult; out must not alias in.
 * fp32 with nvec = 32 (N = 64) and flags = 0 runs on the tensor cores (tcgen05, 3xTF32 split of both operands with
 * fp32 accumulation in short TMEM chains added in registers: fp32 accuracy; A is read from HBM ONCE per launch of up
 * to 16 right-hand sides);
 * every other case (other nvec, LQCD_DAGGER, fp64) applies lqcd_coarse_mult once per right-hand side. */
int lqcd_coarse_mult_mrhs_f32(float* out, const float* in, const float* A, const int cdims[4], int nvec, int nrhs,
                              unsigned flags, void* stream);
int lqcd_coarse_mult_mrhs_f64(double* out, const double* in, const double* A, const int cdims[4], int nvec, int nrhs,
                              unsigned flags, void* stream);

/* The fine operator on nrhs right-hand sides at once: out_k = D in_k (or D^dag in_k), k = 0 .. nrhs-1 (Eq. 1, nrhs
 * times).  in, out: nrhs native spinors back to back (stride lqcd_native_spinor_reals(dims)); out must not alias in.
 * Right-hand sides are taken two at a time by a kernel that loads every link and clover block once for both
 * (576 + 2 x 192 instead of 2 x 768 compulsory bytes per site); an odd one out takes the single-right-hand-side
 * kernel.  flags: LQCD_DAGGER, LQCD_LINKS_12. */
int lqcd_wilson_clover_mult_mrhs_f32(float* out, const float* in, const float* U, const float* clover, float kappa,
                                     const int dims[4], const int bc[4], int nrhs, unsigned flags, void* stream);
int lqcd_wilson_clover_mult_mrhs_f64(double* out, const double* in, const double* U, const double* clover,
                                     double kappa, const int dims[4], const int bc[4], int nrhs, unsigned flags,
                                     void* stream);

/* ---- Sharded fine operator: the halo-exchange step (the paper partitions the lattice over
 * the nodes in 4-D and exchanges the boundary once per application of D) --------------
 * A rank owns the local lattice dims[4] (all fields in the native layouts of that local lattice).  Bit mu of
 * part_mask says that direction mu is partitioned: hops that leave the local lattice there are served by the
 * neighbouring rank (which may be the rank itself).  One application of D (Eq. 1) or D^dag (Eq. 2) is
 *   lqcd_wilson_clover_halo_pack      in  -> send[8]       (independent of the next line: they overlap on two streams)
 *   lqcd_wilson_clover_mult_interior  in  -> out           D with the leaving hops switched off
 *   -- exchange: recv[2 mu + 0] := send[2 mu + 1] of the -mu neighbour, recv[2 mu + 1] := send[2 mu + 0] of the +mu one
 *   lqcd_wilson_clover_halo_add       out -= kappa * (the hops served by recv[8])
 * Face 2 mu + dir holds the sites with x_mu = 0 (dir 0) or x_mu = dims[mu] - 1 (dir 1); face site f is the
 * lexicographic index of the other three coordinates (x fastest); each face site carries the spin-projected half
 * spinor of its hop, 12 reals (not 24), stored as rows of 16 bytes: buf[(j * Fv + f) * NV + q], Fv = V / dims[mu],
 * NV = 4 (fp32) / 2 (fp64), real 2 (3 sp + c) + reim = j NV + q.  The dir-1 face is already multiplied by
 * U_mu^dag(x) (the link of a backward hop lives on the sender); the receiver multiplies the other by its own U_mu(x).
 * send / recv: HOST arrays of 8 DEVICE pointers, each of lqcd_halo_face_reals(dims, mu) reals, 16-byte aligned,
 * caller-owned; entries of unpartitioned directions are ignored (may be NULL).  face_phase[2 mu + dir]: +1, or
 * bc[mu] when that hop wraps the GLOBAL lattice (the rank sits on its edge); bc[] of mult_interior is used in the
 * unpartitioned directions only.  flags: LQCD_DAGGER, LQCD_LINKS_12 (the same on all three calls).  The sum differs
 * from lqcd_wilson_clover_mult on the global lattice by rounding order only.  part_mask = 0: pack and add are no-ops
 * and mult_interior is lqcd_wilson_clover_mult. */
size_t lqcd_halo_face_reals(const int dims[4], int mu);
int lqcd_wilson_clover_halo_pack_f32(float* const send[8], const float* in, const float* U, const int dims[4],
                                     unsigned part_mask, unsigned flags, void* stream);
int lqcd_wilson_clover_halo_pack_f64(double* const send[8], const double* in, const double* U, const int dims[4],
                                     unsigned part_mask, unsigned flags, void* stream);
int lqcd_wilson_clover_mult_interior_f32(float* out, const float* in, const float* U, const float* clover, float kappa,
                                         const int dims[4], const int bc[4], unsigned part_mask, unsigned flags,
                                         void* stream);
int lqcd_wilson_clover_mult_interior_f64(double* out, const double* in, const double* U, const double* clover,
                                         double kappa, const int dims[4], const int bc[4], unsigned part_mask,
                                         unsigned flags, void* stream);
/* The residual r = b - D x of the sharded operator: the interior pass in residual form,
 * r = b - (D with the leaving hops off) x, then lqcd_wilson_clover_halo_add(r, recv, U, -kappa, ...) on faces packed
 * from x (the sign of kappa turns "out -= kappa hops" into "+=").  r must not alias b or x; flags: LQCD_LINKS_12,
 * and, with domain[4] != NULL, LQCD_DOMAIN_EVEN or LQCD_DOMAIN_ODD: only the sites of that group of domains (local
 * colouring) are computed, the others are left as they are -- what SAP needs between two half sweeps (the halo add
 * then also touches face sites of the other group, whose values are not read).  domain may be NULL without them. */
int lqcd_wilson_clover_residual_interior_f32(float* r, const float* b, const float* x, const float* U,
                                             const float* clover, float kappa, const int dims[4], const int bc[4],
                                             const int* domain, unsigned part_mask, unsigned flags, void* stream);
int lqcd_wilson_clover_residual_interior_f64(double* r, const double* b, const double* x, const double* U,
                                             const double* clover, double kappa, const int dims[4], const int bc[4],
                                             const int* domain, unsigned part_mask, unsigned flags, void* stream);
int lqcd_wilson_clover_halo_add_f32(float* out, const float* const recv[8], const float* U, float kappa,
                                    const int dims[4], const int face_phase[8], unsigned part_mask, unsigned flags,
                                    void* stream);
int lqcd_wilson_clover_halo_add_f64(double* out, const double* const recv[8], const double* U, double kappa,
                                    const int dims[4], const int face_phase[8], unsigned part_mask, unsigned flags,
                                    void* stream);

/* The same for the coarse operator ("same pattern on the coarse lattice, N complex per face site").
 * cdims[4]: the LOCAL coarse lattice; A: its blocks (a block of a leaving hop lives on the site it acts on, so no
 * block is ever exchanged and no boundary phase appears: bc is inside A).  Face 2 mu + dir: the coarse vectors of the
 * sites with X_mu = 0 (dir 0) / cdims[mu] - 1 (dir 1), [face site][chi][i] complex, face site = lexicographic index of
 * the other three coordinates; lqcd_coarse_halo_face_reals(cdims, nvec, mu) reals each.  Exchange as above
 * (recv[2 mu] := send[2 mu + 1] of the -mu neighbour, recv[2 mu + 1] := send[2 mu] of the +mu neighbour).
 *   lqcd_coarse_halo_pack      in -> send[8]
 *   lqcd_coarse_mult_interior  out = D_c in without the blocks of leaving hops (their sources are not read)
 *   lqcd_coarse_halo_add       out += those blocks applied to recv[8]            (one launch per face, over its sites only)
 * flags: LQCD_DAGGER on mult_interior and halo_add alike.  A partitioned direction may have local extent 1. */
size_t lqcd_coarse_halo_face_reals(const int cdims[4], int nvec, int mu);
int lqcd_coarse_halo_pack_f32(float* const send[8], const float* in, const int cdims[4], int nvec, unsigned part_mask,
                              void* stream);
int lqcd_coarse_halo_pack_f64(double* const send[8], const double* in, const int cdims[4], int nvec,
                              unsigned part_mask, void* stream);
int lqcd_coarse_mult_interior_f32(float* out, const float* in, const float* A, const int cdims[4], int nvec,
                                  unsigned part_mask, unsigned flags, void* stream);
int lqcd_coarse_mult_interior_f64(double* out, const double* in, const double* A, const int cdims[4], int nvec,
                                  unsigned part_mask, unsigned flags, void* stream);
int lqcd_coarse_halo_add_f32(float* out, const float* const recv[8], const float* A, const int cdims[4], int nvec,
                             unsigned part_mask, unsigned flags, void* stream);
int lqcd_coarse_halo_add_f64(double* out, const double* const recv[8], const double* A, const int cdims[4], int nvec,
                             unsigned part_mask, unsigned flags, void* stream);

/* The coarse solver (1b) on a sharded coarse lattice: the same BiCGStab recurrences (same kernels, scalars resident
 * on the device) with the two things that cross ranks supplied by the caller as plain C callbacks:
 *   apply (out, in, stream, user): out = D_c in on this rank's part (pack -> interior -> add above); device pointers
 *          to vectors of the local coarse lattice cdims[4]; must enqueue on `stream` (or order itself after it);
 *   reduce(reals, count, real_bytes, stream, user): sum the device array reals[count] element by element over all
 *          ranks, in place, ordered on `stream` (an NCCL all-reduce); NULL = single rank.  The array holds the
 *          per-CTA partial sums of one dot product; every rank then adds them in the same fixed order, so all ranks
 *          hold bit-identical scalars.
 * Both return 0 on success.  ws_dev: lqcd_coarse_bicgstab_workspace_bytes(cdims, nvec, real_bytes).  x, b, r_out as
 * for lqcd_coarse_bicgstab; a local extent of 1 is allowed. */
typedef int (*lqcd_apply_fn)(void* out_dev, const void* in_dev, void* stream, void* user);
typedef int (*lqcd_reduce_fn)(void* reals_dev, size_t count, int real_bytes, void* stream, void* user);
int lqcd_coarse_bicgstab_hooks_f32(float* x, float* r_out, const float* b, const int cdims[4], int nvec, int niter,
                                   lqcd_apply_fn apply, lqcd_reduce_fn reduce, void* user, void* ws_dev, void* stream);
int lqcd_coarse_bicgstab_hooks_f64(double* x, double* r_out, const double* b, const int cdims[4], int nvec, int niter,
                                   lqcd_apply_fn apply, lqcd_reduce_fn reduce, void* user, void* ws_dev, void* stream);

/* ---- end-to-end entry points on HOST vectors (fp32 and fp64) ---------------------------------
 * The operator fields (U, clover, A, nullvecs) stay resident on the device in native layout; the
 * right-hand side comes from and the result goes back to HOST memory in CANONICAL layout (pinned
 * memory recommended).  Each call: cudaMemcpyAsync H2D -> pack -> the mult kernel -> unpack ->
 * cudaMemcpyAsync D2H -> cudaStreamSynchronize.  A fine vector of at least three slabs of ~16 MB
 * (knob "host_slab_mb": smallest slab in MB, -1 = never) travels in SLABS of time slices: the upload
 * of slab k+1 runs under pack / kernel / unpack of slab k (on `stream`) and under the download of
 * slab k-1, on two copy streams and a set of events that the library creates ONCE per calling host
 * thread and device and keeps (the only state of these calls; nothing is allocated per call).  The
 * kernels are the same ones on a range of tiles / aggregates: results are bit-identical with the
 * one-shot path.  The call returns after everything it enqueued has completed, as before.
 * ws_dev is caller-owned device scratch of at least
 * lqcd_host_workspace_bytes(...) bytes (the _f32 calls) or lqcd_host_workspace_bytes_f64(...) bytes
 * (the _f64 calls; host and device data are then all double).  Same errors as the device calls. */
size_t lqcd_host_workspace_bytes(const int dims[4], const int block[4], int nvec);
size_t lqcd_host_workspace_bytes_f64(const int dims[4], const int block[4], int nvec);
int lqcd_wilson_clover_mult_host_f32(float* out_host, const float* in_host, const float* U, const float* clover,
                                     float kappa, const int dims[4], const int bc[4], unsigned flags,
                                     void* ws_dev, void* stream);
int lqcd_coarse_mult_host_f32(float* out_host, const float* in_host, const float* A, const int cdims[4],
                              int nvec, unsigned flags, void* ws_dev, void* stream);
int lqcd_restrict_host_f32(float* out_c_host, const float* in_f_host, const float* nullvecs, const int dims[4],
                           const int block[4], int nvec, void* ws_dev, void* stream);
int lqcd_prolong_host_f32(float* out_f_host, const float* in_c_host, const float* nullvecs, const int dims[4],
                          const int block[4], int nvec, void* ws_dev, void* stream);
int lqcd_wilson_clover_mult_host_f64(double* out_host, const double* in_host, const double* U, const double* clover,
                                     double kappa, const int dims[4], const int bc[4], unsigned flags,
                                     void* ws_dev, void* stream);
int lqcd_coarse_mult_host_f64(double* out_host, const double* in_host, const double* A, const int cdims[4],
                              int nvec, unsigned flags, void* ws_dev, void* stream);
int lqcd_restrict_host_f64(double* out_c_host, const double* in_f_host, const double* nullvecs, const int dims[4],
                           const int block[4], int nvec, void* ws_dev, void* stream);
int lqcd_prolong_host_f64(double* out_f_host, const double* in_c_host, const double* nullvecs, const int dims[4],
                          const int block[4], int nvec, void* ws_dev, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* LQCD_B200_H */

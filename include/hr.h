/*
 * hr.h -- C ABI of the B200-native Wilson-Dirac hopping term for higher-representation SU(N) fermions.
 *
 * What the library computes (BASELINE.json:north_star; workload: section 3.1 "Wilson-Dirac
 * operator in single and double precision for general higher representations of SU(N_c)", even-odd;
 * the represented link is a d_R x d_R matrix acting on the colour index of the spinor):
 *
 *   Dphi psi (x) = -1/2 sum_{mu=0..3} [ (1 - gamma_mu) s+_mu(x) U^R_mu(x)            psi(x + mu)
 *                                     + (1 + gamma_mu) s-_mu(x) U^R_mu(x - mu)^dagger psi(x - mu) ]
 *   D psi (x)    = (4 + m0) psi(x) + Dphi psi (x)
 *
 * on a periodic T x X x Y x Z lattice, s+-_mu(x) = bc[mu] on the hop that crosses the seam between
 * x_mu = L_mu-1 and 0, else 1 (antiperiodic fermions: bc = -1), and the link map U -> U^R
 * (fundamental, adjoint [real], two-index symmetric / antisymmetric).  Everything the paper is silent
 * on (gamma basis, site order, parity, generator and tensor bases) is fixed in DESIGN.md "Readings"
 * (C1..C19); the ones a caller needs are restated below.
 *
 * CANONICAL (interchange) LAYOUT, used only by the import/export calls (reading C4):
 *   dims = {T, X, Y, Z}, mu = 0,1,2,3 = t,x,y,z.  Full-lattice site index i = ((t*X + x)*Y + y)*Z + z.
 *   parity(i) = (t+x+y+z) & 1.  A parity-p half field lists the parity-p sites by increasing i, so its
 *   half index is i >> 1 (every extent is even).
 *   spinor site  = [spin alpha = 0..3][colour a = 0..d_R-1] complex (re, im)
 *   gauge field  = [site i][mu][row][col] complex (re, im), row-major; a REPRESENTED ADJOINT field is
 *                  real: [site i][mu][row][col] real.
 * INTERNAL device layout (private): per parity, per 16-byte vector
 * plane, contiguous in the half index.  Spinor buffers passed to hr_dphi_eo / hr_dirac are in the
 * internal layout: fill them with hr_spinor_import, read them with hr_spinor_export.  Their size is
 * hr_spinor_bytes() per parity (the same number of bytes as the canonical half field).
 *
 * Pointers: every `void *` spinor/gauge buffer handed to a compute call is DEVICE memory owned by the
 * caller (e.g. a torch tensor's data_ptr()), 16-byte aligned.  `canon` pointers of import/export may
 * be HOST or DEVICE memory (detected).  `stream` is a cudaStream_t passed as void* (NULL = default
 * stream).  All device work is enqueued on that stream; the compute calls never synchronise and never
 * allocate.  No call throws or exits: each returns an hr_status, and hr_last_error() gives the text.
 * There is NO CPU fallback: without a usable CUDA device every compute call returns HR_ECUDA.
 */
#ifndef HR_H
#define HR_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { HR_OK = 0, HR_EINVAL = -1, HR_EUNSUPPORTED = -2, HR_ECUDA = -3, HR_ENOMEM = -4 } hr_status;
typedef enum { HR_F64 = 0, HR_F32 = 1 } hr_prec;
typedef enum { HR_REP_FUND = 0, HR_REP_ADJ = 1, HR_REP_SYM = 2, HR_REP_ASYM = 3 } hr_rep;

typedef struct hr_ctx hr_ctx;     /* immutable problem description: dims, bc, N, rep, device            */
typedef struct hr_gauge hr_gauge; /* one link field: fundamental (N x N) or represented (d_R x d_R), one precision */

/* Library version string, e.g. "hr-dphi 0.1 (sm_100a)". */
const char *hr_version(void);
/* Text of the last error raised on the calling thread ("" if none); valid until the next call. */
const char *hr_last_error(void);

/*
 * Describe the problem.  dims[mu] even and >= 2 (reading C11: odd extents break the even/odd
 * bipartition), bc[mu] in {+1,-1}, N in {2,3,4}.  Supported (N, rep): N=2: FUND, ADJ, SYM;
 * N=3: FUND, ADJ, SYM, ASYM; N=4: FUND, ASYM, SYM (d_R = 10), ADJ (d_R = 15; these two run on the colour-parallel
 * kernel of PAPER.md:92-96 and have no clover / on-the-fly-link kernels).  Anything else (e.g. ASYM for N=2, d_R = 1)
 * -> HR_EUNSUPPORTED.  Does not touch the GPU; `device` is the CUDA ordinal later calls run on.
 */
hr_status hr_ctx_create(hr_ctx **ctx, const int dims[4], const int bc[4], int N, hr_rep rep, int device);
void hr_ctx_destroy(hr_ctx *ctx); /* also frees the host-path workspace, if one was created */

int hr_rep_dim(const hr_ctx *ctx);          /* d_R */
int hr_links_are_real(const hr_ctx *ctx);   /* 1 for the adjoint (reading C7), else 0 */
size_t hr_half_volume(const hr_ctx *ctx);   /* V/2 = output sites of one hr_dphi_eo */
size_t hr_gauge_bytes(const hr_ctx *ctx, int represented, hr_prec prec); /* whole field, both parities, INTERNAL layout:
                                             * represented real links of an odd d_R > 8 (SU(4) adjoint) are held with rows
                                             * of d_R + 1 reals (the last one zero); the canonical record that
                                             * hr_gauge_import / hr_gauge_export exchange stays d_R x d_R */
size_t hr_spinor_bytes(const hr_ctx *ctx, hr_prec prec);                 /* ONE parity: V/2 sites      */

/*
 * hr_gauge_alloc -- make a link-field handle (BASELINE.json:north_star "hr_gauge_alloc").
 * represented = 0: fundamental N x N complex links; 1: represented d_R x d_R links (real for ADJ);
 * 2: fundamental links stored as their first N-1 rows (hr_gauge_compress below; SU(2), SU(3) only).
 * dev_mem == NULL: the library allocates hr_gauge_bytes() of device memory and owns it;
 * else it borrows caller memory (>= hr_gauge_bytes(), 16-byte aligned), which must outlive the handle.
 * Contents are undefined until hr_gauge_import / hr_represent_links writes them.
 */
hr_status hr_gauge_alloc(const hr_ctx *ctx, int represented, hr_prec prec, void *dev_mem, hr_gauge **out);
void hr_gauge_free(hr_gauge *g);
void *hr_gauge_data(const hr_gauge *g);  /* device pointer of the internal-layout storage */

/* canonical <-> internal.  canon_prec is the precision of the canonical array; conversion (one
 * rounding) happens in the pack kernel.  For host `canon` the copy is staged through device memory
 * the call allocates and frees (set-up path, not a hot call); the call returns after the data has
 * left / reached `canon` (it synchronises the stream when `canon` is host memory). */
hr_status hr_gauge_import(hr_gauge *dst, const void *canon, hr_prec canon_prec, void *stream);
hr_status hr_gauge_export(const hr_gauge *src, void *canon, hr_prec canon_prec, void *stream);
hr_status hr_spinor_import(const hr_ctx *ctx, void *dst_dev, hr_prec prec, const void *canon,
                           hr_prec canon_prec, int parity, void *stream);
hr_status hr_spinor_export(const hr_ctx *ctx, const void *src_dev, hr_prec prec, void *canon,
                           hr_prec canon_prec, int parity, void *stream);

/*
 * hr_gauge_compress -- row-compressed fundamental links (reading C30 of DESIGN.md; SU(2) and SU(3)).
 * hr_gauge_alloc(ctx, 2, prec, ...) makes a field that keeps only the first N-1 rows of every fundamental link
 * (SU(3): 12 of 18 reals, SU(2): 4 of 8); hr_gauge_compress fills it from a fundamental field of the same precision.
 * Every compute call that takes `links` accepts it for the FUNDAMENTAL representation (the last row is rebuilt in
 * registers: conj(row0 x row1), resp. (-conj u01, conj u00)), for the SU(2) ADJOINT (the real 3x3 link is built from
 * the four reals of the first row: 32 instead of 72 bytes per link in fp64) and for the SU(3) ADJOINT (applied on the
 * fly, 96 instead of 512 bytes).  Only for links that ARE special unitary:
 * the result equals that of the full links up to their unitarity violation.  Such a field cannot be imported/exported.
 */
hr_status hr_gauge_compress(hr_gauge *rows_out, const hr_gauge *fund_in, void *stream);

/*
 * hr_represent_links -- the link map U -> U^R, one kernel launch over the 4V links
 * (BASELINE.json:north_star "fundamental-to-representation link map"; configs[2]:
 * U^adj_ab = 2 tr(T_a U T_b U^dagger), T_a = lambda_a/2 in the nested Gell-Mann order, reading C6;
 * configs[3]: two-index symmetric basis e^(ij), pairs lexicographic i<=j, reading C8:
 * R_(ij),(kl) = n_ij n_kl (U_ik U_jl +- U_il U_jk), n = 1/sqrt2 on diagonal pairs; FUND = copy).
 * fund_in: fundamental field, repr_out: represented field of the same ctx; precisions may differ
 * (arithmetic in fund_in's precision, one rounding on store).
 */
hr_status hr_represent_links(hr_gauge *repr_out, const hr_gauge *fund_in, void *stream);

/*
 * hr_dphi_eo -- the even-odd hopping term, ONE kernel launch over the V/2 output sites
 * (BASELINE.json:north_star "hr_dphi_eo(out, in, links, parity, stream)").
 * parity = parity of the OUTPUT sites (reading C5).  out: parity-`parity` half field, in:
 * parity-(1-parity) half field, both internal layout, precision = precision of `links`.
 * out must not alias in.
 * `links` is a represented field, OR ("on-the-fly representation") the
 * FUNDAMENTAL field when the representation is two-index symmetric / antisymmetric (or fundamental):
 * the kernel then reads the N x N link (e.g. 144 instead of 576 bytes for the SU(3) sextet in fp64) and
 * applies R(U) psi as U Psi U^T, R(U)^dagger psi as U^dagger Psi U^*, Psi = sum_a psi_a e_a in the basis
 * of reading C8 -- the same operator, never forming R(U).  The SU(3) adjoint likewise accepts the
 * fundamental field ((R psi)_a = 2 tr(T_a U Psi U^dagger), Psi = sum_a psi_a T_a: 144 instead of 512 bytes
 * per link in fp64); the SU(2) adjoint accepts the row-compressed field of hr_gauge_compress (32 instead of
 * 72 bytes) but not the full fundamental one (-> HR_EINVAL).  The same holds for every call below that
 * takes `links`.
 */
hr_status hr_dphi_eo(void *out, const void *in, const hr_gauge *links, int parity, void *stream);

/*
 * hr_dirac -- D = (4+m0) + Dphi on full fields (BASELINE.json:north_star "hr_dirac(m0)").
 * Full field = [even half | odd half], each half in the internal layout (2 * hr_spinor_bytes()).
 * Two launches (one per output parity) with the (4+m0) psi(x) term fused.  out_full != in_full.
 */
hr_status hr_dirac(double m0, void *out_full, const void *in_full, const hr_gauge *links, void *stream);

/*
 * hr_dphi_eo_host -- the same operation end to end from HOST memory: copies the canonical parity-
 * (1-parity) half spinor `in_canon` (host, ideally pinned) to the device, packs it, runs hr_dphi_eo,
 * unpacks and copies the canonical result into `out_canon` (host).  `links` stays resident on the
 * device (a gauge field changes once per molecular-dynamics step, a spinor every call).  The
 * workspace (two internal half spinors + two 256 MiB staging buffers, two copy streams) is created on
 * first use and cached in the ctx.  With host arrays and at least 8 time slices the call is a pipeline
 * over chunks of time slices: upload of chunk k+1 || pack, Dphi_eo on the output slices of chunk k-1,
 * unpack || download of chunk k-2 (the same result as the single launch up to the kernel variant's
 * rounding).  Device pointers are accepted too (no staging).  Synchronises `stream` before returning:
 * the host arrays are valid / reusable then.
 */
hr_status hr_dphi_eo_host(hr_ctx *ctx, void *out_canon, const void *in_canon, hr_prec canon_prec,
                          const hr_gauge *links, int parity, void *stream);

/* =====================================================================================================
 * Second part -- SURVEY.md section 8(f) NEXT-1: what the hopping term is FOR ("We are
 * supporting even-odd preconditioning"; section 3.2 "Linear Algebra"
 * section 3.3 "Conjugate Gradient").  The paper prints no formula for any of these; the definitions are
 * readings C20-C24 of DESIGN.md, restated at each call.  All spinor buffers are ONE-parity half fields in
 * the internal layout (hr_spinor_bytes()), device memory owned by the caller, 16-byte aligned.
 * Calls that reduce (dot, norm2, the CG) use a scratch area the ctx creates on first use (3 MiB, freed by
 * hr_ctx_destroy): issue them on ONE stream at a time per ctx.
 * ===================================================================================================== */

/*
 * Spinor linear algebra (Fig. 7: "Copy spinor field", "g5 application", "g5 mulc add
 * assign").  One streaming kernel each, no synchronisation, no allocation.
 *   hr_spinor_lincomb:            out = ca * G(x) + cb * y,  G = gamma5 if g5 != 0 else 1; ca, cb complex
 *                                 (re, im); y (and cb) may be NULL; out may alias x and/or y.
 *   hr_spinor_copy:               out = in
 *   hr_spinor_g5:                 out = gamma5 in            (gamma5 = diag(1,1,-1,-1) on spin, reading C1)
 *   hr_spinor_mulc_add_assign:    out += c in                (reading C23)
 *   hr_spinor_g5_mulc_add_assign: out += c gamma5 in         (reading C23)
 */
hr_status hr_spinor_lincomb(const hr_ctx *ctx, hr_prec prec, void *out, const double ca[2], int g5, const void *x,
                            const double cb[2], const void *y, void *stream);
hr_status hr_spinor_copy(const hr_ctx *ctx, hr_prec prec, void *out, const void *in, void *stream);
hr_status hr_spinor_g5(const hr_ctx *ctx, hr_prec prec, void *out, const void *in, void *stream);
hr_status hr_spinor_mulc_add_assign(const hr_ctx *ctx, hr_prec prec, void *out, double c_re, double c_im,
                                    const void *in, void *stream);
hr_status hr_spinor_g5_mulc_add_assign(const hr_ctx *ctx, hr_prec prec, void *out, double c_re, double c_im,
                                       const void *in, void *stream);

/*
 * Reductions ("inner products and norms"; the paper runs a site-wise kernel and then
 * cub -- two passes over global memory; here ONE kernel reads the field(s) once).  Reading C22:
 *   hr_spinor_dot:   result[0] + i result[1] = <x, y> = sum conj(x) y     (2 doubles)
 *   hr_spinor_norm2: result[0] = <x, x>                                   (1 double)
 * Sums are accumulated in fp64 for both precisions, in an order fixed by the launch geometry (bitwise
 * reproducible).  `result` may be DEVICE memory (no synchronisation) or HOST memory (the call
 * synchronises the stream before returning).
 */
hr_status hr_spinor_dot(hr_ctx *ctx, hr_prec prec, const void *x, const void *y, double *result, void *stream);
hr_status hr_spinor_norm2(hr_ctx *ctx, hr_prec prec, const void *x, double *result, void *stream);
/*
 * hr_spinor_dot_noalloc -- hr_spinor_dot for callers that may not allocate (CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc): same one-pass reduction, same result (result_dev[0] + i result_dev[1] = <x, y>; x == y gives the
 * norm with result_dev[1] = 0), but the per-CTA partial sums live in a 33 KB file-scope device array of libhr.so instead
 * of the context's cudaMalloc'ed scratch.  The call makes no cudaMalloc / cudaFree and no synchronisation.
 *   x, y        DEVICE half fields, internal layout, 16-byte aligned, hr_spinor_bytes(ctx, prec) each; not modified
 *   result_dev  DEVICE memory, 2 doubles, written by the kernel on `stream` (host pointers are rejected: HR_EINVAL)
 * Limits: half fields of at most hr_spinor_dot_noalloc_max_bytes() = 4 GiB; beyond that HR_EUNSUPPORTED, nothing launched.
 * The array is shared by every call on a device: calls that can overlap on the GPU (different streams without an ordering
 * between them, concurrent host threads) race on it -- order them on one stream or with events.
 */
size_t hr_spinor_dot_noalloc_max_bytes(void);
hr_status hr_spinor_dot_noalloc(hr_ctx *ctx, hr_prec prec, const void *x, const void *y, double *result_dev, void *stream);

/*
 * hr_dhat -- the even-odd preconditioned operator on EVEN sites (reading C20):
 *     out_e = Dhat in_e = (4+m0)^2 in_e - Dphi_eo Dphi_oe in_e          (g5 == 0)
 *     out_e = gamma5 Dhat in_e                                          (g5 != 0; Hermitian, reading C21)
 * Two Dphi launches; the diagonal term, the sign and gamma5 are fused into the second one's epilogue.
 * tmp_o: caller-owned odd-parity half field (overwritten).  out_e, in_e, tmp_o distinct.
 */
hr_status hr_dhat(double m0, int g5, void *out_e, const void *in_e, void *tmp_o, const hr_gauge *links, void *stream);

/*
 * Conjugate gradient (reading C21).  hr_cg_dhat solves Dhat x_e = b_e on the even sites by
 * the textbook CG on the normal equations Dhat^dagger Dhat x = Dhat^dagger b (Dhat^dagger = gamma5 Dhat
 * gamma5), x0 = 0, recursive residual, stopping at the first k with |r_k|^2 <= tol^2 |Dhat^dagger b|^2 or
 * k = maxiter.  alpha, beta, the iteration counter and the stop flag live on the device: iterations are
 * enqueued in batches and the host synchronises `stream` once per batch (and before returning).
 *   workspace: hr_cg_workspace_bytes(ctx, prec of links, maxiter) bytes of device memory, 256-byte aligned.
 *   iters (may be NULL): iterations done.  rel_res2 (may be NULL): |r_k|^2 / |rhs|^2 at exit.
 *   hist (may be NULL): HOST array of maxiter+1 doubles, receives |r_k|^2 / |rhs|^2 for k = 0..iters.
 * hr_dirac_solve solves the FULL system D x = b, D = (4+m0) + Dphi, fields [even half | odd half], through
 * the preconditioned one (reading C24):  Dhat x_e = (4+m0) b_e - Dphi_eo b_o ;  x_o = (b_o - Dphi_oe x_e)/(4+m0).
 * x must not alias b.  Not converged within maxiter is not an error: check iters / rel_res2.
 * WHICH residual: rel_res2 of hr_dirac_solve is that of the system the iteration runs on -- the normal equations of the
 * preconditioned system, |Dhat^dag (rhs_e - Dhat x_e)|^2 / |Dhat^dag rhs_e|^2 --, of hr_dirac_solve_bicgstab and
 * hr_dirac_clover_solve that of the preconditioned system, |rhs_e - Dhat x_e|^2 / |rhs_e|^2; neither is |b - D x|^2 / |b|^2
 * of the full system (the odd half is solved exactly given x_e, so the full residual lives on the even sites and equals
 * |rhs_e - Dhat x_e| / (4+m0) there).  A caller who needs the full-system number applies hr_dirac to x once.
 */
size_t hr_cg_workspace_bytes(const hr_ctx *ctx, hr_prec prec, int maxiter);
/*
 * hr_bicgstab_dhat -- the stabilised bi-conjugate gradient ("stabilized Bi-Conjugate Gradient"; reading
 * C29: textbook BiCGstab applied to Dhat ITSELF, no normal equations, x0 = 0, shadow residual = b, stopping at the
 * first k with |r_k|^2 <= tol^2 |b|^2 or k = maxiter).  rho, alpha, omega live on the device like the CG's scalars.
 * Arguments as hr_cg_dhat; workspace of hr_bicgstab_workspace_bytes().  rel_res2 / hist are relative to |b|^2.
 */
size_t hr_bicgstab_workspace_bytes(const hr_ctx *ctx, hr_prec prec, int maxiter);
hr_status hr_bicgstab_dhat(hr_ctx *ctx, double m0, void *x_e, const void *b_e, const hr_gauge *links, double tol,
                           int maxiter, void *workspace, int *iters, double *rel_res2, double *hist, void *stream);
hr_status hr_cg_dhat(hr_ctx *ctx, double m0, void *x_e, const void *b_e, const hr_gauge *links, double tol, int maxiter,
                     void *workspace, int *iters, double *rel_res2, double *hist, void *stream);
/*
 * hr_cg_dhat_dist -- the CG of hr_cg_dhat (reading C21: textbook CG on Dhat^dagger Dhat x = Dhat^dagger b, x0 = 0, stop at
 * the first k with |r_k|^2 <= tol^2 |rhs|^2 or k = maxiter) on a lattice that is DISTRIBUTED over several ranks
 * (DESIGN.md section 13).  The library owns every step of the algorithm -- the vector updates are its
 * kernels on the local half fields, the scalar recurrences (alpha = rr / <p, A p>, beta = rr' / rr, the stopping test)
 * run here -- and calls back for the two things only the caller can do:
 *   dphi(user, out, in, parity):   the distributed Dphi_eo on the caller's decomposition (pack / exchange / interior /
 *                                  apply, e.g. halo.py), enqueued on `stream`; out: parity-`parity` local half field.
 *                                  Returns 0 on success.
 *   allsum(user, vals, n):         sum of n host doubles over all ranks, in place (an all-reduce); returns 0 on success.
 *                                  May be NULL on a single rank.
 * x_e, b_e: local even half fields, precision `prec`.  workspace: hr_cg_dist_workspace_bytes(ctx, prec) bytes of device
 * memory, 256-byte aligned.  iters / hist as hr_cg_dhat (hist: HOST array of maxiter+1 doubles or NULL).  Host-driven: two
 * synchronisations of `stream` and two all-reduces per iteration (the sums must cross the ranks anyway).
 * Errors: HR_EINVAL (NULL / misaligned / aliased arguments), HR_ECUDA (a callback failed or a CUDA call did).
 */
typedef int (*hr_dphi_fn)(void *user, void *out, const void *in, int parity);
typedef int (*hr_allsum_fn)(void *user, double *vals, int n);
size_t hr_cg_dist_workspace_bytes(const hr_ctx *ctx, hr_prec prec);
hr_status hr_cg_dhat_dist(hr_ctx *ctx, hr_prec prec, double m0, void *x_e, const void *b_e, double tol, int maxiter,
                          void *workspace, hr_dphi_fn dphi, hr_allsum_fn allsum, void *user, int *iters, double *hist,
                          void *stream);
/*
 * hr_qmr_dhat -- the gamma5-QMR ("QMR gamma_5 inverters"; reading C33): quasi-minimal residual method without
 * look-ahead on Dhat ITSELF, built on the Lanczos process in the indefinite inner product (x, y)_J = <x, gamma5 y>, in which
 * Dhat is self-adjoint (reading C21) -- ONE operator application per iteration, no Dhat^dagger.  x0 = 0.  After step k,
 * |eta_k| is the norm of the quasi-residual (|b - Dhat x_k| <= sqrt(k+1) |eta_k|); when |eta_k| <= tol |b| the TRUE
 * residual is computed (one more operator application) and the iteration ends if |b - Dhat x_k| <= tol |b|; it also ends at
 * k = maxiter, when the Krylov space is exhausted and at a Lanczos breakdown ((v_k, v_k)_J = 0).  The Lanczos scalars and the
 * Givens rotations live on the DEVICE (a small state owned by the context), like the CG's: the host enqueues batches of 4, 8,
 * ... 32 iterations -- per iteration two Dphi launches, two fused vector kernels and two one-thread kernels -- and reads the
 * state once per batch; once a stop flag is set the rest of a batch returns at once.  Arguments as hr_cg_dhat; workspace of
 * hr_qmr_workspace_bytes(), 256-byte aligned.
 *   rel_res2: TRUE |b - Dhat x|^2 / |b|^2 at exit.  hist (HOST, maxiter+1 doubles): |eta_k| / |b| for k = 0..iters.
 */
size_t hr_qmr_workspace_bytes(const hr_ctx *ctx, hr_prec prec);
hr_status hr_qmr_dhat(hr_ctx *ctx, double m0, void *x_e, const void *b_e, const hr_gauge *links, double tol, int maxiter,
                      void *workspace, int *iters, double *rel_res2, double *hist, void *stream);
hr_status hr_dirac_solve(hr_ctx *ctx, double m0, void *x_full, const void *b_full, const hr_gauge *links, double tol,
                         int maxiter, void *workspace, int *iters, double *rel_res2, void *stream);
/*
 * hr_bicgstab_dhat_mixed -- mixed precision (the operator exists "in single and double precision"): defect
 * correction x += e, Dhat e = r, with the defect equation solved by hr_bicgstab_dhat in fp32 (links32, to inner_tol on
 * the normalised residual) and the TRUE residual r = b - Dhat x recomputed in fp64 (links64) after every inner solve; stops
 * when |r|^2 <= tol^2 |b|^2 (fp64, true residual) or after maxiter inner iterations in total.  x_e, b_e: fp64 half
 * fields; workspace of hr_mixed_workspace_bytes(ctx, maxiter), 256-byte aligned.  iters: inner iterations in total,
 * outer_steps: number of defect corrections, rel_res2: true |r|^2 / |b|^2 of the x that is returned.  Synchronises once per
 * outer step.  Also ends after 100 outer steps or when an inner solve makes no iteration; NOT converged is not an error:
 * the caller compares rel_res2 with tol^2 (as for hr_cg_dhat: check iters / rel_res2).
 */
size_t hr_mixed_workspace_bytes(const hr_ctx *ctx, int maxiter);
hr_status hr_bicgstab_dhat_mixed(hr_ctx *ctx, double m0, void *x_e, const void *b_e, const hr_gauge *links64,
                                 const hr_gauge *links32, double tol, double inner_tol, int maxiter, void *workspace,
                                 int *iters, int *outer_steps, double *rel_res2, void *stream);

/* The same full solve with hr_bicgstab_dhat as the inner solver (workspace of hr_bicgstab_workspace_bytes();
 * tol and rel_res2 refer to the preconditioned system Dhat x_e = (4+m0) b_e - Dphi_eo b_o). */
hr_status hr_dirac_solve_bicgstab(hr_ctx *ctx, double m0, void *x_full, const void *b_full, const hr_gauge *links,
                                  double tol, int maxiter, void *workspace, int *iters, double *rel_res2, void *stream);

/* =====================================================================================================
 * Third part -- SURVEY.md section 8(e)/(f) NEXT-2: the lattice split into slabs along t, one slab per GPU,
 * with the paper's half-spinor exchange (send buffers, "it is only necessary to send a
 * half-spinor"; interior sites are computed while the messages travel).
 * The ctx of a rank describes its LOCAL slab: dims[0] = T_local (even), bc[0] = the sign of the GLOBAL
 * time seam (applied only by the first / last rank).  Rank r owns global t in [r T_local, (r+1) T_local).
 * One distributed Dphi_eo(parity p) is, on every rank:
 *   1. hr_dphi_eo_halo_pack   -> send_up  (for the NEXT rank):     chi = U_0(y)^dagger P+ psi(y), y in my last slice
 *                                send_dn  (for the PREVIOUS rank): h   = P- psi(y),               y in my first slice
 *   2. the exchange: my send_up becomes the next rank's recv_prev, my send_dn the previous rank's recv_next
 *      (NCCL send/recv via torch.distributed -- paper_2405_19294_b200.halo.exchange -- or no copy at all: the
 *      send pointers may be PEER memory (the neighbour's receive buffers mapped over NVLink), in which case
 *      the pack kernel's stores ARE the transfer; ordering is then the caller's: an event or barrier
 *      between pack and apply);
 *   3. hr_dphi_eo_interior    -> out = Dphi_eo restricted to hops inside the slab (overlaps with 2);
 *   4. hr_dphi_eo_halo_apply  -> out += the two face contributions, with bc[0] on the global seam.
 * With one rank (first_rank = last_rank = 1, recv_prev = own send_up, recv_next = own send_dn) steps 1-4
 * reproduce hr_dphi_eo exactly.  A message holds 2 d_R complex per face site, hr_halo_bytes() in all, in
 * the plane layout over the X*Y*Z/2 face sites.  `links` as for hr_dphi_eo (represented, or fundamental
 * for the two-index representations); all buffers device memory, 16-byte aligned; no synchronisation.
 * ===================================================================================================== */
size_t hr_halo_bytes(const hr_ctx *ctx, hr_prec prec);
/*
 * Peer memory for the messages (the fused projection + transfer of step 2): hr_halo_buffers_alloc makes ONE cudaMalloc
 * allocation of 6 hr_halo_bytes(): [send_up | send_dn | recv_prev[0] | recv_next[0] | recv_prev[1] | recv_next[1]]
 * (receive buffers double-buffered by call parity); hr_ipc_export / hr_ipc_open / hr_ipc_close wrap
 * cudaIpcGetMemHandle / OpenMemHandle / CloseMemHandle (64-byte handle) so that a neighbouring PROCESS -- on another
 * GPU over NVLink, or on the same GPU -- maps the allocation and passes  peer_base + offset  as the send pointers of
 * hr_dphi_eo_halo_pack.  Ordering between the neighbour's pack and the own apply is the caller's (halo.py:
 * PeerSlabDphi uses one barrier per call).
 */
/*
 * 4-D block decomposition ("4-D block partition, split t first, then z, y, x"): the same three steps
 * for any direction mu in {0: t, 1: x, 2: y, 3: z}.  hr_face_bytes(ctx, prec, mu) = bytes of one message of that direction
 * (V_local/2 / L_mu face sites x 2 d_R complex); hr_dphi_eo_face_pack / _face_apply are hr_dphi_eo_halo_pack / _halo_apply
 * for direction mu (the seam sign is bc[mu]); hr_dphi_eo_interior_mask drops the hops across the boundaries of every
 * direction whose bit is set in split_mask (bit mu).  A rank packs every split direction from the SAME input field, runs
 * the interior launch, and applies the directions one after the other on the same stream (edge and corner sites receive
 * a term from each).  Local extents stay even (site parity is global); a split in z needs an even local Y.
 */
size_t hr_face_bytes(const hr_ctx *ctx, hr_prec prec, int mu);
hr_status hr_dphi_eo_face_pack(int mu, void *send_up, void *send_dn, const void *in, const hr_gauge *links, int parity,
                               void *stream);
/* hr_dphi_eo_faces_pack -- hr_dphi_eo_face_pack for ALL split directions (bit mu of split_mask) in ONE launch: the faces of a
 * 4-D block decomposition are packed from the same input field, and four launches of 7-40 us were
 * launch-bound.  send_up[mu] / send_dn[mu]: the two messages of direction mu (device or peer memory, hr_face_bytes each);
 * entries of unsplit directions are ignored.  Results are bitwise those of the per-direction calls. */
hr_status hr_dphi_eo_faces_pack(int split_mask, void *const send_up[4], void *const send_dn[4], const void *in, const hr_gauge *links,
                                int parity, void *stream);
hr_status hr_dphi_eo_interior_mask(void *out, const void *in, const hr_gauge *links, int parity, int split_mask, void *stream);
hr_status hr_dphi_eo_face_apply(int mu, void *out, const void *recv_prev, const void *recv_next, const hr_gauge *links,
                                int parity, int first_rank, int last_rank, void *stream);
/* hr_dphi_eo_faces_apply -- hr_dphi_eo_face_apply for ALL split directions (bit mu of split_mask) in ONE launch.  An edge or
 * corner site of the block receives a term from each of its faces; every boundary site is updated by exactly one thread, which
 * adds the terms of its faces in ascending mu, so the result is bitwise that of the per-direction calls made in ascending mu.
 * recv_prev[mu] / recv_next[mu]: the messages received from the previous / next rank in mu (hr_face_bytes each; entries of
 * unsplit directions are ignored); bit mu of first_mask / last_mask: this rank is the first / last along mu (its outer face
 * carries the seam sign bc[mu]).  `out` already holds hr_dphi_eo_interior_mask's result; no synchronisation. */
hr_status hr_dphi_eo_faces_apply(int split_mask, void *out, const void *const recv_prev[4], const void *const recv_next[4],
                                 const hr_gauge *links, int parity, int first_mask, int last_mask, void *stream);
hr_status hr_halo_buffers_alloc(const hr_ctx *ctx, hr_prec prec, void **base);             /* direction t */
hr_status hr_face_buffers_alloc(const hr_ctx *ctx, hr_prec prec, int mu, void **base);     /* 6 hr_face_bytes(mu) */
void hr_halo_buffers_free(const hr_ctx *ctx, void *base);
hr_status hr_ipc_export(const hr_ctx *ctx, const void *base, unsigned char handle[64]);
hr_status hr_ipc_open(const hr_ctx *ctx, const unsigned char handle[64], void **peer_base);
hr_status hr_ipc_close(const hr_ctx *ctx, void *peer_base);
hr_status hr_dphi_eo_halo_pack(void *send_up, void *send_dn, const void *in, const hr_gauge *links, int parity,
                               void *stream);
hr_status hr_dphi_eo_interior(void *out, const void *in, const hr_gauge *links, int parity, void *stream);
hr_status hr_dphi_eo_halo_apply(void *out, const void *recv_prev, const void *recv_next, const hr_gauge *links,
                                int parity, int first_rank, int last_rank, void *stream);

/* =====================================================================================================
 * Fourth part -- SURVEY.md section 8(f) NEXT-4: the clover term ("clover [17]").  The paper prints
 * no formula; reading C28 of DESIGN.md:
 *     D_sw = D + T,   T(x) = -(c_sw/2) sum_{mu<nu} sigma_{mu nu} (x) F_{mu nu}(x),  sigma = (i/2)[gamma_mu, gamma_nu],
 *     F_{mu nu} = (Q_{mu nu} - Q_{mu nu}^dagger)/(8 i),  Q = the four counter-clockwise plaquettes ("leaves") of the
 *     mu-nu plane that start and end at x, built from the REPRESENTED links (U = exp(iA) gives F = dA).
 * hr_clover_build: one launch over all V sites; `clover` is caller-owned device memory of hr_clover_bytes(),
 *     precision of `links` (a represented field); T is stored as two packed Hermitian 2 d_R x 2 d_R blocks per site
 *     (the chiral basis makes sigma block diagonal), [even sites | odd sites].
 * hr_dirac_clover: out = (4+m0) in + Dphi in + T in on full fields [even half | odd half]; the two hr_dirac launches
 *     followed by one site-local launch per parity.  out != in.
 * hr_clover_exp: the exponentiated clover term ("exponentiated clover improvement [8]"; reading C31: the
 *     site-diagonal part (4+m0) + T of D_sw becomes (4+m0) exp(T/(4+m0)), positive definite on every gauge field).
 *     Replaces, IN PLACE, the T written by hr_clover_build by E = (4+m0)[exp(T/(4+m0)) - 1]; hr_dirac_clover with the
 *     same m0 then applies D_exp = Dphi + (4+m0) exp(T/(4+m0)).  One launch over the 2V blocks; 4 + m0 > 0.
 * Even-odd preconditioning WITH the clover term ("even-odd preconditioning, clover"; reading C32): with
 * A(x) = (4+m0) + T(x)  [or (4+m0) exp(T/(4+m0)) after hr_clover_exp]  and  D_sw = [[A_ee, Dphi_eo], [Dphi_oe, A_oo]],
 *     Dhat_sw = A_ee - Dphi_eo A_oo^{-1} Dphi_oe                                  (Schur complement on the even sites).
 * hr_clover_finalize: IN PLACE site_term (T or E, as written by hr_clover_build / hr_clover_exp) -> A = (4+m0) + it, and
 *     A^{-1} (every 2 d_R x 2 d_R block inverted in fp64: Cholesky where it is positive definite -- any physical mass --, else
 *     Gauss-Jordan elimination with partial pivoting) into site_inverse, a second buffer
 *     of hr_clover_bytes().  After this call the buffers serve hr_dhat_clover / hr_dirac_clover_solve (NOT
 *     hr_dirac_clover, which expects T and adds 4+m0 itself).
 * hr_dhat_clover: out_e = Dhat_sw in_e; two Dphi launches and two site-local launches; tmp_o, tmp2_o: odd-parity half
 *     fields owned by the caller; the four spinor buffers distinct.
 * hr_dirac_clover_solve: x = D_sw^{-1} b on full fields [even half | odd half] through
 *     Dhat_sw x_e = b_e - Dphi_eo A_oo^{-1} b_o,  x_o = A_oo^{-1} (b_o - Dphi_oe x_e),  the preconditioned system solved
 *     by BiCGstab (reading C29; tol, iters and rel_res2 refer to it); workspace of hr_clover_solve_workspace_bytes().
 */
size_t hr_clover_bytes(const hr_ctx *ctx, hr_prec prec);
hr_status hr_clover_finalize(const hr_ctx *ctx, hr_prec prec, void *site_term, void *site_inverse, double m0, void *stream);
hr_status hr_dhat_clover(void *out_e, const void *in_e, void *tmp_o, void *tmp2_o, const hr_gauge *links,
                         const void *site_term, const void *site_inverse, void *stream);
size_t hr_clover_solve_workspace_bytes(const hr_ctx *ctx, hr_prec prec, int maxiter);
hr_status hr_dirac_clover_solve(hr_ctx *ctx, void *x_full, const void *b_full, const hr_gauge *links, const void *site_term,
                                const void *site_inverse, double tol, int maxiter, void *workspace, int *iters,
                                double *rel_res2, void *stream);
hr_status hr_clover_exp(const hr_ctx *ctx, hr_prec prec, void *clover, double m0, void *stream);
hr_status hr_clover_build(void *clover, const hr_gauge *links, double csw, void *stream);
hr_status hr_dirac_clover(double m0, void *out_full, const void *in_full, const hr_gauge *links, const void *clover,
                          void *stream);

/*
 * Kernel tuning (experiments and ncu evidence; defaults are chosen per (d_R, precision) from
 * measurements).  key: "variant" (kernel variant id, -1 = default table; 0 site, 1 site_ef,
 * 2 pair, 3 pair_ef, 4 site_l1, 5 site_pf, 6 colour = one thread per (site, colour row)),
 * "block" (threads per CTA, 0 = default), "xblock" (x-extent of the thread order's blocks, a divisor
 * of X; 0 = default from the L2 working-set rule), "cg_graph" (the CG replays one captured iteration as a
 * CUDA graph: 1 = default, on lattices below 2^19 sites per parity, where launch overhead shows; 2 = always;
 * 0 = plain kernel launches).  Unknown key or value -> HR_EINVAL.
 */
hr_status hr_ctx_set_tuning(hr_ctx *ctx, const char *key, int value);
/* Name of the Dphi kernel variant a call with this precision would launch (for logs/bench). */
const char *hr_dphi_variant_name(const hr_ctx *ctx, hr_prec prec);
/* Number of kernel launches this library has enqueued since load (all threads). */
unsigned long long hr_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* HR_H */

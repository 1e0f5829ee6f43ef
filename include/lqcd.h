/*
 * lqcd.h -- C ABI of the B200-native staggered Dslash / CG / multi-shift CG library
 *           (liblqcd_b200.so, built from paper_1701_00426_b200/csrc/ for sm_100a).
 *
 * The calls follow the paper's statement of the problem (arxiv/paper_1701_00426, cited as
 * PAPER.md:LINE):
 *   - lqcd_dslash          : D_eo / D_oe of Eq. 7; the paper's
 *                            acc_Deo(u, out, in, backfield) of Listing 2
 *   - lqcd_mdagm           : m^2 - D_eo D_oe of Eq. 8
 *   - lqcd_cg              : "the conjugate gradient" on Eq. 8
 *   - lqcd_cg_multishift   : the "multishift inverter routine" for Eq. 6
 *
 *   - lqcd_rational_apply  : c0 b + sum_i c_i (A + sigma_i)^-1 b, the rational function whose
 *                            poles are the shifts of Eq. 6, fused into the
 *                            multi-shift solve
 *   - lqcd_pack_* / unpack : canonical <-> native SoA, parity-split fields (PAPER.md:245-272,
 *                            Figs 1-2, Eq. 9) with optional 2-row ("12-real") links whose third
 *                            row is rebuilt in registers as r2 = (r0 ^ r1)^*
 * What the paper leaves unstated (stencil, phases, boundary conditions, CG recurrences) is
 * fixed by the readings R1..R19 of DESIGN.md.
 *
 * General conventions
 *   - Plain C; no torch / C++ types.  Every function returns an int status (LQCD_OK = 0) unless
 *     stated otherwise.  No exceptions, no abort(), nothing written to stdout/stderr.
 *   - "dev" pointers are CUDA device pointers on the context's device, >= 16-byte aligned,
 *     owned by the caller (e.g. torch.empty(...).data_ptr()).  The library never allocates or
 *     frees field memory; it owns only the context (host struct, < 64 KiB of device scalars,
 *     one pinned flag word), the staging buffers of the *_host* calls and, in slab mode over the
 *     peer transport, the rank's communication block (flags, slots, four face-sized landing buffers).  "host" pointers are ordinary host memory (pinned or not).
 *   - All device work is enqueued on the CUDA stream given to lqcd_create.  Functions marked
 *     "async" return after enqueueing; functions marked "blocking" synchronise that stream.
 *   - out/in buffers of one call must not alias unless stated.
 *   - A context is not thread-safe: one context per host thread (several contexts may share a
 *     device and a stream).
 *   - Errors: bad arguments are detected before any launch (LQCD_ERR_ARG / _WORKSPACE);
 *     CUDA failures give LQCD_ERR_CUDA; lqcd_last_error() returns a message.
 *
 * Canonical layout (interchange format; identical to lqcd_inputs/fields.py and the oracle):
 *   lex   = x0 + N0*(x1 + N1*(x2 + N2*x3))                       (numerator of Eq. 9)
 *   links : complex128 U[lex][mu][row][col], mu = 0..3, row-major 3x3 (rows = r0,r1,r2)
 *   half spinor of parity p = (x0+x1+x2+x3)%2 : complex128 phi[idxh][c], idxh = lex/2  (Eq. 9)
 * Canonical arrays are ALWAYS complex128, also for an LQCD_F32 context (packing rounds to
 * nearest; unpacking widens exactly).
 *
 * Native layout: private to the library; sizes from
 * lqcd_spinor_bytes / lqcd_links_bytes.
 */
#ifndef LQCD_H
#define LQCD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lqcd_ctx lqcd_ctx; /* opaque, library-owned */

enum { LQCD_OK = 0, LQCD_ERR_ARG = 1, LQCD_ERR_UNSUPPORTED = 2, LQCD_ERR_CUDA = 3,
       LQCD_ERR_NOT_CONVERGED = 4, LQCD_ERR_WORKSPACE = 5 };
enum { LQCD_F64 = 0, LQCD_F32 = 1 };          /* arithmetic and storage type of native fields */
enum { LQCD_RECON_18 = 0, LQCD_RECON_12 = 1 };/* links stored as 3 rows / 2 rows */
enum { LQCD_EVEN = 0, LQCD_ODD = 1 };         /* parity of the OUTPUT sites (reading R5)        */
#define LQCD_MAX_SHIFTS 32

/* Library version string (static storage). */
const char *lqcd_version(void);

/*
 * Create a context.
 *   dims            N0..N3 (x0 fastest), each even and >= 2 (PAPER.md:249 and footnote d);
 *                   N0*N1*N2*N3 < 2^31
 *   prec            LQCD_F64 | LQCD_F32   (single-precision variants)
 *   recon           LQCD_RECON_18 | LQCD_RECON_12
 *   antiperiodic_t  1: fermion field antiperiodic across the x3 boundary (reading R4), 0: periodic
 *   device          CUDA device ordinal
 *   cuda_stream     a cudaStream_t (as void*), or NULL for the legacy default stream
 * Errors: LQCD_ERR_ARG (null ctx, bad dims/enums), LQCD_ERR_CUDA (no device / allocation).
 */
int lqcd_create(lqcd_ctx **ctx, const int dims[4], int prec, int recon, int antiperiodic_t,
                int device, void *cuda_stream);
int lqcd_destroy(lqcd_ctx *ctx); /* blocking; frees only library-owned memory */

/* Message for the last non-OK status returned with this context ("" if none).
 * With ctx == NULL: message of the last failed lqcd_create on this thread. */
const char *lqcd_last_error(const lqcd_ctx *ctx);

/*
 * Private tuning knobs (block sizes, layout variant, cache policy); see DESIGN.md "Tuning".
 * Unknown names -> LQCD_ERR_ARG.  "layout" may only be changed before any field is packed.
 * Side effect of "l2_persist" > 0: the device-wide persisting-L2 limit is raised and an access-policy window
 * is set on the context's stream; both are restored to the values found when the option is cleared, the
 * workspace changes or the context is destroyed.
 */
int lqcd_set_option(lqcd_ctx *ctx, const char *name, long value);
long lqcd_get_option(const lqcd_ctx *ctx, const char *name); /* -1 if unknown */

/* Sizes in bytes of native buffers the caller must allocate (0 if ctx is NULL). */
size_t lqcd_spinor_bytes(const lqcd_ctx *ctx); /* one half-lattice colour vector              */
size_t lqcd_links_bytes(const lqcd_ctx *ctx);  /* whole link field, both parities, 4 directions */
size_t lqcd_workspace_bytes(const lqcd_ctx *ctx, int nshift); /* solver workspace, nshift>=1   */

/* Hand the solvers (and lqcd_mdagm) a caller-owned device workspace of >= lqcd_workspace_bytes
 * bytes for the largest nshift that will be used.  Errors: LQCD_ERR_ARG, LQCD_ERR_WORKSPACE. */
int lqcd_set_workspace(lqcd_ctx *ctx, void *dev_ptr, size_t bytes);

/* Canonical <-> native, on the device.  async. */
int lqcd_pack_links(lqcd_ctx *ctx, void *native_dev, const void *canonical_dev /* c128 [V][4][3][3] */);
int lqcd_pack_spinor(lqcd_ctx *ctx, int parity, void *native_dev, const void *canonical_dev /* c128 [V/2][3] */);
int lqcd_unpack_spinor(lqcd_ctx *ctx, int parity, void *canonical_dev, const void *native_dev);

/*
 * out = D in on the sites of `parity` (Eq. 7; readings R1-R5):
 *   (D psi)(x) = 1/2 sum_mu eta_mu(x) [ s+ U_mu(x) psi(x+mu) - s- U_mu(x-mu)^dagger psi(x-mu) ]
 * parity = LQCD_EVEN: out_e = D_eo in_o;  parity = LQCD_ODD: out_o = D_oe in_e.
 * out, in: native half spinors (device); links: native link field (device).  async.
 * Errors: LQCD_ERR_ARG (null pointer, parity not 0/1, out == in), LQCD_ERR_CUDA.
 */
int lqcd_dslash(lqcd_ctx *ctx, int parity, void *out, const void *in, const void *links);

/*
 * Block Dslash: outs[r] = D ins[r] on the sites of `parity` for r = 0..n-1 (Eq. 7, same operator as
 * lqcd_dslash).  Every thread loads each of its 8 links once per block of right-hand sides (option "force_block": 8,
 * the default, or 4 per launch; a remainder runs in blocks of 4, 2 and 1) instead of once per vector: 1152 + 96 k bytes per
 * site and block of k vectors in fp64 with 18-real links, against 1248 k.  Per vector the arithmetic and its order are
 * those of lqcd_dslash: the results are bit-identical.  lqcd_fermion_force computes its y_i = D_oe x_i this way
 * (PAPER.md:315).
 *   outs, ins   host arrays of n device pointers (native half vectors); no output may alias any input
 *   1 <= n <= LQCD_MAX_SHIFTS
 * async.  Errors: LQCD_ERR_ARG; LQCD_ERR_UNSUPPORTED with a backfield attached or on a slab context (use lqcd_dslash).
 */
int lqcd_dslash_multi(lqcd_ctx *ctx, int parity, int n, void *const *outs, const void *const *ins,
                      const void *links);

/*
 * The `backfield` argument of the paper's acc_Deo(u, out, in, backfield) (Listing 2): one
 * real per link (the paper's double_soa), never explained in the text.  Reading R6 of DESIGN.md: an external
 * U(1) phase theta_mu(x); every link enters D as e^{i theta_mu(x)} U_mu(x), i.e. the forward hop out of x is
 * multiplied by e^{+i theta_mu(x)} and the backward hop by e^{-i theta_mu(x-mu)}.  The SU(3) link itself is
 * untouched, so 2-row storage still works: the third row is rebuilt first, the phase is applied after
 * (PAPER.md:272); eta and the boundary sign stay computed in-kernel.
 *   canonical: float64 theta[lex][mu] (radians, any range);  native: one real of the context's precision per
 *   link, layout private, lqcd_backfield_bytes bytes.
 * lqcd_dslash_backfield is lqcd_dslash with the phases of that one call (the paper's four-argument form).
 * lqcd_set_backfield attaches a native phase field to the context (NULL detaches): every later lqcd_dslash,
 * lqcd_dslash_slices, lqcd_mdagm, lqcd_cg, lqcd_cg_multishift, lqcd_rational_apply and *_host* call of this
 * context then uses it, at 8 (4) extra bytes per link and application: 1248 + 64 B per site in fp64.  The
 * buffer must stay valid while attached.  lqcd_fermion_force uses it too (the y_i = D_oe x_i of the phased operator
 * and F = TA[e^{i theta} U Q]); the gauge staples do not depend on it.  With a backfield the Dslash tuning options
 * dslash_minblocks and l2_hints have no effect.  Option "backfield_format" (before the first pack): 0 (default)
 * stores theta and evaluates sincos in the kernel; 1 stores (cos theta, sin theta), twice the bytes and no
 * sincos -- measured at 32^4: 104 vs 105 us (fp64 18-real), 90 vs 82 us (fp64 12-real).  async.
 */
size_t lqcd_backfield_bytes(const lqcd_ctx *ctx);
int lqcd_pack_backfield(lqcd_ctx *ctx, void *native_dev, const void *canonical_dev /* f64 [V][4] */);
int lqcd_set_backfield(lqcd_ctx *ctx, const void *backfield_native_dev /* or NULL */);
int lqcd_dslash_backfield(lqcd_ctx *ctx, int parity, void *out, const void *in, const void *links,
                          const void *backfield_native_dev);

/*
 * out_e = (mass^2 + sigma) in_e - D_eo (D_oe in_e)   (Eq. 8, shifted as in Eq. 6).
 * Needs a workspace (one odd-site temporary).  async.
 */
int lqcd_mdagm(lqcd_ctx *ctx, void *out_e, const void *in_e, const void *links, double mass,
               double sigma);

/*
 * lqcd_mdagm for callers that cannot supply a workspace because they cannot allocate device memory: a library
 * embedded in a program whose own allocator has already claimed the GPU's memory, a service that bans
 * cudaMalloc / cudaFree after start-up because both stall the whole device, a run planned to the last GB of HBM.
 * Same arguments, same arithmetic, same two Dslash launches (Eq. 8); the odd-site temporary sits in a
 * fixed array inside the library's device image instead of the caller's workspace, so no lqcd_set_workspace is
 * needed and the call makes no cudaMalloc, cudaFree or other allocating call.  (lqcd_create, which every context
 * needs once, does allocate < 1 MiB; do that at start-up.)
 *   Limit   lqcd_spinor_bytes(ctx) <= LQCD_NOALLOC_SCRATCH_BYTES (8 MiB: up to 24^4 or 32^3 x 8 in fp64, 32^3 x 16
 *           in fp32); beyond it LQCD_ERR_WORKSPACE with a message naming both sizes, nothing launched.
 *   Cost    every GPU onto which the library's device code is loaded holds those 8 MiB until the process ends,
 *           used or not.
 *   First call per device: looks up the array's device address (cudaGetSymbolAddress, which may load the device
 *           code); make that call during start-up, before any stream capture is begun.  Later calls only launch.
 *   Sharing  one array per device and process, used by every context and every call.  Nothing in it needs
 *           clearing (each call overwrites all it later reads), but it keeps the previous call's contents and
 *           two calls that can overlap on the GPU (issued on different streams) race on it.  Calls on one
 *           stream are safe.
 * async.  Errors: as lqcd_mdagm, plus LQCD_ERR_WORKSPACE (too large) and LQCD_ERR_UNSUPPORTED (slab contexts).
 */
#define LQCD_NOALLOC_SCRATCH_BYTES (8u << 20)
int lqcd_mdagm_noalloc(lqcd_ctx *ctx, void *out_e, const void *in_e, const void *links, double mass,
                       double sigma);

/*
 * Solve (mass^2 - D_eo D_oe) x_e = b_e by CG from x = 0 until ||r|| <= tol ||b|| (reading R10).
 *   x_e, b_e    native even-site vectors (device)
 *   iters       host, out: iterations performed (may be NULL)
 *   rel_resid   host, out: TRUE residual ||b - A x|| / ||b|| recomputed at exit (may be NULL)
 * blocking.  Returns LQCD_ERR_NOT_CONVERGED when max_iter is hit (outputs still filled, x at the
 * last iterate); LQCD_ERR_ARG for tol <= 0, max_iter < 1, null pointers; LQCD_ERR_WORKSPACE.
 */
int lqcd_cg(lqcd_ctx *ctx, void *x_e, const void *b_e, const void *links, double mass,
            double tol, int max_iter, int *iters, double *rel_resid);

/*
 * Solve (mass^2 + shifts[i] - D_eo D_oe) x_i = rhs_e for i = 0..nshift-1 with ONE operator
 * application per iteration (reading R11): shift i is frozen (sticky) once
 * |zeta_i| ||r|| <= tol ||rhs||; the loop ends when every shift is frozen.
 *   shifts        host, nshift doubles >= 0, any order; 1 <= nshift <= LQCD_MAX_SHIFTS
 *   rhs_e         native even-site vector (device)
 *   solutions_e   host array of nshift device pointers to native even-site vectors (out)
 *   iters         host, out: total iterations (may be NULL)
 *   conv_iter     host, out [nshift]: iteration at which each shift froze (may be NULL)
 *   rel_resid     host, out [nshift]: TRUE residuals at exit (may be NULL)
 * blocking.  Error behaviour as lqcd_cg; a negative shift is LQCD_ERR_ARG.  Also LQCD_ERR_ARG (before any
 * launch): a solution vector that is null, not 16-byte aligned, or overlaps rhs, another solution, the
 * workspace or the link field (the kernels assume distinct 16-byte aligned operands).
 */
int lqcd_cg_multishift(lqcd_ctx *ctx, int nshift, const double *shifts, const void *rhs_e,
                       void *const *solutions_e, const void *links, double mass, double tol,
                       int max_iter, int *iters, int *conv_iter, double *rel_resid);

/*
 * Rational function of A = mass^2 - D_eo D_oe applied to a vector, fused into the multi-shift
 * solve:
 *     y_e = c0 * rhs_e + sum_i coeffs[i] * x_i ,   (A + shifts[i]) x_i = rhs_e        (Eq. 6)
 * "the algebraic matrix function appearing in Eq. (3) is approximated ... by a
 * rational function" with the poles sigma_i of Eq. 6; this sum is what the
 * pseudofermion heatbath and the action evaluation (Algorithm 1 steps 3 and 6)
 * take from "the multishift inverter routine".  The solutions x_i are never stored: every
 * iteration adds coeffs[i]*alpha_i*p_i of the still-active shifts to y.  Same recurrences,
 * stopping rule and freezing as lqcd_cg_multishift (readings R11, R12).
 *   shifts, coeffs  host, nshift doubles each (shifts >= 0; coefficients any sign)
 *   rhs_e, y_e      native even-site vectors (device); must not alias
 *   iters, conv_iter  host outputs as in lqcd_cg_multishift (may be NULL)
 * blocking.  Needs the workspace of lqcd_workspace_bytes(ctx, nshift).  Errors as lqcd_cg_multishift
 * (LQCD_ERR_NOT_CONVERGED leaves y at the last iterate).
 */
int lqcd_rational_apply(lqcd_ctx *ctx, int nshift, const double *shifts, double c0,
                        const double *coeffs, const void *rhs_e, void *y_e, const void *links,
                        double mass, double tol, int max_iter, int *iters, int *conv_iter);

/*
 * Fermion-force outer products (the step after the
 * multi-shift solve).  The paper prints no formula (it follows its ref. 33); reading R21 of DESIGN.md:
 * for S = phi^dagger [c0 + sum_i c_i (A + sigma_i)^-1] phi, A = mass^2 - D_eo D_oe (Eq. 3, 6, 8), with
 * x_i = (A + sigma_i)^-1 phi on even sites, y_i = D_oe x_i on odd sites and w_i = x_i | y_i by parity,
 *     F_mu(x) = TA[ U_mu(x) Q_mu(x) ],
 *     Q_mu(x) = 1/2 eta_mu(x) s+_mu(x) (-1)^{p(x)} sum_i c_i w_i(x+mu) w_i(x)^dagger,
 *     TA[M]   = (M - M^dagger)/2 - Tr(M - M^dagger)/6,
 * so that dS/d eps = 2 Re Tr[ i T F_mu(x) ] under U_mu(x) -> exp(i eps T) U_mu(x).
 *   coeffs   host, nshift doubles (the c_i; c0 does not enter the force)
 *   xs_e     host array of nshift device pointers: the solutions x_i (native even-site vectors, e.g.
 *            from lqcd_cg_multishift); read only
 *   force    native force field (device, lqcd_tamat_bytes; out).  F is traceless anti-Hermitian, so it is
 *            stored as 8 reals per link -- the paper's tamat_soa: F01, F02, F12 and
 *            (Im F00, Im F11); layout private, read it back with lqcd_unpack_tamat
 * The y_i are computed inside (nshift Dslash applications into the workspace of
 * lqcd_workspace_bytes(ctx, nshift)).  async.  In slab mode (either transport) xs_e are vectors of the context's
 * solve_parity, the ghost slices of the x_i and y_i are filled by halo exchanges inside the call (those of the caller's
 * x_i are overwritten), and only the owned links of `force` are written.
 */
size_t lqcd_tamat_bytes(const lqcd_ctx *ctx); /* 8-real traceless anti-Hermitian field (fermion force)  */
size_t lqcd_force_bytes(const lqcd_ctx *ctx); /* generic 3x3-complex-per-link field (gauge staples)          */
int lqcd_fermion_force(lqcd_ctx *ctx, int nshift, const double *coeffs, void *const *xs_e,
                       const void *links, void *force);
/* native 8-real (tamat) field -> canonical complex128 F[lex][mu][row][col] (device).  async. */
int lqcd_unpack_tamat(lqcd_ctx *ctx, void *canonical_dev /* c128 [V][4][3][3] */, const void *native);
/* native 3x3-per-link field (staples) -> canonical complex128 [lex][mu][row][col] (device).  async. */
int lqcd_unpack_force(lqcd_ctx *ctx, void *canonical_dev /* c128 [V][4][3][3] */, const void *native);

/*
 * Gauge staples of the tree-level Symanzik improved action (PAPER.md:105,
 * 365-393: "products of 3 and 5 SU(3) matrices representing links on C-shaped paths", Listing 3).
 * The paper prints neither paths nor coefficients; reading R22 of DESIGN.md: with
 *   W[U] = sum_x sum_{mu<nu} { c0 Re Tr P_{mu nu}(x) + c1 [Re Tr R_{mu nu}(x) + Re Tr R_{nu mu}(x)] }
 * (P the 1x1 plaquette, R_{mu nu} the 2x1 rectangle; tree-level Symanzik: c0 = 5/3, c1 = -1/12),
 *   staples[x][mu] = S_mu(x) = sum over the loops of W through U_mu(x) of coefficient x (remaining
 *   links, ordered from x+mu back to x), i.e. W = Re Tr[U_mu(x) S_mu(x)] + (terms without U_mu(x)):
 * per nu != mu two 3-link and six 5-link paths.  Links are periodic in all four directions.
 *   links    native link field (device); staples: native 3x3-per-link field (device, lqcd_force_bytes;
 *            layout private: read it back with lqcd_unpack_force)
 * Algorithm (option "staples_variant"): 2 (default) runs two passes through the 24 stored 3-link staples per
 * site, 39 SU(3) products per link; it needs lqcd_staples_workspace_bytes(ctx) bytes in the workspace given to
 * lqcd_set_workspace (contents destroyed) -- with no or a smaller workspace, and for variant 1, the one-pass
 * kernel with shared sub-products runs (66 products per link, no workspace); 0 walks every path on its own
 * (84 products).  All three agree to rounding.  Read-only option "staples_ran": the variant the last call used.
 * async.  LQCD_ERR_UNSUPPORTED in slab mode.
 */
size_t lqcd_staples_workspace_bytes(const lqcd_ctx *ctx);
int lqcd_gauge_staples(lqcd_ctx *ctx, const void *links, void *staples, double c0, double c1);

/*
 * ---- Slab mode: one x3 slab per GPU (the paper leaves the
 * multi-device version as future work) --------------------------------------
 * A rank that owns L3 = N3/P time slices creates its context with dims (N0,N1,N2,L3+2) and
 * antiperiodic_t = 0: slices 1..L3 are owned, slices 0 and L3+1 are ghost copies of the neighbours'
 * boundary slices (ghost depth 1, so the local parity is the opposite of the global one when
 * r*L3 is even).  The staggered phases do not depend on x3 and the antiperiodic sign is applied to
 * the ghost data when it crosses the global boundary (lqcd_halo_pack's `sign`), so the slab is an
 * ordinary lattice on which only the owned slices are computed.
 */

/* out(x) = (D in)(x) for the sites of `parity` with x3 in [x3_lo, x3_hi) only; the other sites of
 * `out` are not touched.  0 <= x3_lo < x3_hi <= N3.  async.  Lets the caller run the interior
 * slices while the halo is in flight and the two boundary slices afterwards. */
int lqcd_dslash_slices(lqcd_ctx *ctx, int parity, void *out, const void *in, const void *links,
                       int x3_lo, int x3_hi);

/* Bytes of one x3 slice of a native half vector (both parities have N0*N1*N2/2 sites per slice). */
size_t lqcd_halo_bytes(const lqcd_ctx *ctx);
/* buf = sign * (slice x3 of spinor), contiguous (device, lqcd_halo_bytes);  async. */
int lqcd_halo_pack(lqcd_ctx *ctx, void *buf, const void *spinor, int x3, double sign);
/* slice x3 of spinor = buf;  async. */
int lqcd_halo_unpack(lqcd_ctx *ctx, void *spinor, const void *buf, int x3);

/* Both faces in one launch each way, for a context whose owned slices were set with lqcd_set_slab:
 * buf_top = sign_top * (slice x3_hi-1), buf_bottom = sign_bottom * (slice x3_lo); and ghost slice
 * x3_lo-1 = buf_from_down, ghost slice x3_hi = buf_from_up.  async. */
int lqcd_halo_pack_faces(lqcd_ctx *ctx, void *buf_top, void *buf_bottom, const void *spinor,
                         double sign_top, double sign_bottom);
int lqcd_halo_unpack_ghosts(lqcd_ctx *ctx, void *spinor, const void *buf_from_down, const void *buf_from_up);

/*
 * Communication hooks for the solvers in slab mode.  The library does not link a communication
 * library: the caller (torch.distributed / NCCL in paper_1701_00426_b200/slab.py) supplies
 *   halo(user, vec, parity)       fill the ghost slices 0 and N3-1 of the native half vector `vec`
 *                                 from the neighbours (work enqueued on / ordered with the context's
 *                                 stream); returns 0 on success
 *   allreduce(user, dev, count)   sum `count` device doubles at `dev` over all ranks, in place,
 *                                 ordered with the context's stream; returns 0 on success
 * With hooks set, lqcd_cg / lqcd_cg_multishift / lqcd_rational_apply / lqcd_mdagm restrict every
 * vector operation and dot product to the owned slices [x3_lo, x3_hi), call `halo` before each
 * Dslash, and complete each dot product with `allreduce` before the scalar recurrences (which then
 * run in a one-thread kernel instead of the last CTA of the reduction).  Pass NULLs to clear.
 * x3_lo/x3_hi: owned slices (1 and N3-1 for ghost depth 1).  solve_parity: LOCAL parity of the sites
 * the solvers and lqcd_mdagm act on -- the paper's even sites (Eq. 8) are the local ODD sites of a slab
 * whose first owned slice sits at an odd local x3 (ghost depth 1, even global offset); the solver then
 * uses D(1-solve_parity <- solve_parity) first.  The "_e" buffers of those calls are vectors of that parity.
 */
typedef int (*lqcd_halo_fn)(void *user, void *vec, int parity);
typedef int (*lqcd_allreduce_fn)(void *user, void *dev_doubles, int count);
int lqcd_set_slab(lqcd_ctx *ctx, int x3_lo, int x3_hi, int solve_parity, lqcd_halo_fn halo,
                  lqcd_allreduce_fn allreduce, void *user);

/*
 * ---- Slab mode over peer-to-peer memory inside one node (the native transport; "direct
 * P2P stores into the neighbour's ghost slice", two all-reduces of one double per CG iteration) --------------------
 * No communication library and no host code between the kernels: every rank owns one block of device memory
 * (flags, P slots per reduction, four landing buffers for halo faces) that all ranks of the node map -- through
 * CUDA IPC with one process per GPU, or as plain pointers when the ranks share a process.  The protocol as built
 * (csrc/peer.cuh is the reference; this is its summary):
 *   Halo.  The two boundary slices of a vector (times the boundary sign) are stored straight into the neighbours'
 *     landing buffers by the kernel that PRODUCES the vector inside a solve (the init kernel and K2 for p, the first
 *     Dslash of the iteration for D p); a stand-alone lqcd_dslash / lqcd_dslash_backfield / lqcd_mdagm uses one small
 *     push kernel instead.  Thread 0 of the Dslash that follows in the stream raises the neighbours' flags (the kernel
 *     boundary has completed the stores), and only the tiles of that Dslash that touch a boundary slice wait for the
 *     rank's own two flags; they take the x3 hops that leave the slab from the landing buffers, the interior tiles
 *     compute meanwhile.
 *   Dot products.  The producer (Dslash with <p,q>, K1 with <r,r>) leaves per-CTA partials, as on one GPU.  Every CTA
 *     of the CONSUMER kernel (K1, K2) adds them up for itself; its CTA 0 stores the rank's sum into every rank's slot
 *     and raises the flags; every CTA waits for the OTHER ranks' flags only and adds the P sums in rank order, so
 *     every rank gets the bit-identical total and takes the same decisions.
 * The waits are inside the kernels: the CG loop stays one CUDA graph per chunk of iterations.  Flags are monotone
 * counters; re-use of slots and landing buffers is ordered by the two all-reduces of every iteration and by the
 * alternation of the two exchange kinds (even / odd input vector); where a caller exchanges the same kind twice in a
 * row (lqcd_dslash twice for one parity, a solve right after it) the library puts a device-side barrier (a dummy
 * all-reduce) in between by itself.
 * STATUS: verified on ONE GPU only (virtual ranks in lock step, P = 1, 2, 4, and a cooperative-kernel self-test of
 * the flag protocol under real concurrency).  With P >= 2 real devices the path has never executed: the assumption
 * it rests on -- peer stores issued by kernel N are performed at the remote GPU before the st.release.sys that
 * kernel N+1 issues after its griddepcontrol.wait -- is UNVERIFIED ON HARDWARE.
 * Teardown: lqcd_peer_disconnect and lqcd_destroy free the rank's block after finishing only this rank's stream; a
 * neighbour's last kernel may still be storing into it.  Every rank must finish its stream and meet the others at a
 * host barrier before any rank disconnects or destroys (SlabLattice.close does).
 *   lqcd_peer_init      allocate the block; the context must have local extents (N0,N1,N2,L3+2) and antiperiodic_t
 *                       = 0 as described above; x3_lo/x3_hi/solve_parity as in lqcd_set_slab; sign_up / sign_down:
 *                       factor applied to the face sent to the rank above / below (-1 where the hop crosses an
 *                       antiperiodic global boundary, reading R4).  *block (may be NULL): the block's device
 *                       address.  1 <= nranks <= 16.  blocking.
 *   lqcd_peer_export    CUDA IPC handle (64 bytes) of the block, for the other processes
 *   lqcd_peer_import    map another rank's block from its handle -> device pointer valid in this process
 *   lqcd_peer_connect   blocks[r] = device pointer to rank r's block for every r (blocks[rank] is ignored);
 *                       from now on lqcd_dslash, lqcd_mdagm, lqcd_cg, lqcd_cg_multishift and
 *                       lqcd_rational_apply of this context exchange faces and sums through the blocks.
 *                       lqcd_dslash_slices stays raw (reads the vector's own ghost slices).
 *   lqcd_peer_disconnect  back to a single-rank context (frees the block, closes imported mappings).  blocking.
 * All ranks must issue the same sequence of calls (as with any collective).  With nranks = 1 the rank is its own
 * neighbour.  A backfield works as on one GPU (the slab's phases include the ghost slices, like its links);
 * lqcd_fermion_force works too (faces pushed and then pulled into the vectors' ghost slices);
 * lqcd_gauge_staples is LQCD_ERR_UNSUPPORTED in this mode (it would need ghost depth 2).
 * A wait for another rank never lasts longer than option peer_wait_ms (default 3000): a wait that gives up is counted
 * in the rank's block and the rank's transport is then DEAD -- every later wait returns at once, a running solve stops
 * at its next convergence poll, and this and every later solver call return LQCD_ERR_CUDA ("... waits for other ranks
 * timed out"; the results are meaningless) until lqcd_peer_disconnect + lqcd_peer_init build a new block.
 * lqcd_get_option(ctx, "peer_timeouts") reads the count (blocking) after lqcd_dslash / lqcd_mdagm.
 * The kernels of different ranks wait for one another: run each rank on its own GPU.  (Validation on ONE GPU: the
 * lock-step hook and the protocol self-test of include/lqcd_diag.h.)
 */
size_t lqcd_peer_block_bytes(const lqcd_ctx *ctx);
int lqcd_peer_init(lqcd_ctx *ctx, int nranks, int rank, int x3_lo, int x3_hi, int solve_parity,
                   double sign_up, double sign_down, void **block);
int lqcd_peer_export(lqcd_ctx *ctx, void *handle64);
int lqcd_peer_import(lqcd_ctx *ctx, int rank, const void *handle64, void **block);
int lqcd_peer_connect(lqcd_ctx *ctx, void *const *blocks);
int lqcd_peer_disconnect(lqcd_ctx *ctx);

/*
 * After lqcd_cg / lqcd_cg_multishift: copy up to `n` entries of the per-iteration history
 * (alpha_k, beta_k, ||r_{k+1}||) of the last solve to host arrays (any may be NULL).
 * Returns the number of entries available (<= 64), or a negative status.
 */
int lqcd_solver_history(lqcd_ctx *ctx, int n, double *alpha, double *beta, double *rnorm);

/*
 * End-to-end entry points on HOST buffers in the canonical layout: host->device copy, pack,
 * compute on the GPU, unpack, device->host copy, all inside the call.  blocking.
 * They allocate and free their own device staging memory (cudaMalloc), unlike the calls above.
 */
int lqcd_dslash_host(lqcd_ctx *ctx, int parity, void *out_host /* c128 [V/2][3] */,
                     const void *in_host /* c128 [V/2][3] */,
                     const void *links_host /* c128 [V][4][3][3] */);
/* As lqcd_dslash_host with the link field already resident on the device in NATIVE form (packed once per
 * gauge configuration -- the paper moves fields only at the start and end of an update):
 * only the input and output vectors cross the bus.  blocking. */
int lqcd_dslash_host_vectors(lqcd_ctx *ctx, int parity, void *out_host /* c128 [V/2][3] */,
                             const void *in_host /* c128 [V/2][3] */, const void *links_native_dev);
/* n applications outs_host[j] = D ins_host[j] (output parity parities[j]) in ONE pipelined call: uploads,
 * pack -> Dslash -> unpack, and downloads run on three streams chained by events with double-buffered
 * staging, so the download of application j overlaps the upload of application j+1 (PCIe is full duplex).
 * Host buffers should be pinned (pageable memory works but serialises the copies).  outs/ins: host arrays
 * of n host pointers (c128 [V/2][3] each); an output may not alias any input.  blocking. */
int lqcd_dslash_host_vectors_batch(lqcd_ctx *ctx, int n, const int *parities, void *const *outs_host,
                                   const void *const *ins_host, const void *links_native_dev);
/* lqcd_cg_multishift on host vectors with the link field resident in native form (the operator is uploaded
 * once per gauge configuration): rhs up, nshift solutions down, the 10^2-10^3 operator
 * applications in between (PAPER.md:173 fn. c) never leave the device.  Needs the workspace of
 * lqcd_workspace_bytes(ctx, nshift).  blocking; errors as lqcd_cg_multishift. */
int lqcd_cg_multishift_host_vectors(lqcd_ctx *ctx, int nshift, const double *shifts,
                                    const void *rhs_host /* c128 [V/2][3] */,
                                    void *solutions_host /* c128 [nshift][V/2][3] */,
                                    const void *links_native_dev, double mass, double tol, int max_iter,
                                    int *iters, int *conv_iter, double *rel_resid);
int lqcd_cg_multishift_host(lqcd_ctx *ctx, int nshift, const double *shifts,
                            const void *rhs_host /* c128 [V/2][3] */,
                            void *solutions_host /* c128 [nshift][V/2][3] */,
                            const void *links_host, double mass, double tol, int max_iter,
                            int *iters, int *conv_iter, double *rel_resid);

/* Validation and measurement helpers that are NOT part of the ABI of SURVEY.md section 8(b) live in lqcd_diag.h. */

#ifdef __cplusplus
}
#endif
#endif /* LQCD_H */

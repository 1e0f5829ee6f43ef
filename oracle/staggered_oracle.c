/*
 * staggered_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU (C99, fp64) restatement of what the hot path of
 * arxiv/paper_1701_00426 computes: the even/odd staggered Dirac operator D_eo / D_oe
 * (Eq. 7), the even/odd-preconditioned normal operator
 * m^2 - D_eo D_oe (Eq. 8), the conjugate gradient and the multi-shift
 * ("shifted") conjugate gradient on it (Eq. 6), and the
 * third-row reconstruction r2 = (r0 ^ r1)* (PAPER.md:272).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call this file.  It shares no code, header, table or helper with the CUDA path
 * under paper_1701_00426_b200/ and deliberately uses the opposite data organisation:
 * array-of-structures, full-lattice lexicographic arrays, neighbours from coordinates
 * with '%', no parity-split storage, no blocking, no fusion.
 *
 * The paper never writes the stencil, the phases, the boundary conditions, the CG or the
 * multi-shift recurrences; the readings used here are listed one by one in DESIGN.md
 * ("Readings of the paper", R1..R19 = SURVEY.md section 8(c) #1..#19).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): dense 3V x 3V matrix built independently
 * in numpy at 2^4 and 4^4; free-field plane-wave spectrum m^2 + sum_mu sin^2 p_mu;
 * constant-spinor closed form for the antiperiodic boundary; <phi,D_eo psi> = -<D_oe phi,psi>;
 * gauge covariance; reconstructed row 3 against the generator's Gram-Schmidt row 3;
 * CG / multi-shift against dense numpy.linalg.solve; the identity
 * b - (A + sigma_i) x_i = zeta_i r; one-iteration convergence on a plane wave; the
 * rational-function sum against dense solves and a partial-fraction identity; the fermion-force
 * outer products against finite differences of the action computed with dense solves; the gauge
 * staples against finite differences of the gauge action, a loop-counting sum rule and covariance.
 * The optional backfield (U(1) phase per link, the paper's unexplained fourth argument of acc_Deo; *_bf
 * entry points) is pinned by: theta = 0 reproduces D; the dense matrix built with phased links; the
 * phases absorbed into the links give the same D through the plain entry points; a constant theta_mu
 * shifts the free-field momenta, p_mu -> p_mu + theta_mu; a pure-gauge theta is removed by a U(1) gauge
 * transformation; the fermion force with a backfield by finite differences of the action with phased dense solves.
 * No function in this file is "parity unpinned".
 *
 * OpenMP is used on the site loop of the operator only, so that bench.py can time the
 * oracle on all host cores; every reduction is a plain serial loop in site order.
 *
 * Canonical layout (same as lqcd_inputs/fields.py):
 *   lex = x0 + N0*(x1 + N1*(x2 + N2*x3));  U[lex][mu][row][col];  psi[lex][c];
 *   half vector of parity p: phi[idxh][c], idxh = lex/2 (Eq. 9).
 */
#include <complex.h>
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>

typedef double _Complex cplx;

static size_t vol(const int N[4]) { return (size_t)N[0] * N[1] * N[2] * N[3]; }

static size_t lex_of(const int N[4], const int x[4])
{
    return (size_t)x[0] + (size_t)N[0] * ((size_t)x[1] + (size_t)N[1] * ((size_t)x[2] + (size_t)N[2] * (size_t)x[3]));
}

static void coords_of(const int N[4], size_t lex, int x[4])
{
    x[0] = (int)(lex % (size_t)N[0]); lex /= (size_t)N[0];
    x[1] = (int)(lex % (size_t)N[1]); lex /= (size_t)N[1];
    x[2] = (int)(lex % (size_t)N[2]); lex /= (size_t)N[2];
    x[3] = (int)lex;
}

static int parity_of(const int x[4]) { return (x[0] + x[1] + x[2] + x[3]) % 2; }

/* Reading R3: eta_0 = 1, eta_mu(x) = (-1)^(x_0 + ... + x_{mu-1})  (BASELINE.json config 1). */
static double eta(int mu, const int x[4])
{
    int s = 0;
    for (int nu = 0; nu < mu; ++nu) s += x[nu];
    return (s % 2) ? -1.0 : 1.0;
}

/*
 * (D psi)(x) for ONE site (readings R1, R2, R4):
 *
 *   (D psi)(x) = 1/2 sum_mu eta_mu(x) [ s+_mu(x) U_mu(x) psi(x+mu) - s-_mu(x) U_mu(x-mu)^dagger psi(x-mu) ]
 *
 * x +- mu is taken modulo N_mu; s+- = +1 except, with antiperiodic_t, s+_3 = -1 when
 * x3 = N3-1 and s-_3 = -1 when x3 = 0.  The two hops are separate terms, so N_mu = 2 needs
 * no special case.
 */
/*
 * Optional `backfield` theta[lex][mu] (NULL: none): the fourth argument of the paper's
 * acc_Deo(u, out, in, backfield) (Listing 2), a per-link real field ("double_soa") the
 * paper never explains.  Reading R6 of DESIGN.md: an external U(1) phase -- every link enters D as
 * e^{i theta_mu(x)} U_mu(x), i.e. the forward hop out of x carries e^{+i theta_mu(x)} and the backward hop
 * carries (e^{i theta_mu(x-mu)} U_mu(x-mu))^dagger = e^{-i theta_mu(x-mu)} U_mu(x-mu)^dagger.  The phase
 * multiplies the full 3x3 link (after any third-row reconstruction), never the stored rows.
 */
static void dirac_site(const int N[4], int antiperiodic_t, const cplx *U, const double *theta, const cplx *psi,
                       const int x[4], cplx out[3])
{
    cplx acc[3] = {0.0, 0.0, 0.0};
    for (int mu = 0; mu < 4; ++mu) {
        int xp[4] = {x[0], x[1], x[2], x[3]};
        int xm[4] = {x[0], x[1], x[2], x[3]};
        xp[mu] = (x[mu] + 1) % N[mu];
        xm[mu] = (x[mu] - 1 + N[mu]) % N[mu];
        double sp = 1.0, sm = 1.0;
        if (antiperiodic_t && mu == 3) {
            if (x[3] == N[3] - 1) sp = -1.0;
            if (x[3] == 0) sm = -1.0;
        }
        const cplx *Ufwd = U + (lex_of(N, x) * 4 + (size_t)mu) * 9;   /* U_mu(x)      */
        const cplx *Ubwd = U + (lex_of(N, xm) * 4 + (size_t)mu) * 9;  /* U_mu(x - mu) */
        const cplx *pf = psi + lex_of(N, xp) * 3;
        const cplx *pb = psi + lex_of(N, xm) * 3;
        double e = eta(mu, x);
        for (int a = 0; a < 3; ++a) {
            cplx fwd = 0.0, bwd = 0.0;
            for (int b = 0; b < 3; ++b) {
                fwd += Ufwd[a * 3 + b] * pf[b];
                bwd += conj(Ubwd[b * 3 + a]) * pb[b];   /* (U^dagger)_{ab} = conj(U_{ba}) */
            }
            if (theta) {
                fwd *= cexp(I * theta[lex_of(N, x) * 4 + (size_t)mu]);
                bwd *= cexp(-I * theta[lex_of(N, xm) * 4 + (size_t)mu]);
            }
            acc[a] += e * (sp * fwd - sm * bwd);
        }
    }
    for (int a = 0; a < 3; ++a) out[a] = 0.5 * acc[a];
}

/* Full-lattice D: out(x) = (D psi)(x) on the sites whose parity matches `which`
 * (0 = even only, 1 = odd only, 2 = all); other sites of `out` are left untouched. */
void oracle_dirac_full_bf(const int N[4], int antiperiodic_t, const cplx *U, const double *theta,
                          const cplx *psi, cplx *out, int which)
{
    long long V = (long long)vol(N);
#pragma omp parallel for schedule(static)
    for (long long s = 0; s < V; ++s) {
        int x[4];
        coords_of(N, (size_t)s, x);
        if (which != 2 && parity_of(x) != which) continue;
        dirac_site(N, antiperiodic_t, U, theta, psi, x, out + (size_t)s * 3);
    }
}

void oracle_dirac_full(const int N[4], int antiperiodic_t, const cplx *U, const cplx *psi,
                       cplx *out, int which)
{
    oracle_dirac_full_bf(N, antiperiodic_t, U, NULL, psi, out, which);
}

/* Sites lex in [lo, hi) only (a bounded sample of a large lattice for bench.py's timed CPU
 * baseline); other sites of `out` are left untouched. */
void oracle_dirac_range(const int N[4], int antiperiodic_t, const cplx *U, const cplx *psi,
                        cplx *out, long long lo, long long hi)
{
#pragma omp parallel for schedule(static)
    for (long long s = lo; s < hi; ++s) {
        int x[4];
        coords_of(N, (size_t)s, x);
        dirac_site(N, antiperiodic_t, U, NULL, psi, x, out + (size_t)s * 3);
    }
}

/* One output site, for sampled parity checks at sizes where the full field is not wanted. */
void oracle_dirac_site_bf(const int N[4], int antiperiodic_t, const cplx *U, const double *theta,
                          const cplx *psi, const int x[4], cplx out[3])
{
    dirac_site(N, antiperiodic_t, U, theta, psi, x, out);
}

void oracle_dirac_site(const int N[4], int antiperiodic_t, const cplx *U, const cplx *psi,
                       const int x[4], cplx out[3])
{
    dirac_site(N, antiperiodic_t, U, NULL, psi, x, out);
}

/* ---------------------------------------------------------------------------------------
 * Half-lattice (even/odd) views.  phi[idxh], idxh = lex/2 over the sites of one parity
 * (Eq. 9).
 * ------------------------------------------------------------------------------------- */

/* full <- half of the given parity; sites of the other parity are set to zero. */
void oracle_half_to_full(const int N[4], int parity, const cplx *half, cplx *full)
{
    size_t V = vol(N);
    for (size_t s = 0; s < V; ++s) {
        int x[4];
        coords_of(N, s, x);
        for (int c = 0; c < 3; ++c)
            full[s * 3 + c] = (parity_of(x) == parity) ? half[(s / 2) * 3 + c] : 0.0;
    }
}

void oracle_full_to_half(const int N[4], int parity, const cplx *full, cplx *half)
{
    size_t V = vol(N);
    for (size_t s = 0; s < V; ++s) {
        int x[4];
        coords_of(N, s, x);
        if (parity_of(x) != parity) continue;
        for (int c = 0; c < 3; ++c) half[(s / 2) * 3 + c] = full[s * 3 + c];
    }
}

/*
 * Reading R5: the first index of D_eo / D_oe is the parity of the OUTPUT sites.
 *   out_parity = 0 (even):  out_e = D_eo in_o      out_parity = 1 (odd):  out_o = D_oe in_e
 * Returns 0, or -1 if scratch memory cannot be allocated.
 */
int oracle_dslash_half_bf(const int N[4], int antiperiodic_t, const cplx *U, const double *theta, int out_parity,
                          const cplx *in_half, cplx *out_half)
{
    size_t V = vol(N);
    cplx *full_in = (cplx *)malloc(V * 3 * sizeof(cplx));
    cplx *full_out = (cplx *)malloc(V * 3 * sizeof(cplx));
    if (!full_in || !full_out) { free(full_in); free(full_out); return -1; }
    oracle_half_to_full(N, 1 - out_parity, in_half, full_in);
    oracle_dirac_full_bf(N, antiperiodic_t, U, theta, full_in, full_out, out_parity);
    oracle_full_to_half(N, out_parity, full_out, out_half);
    free(full_in);
    free(full_out);
    return 0;
}

int oracle_dslash_half(const int N[4], int antiperiodic_t, const cplx *U, int out_parity,
                       const cplx *in_half, cplx *out_half)
{
    return oracle_dslash_half_bf(N, antiperiodic_t, U, NULL, out_parity, in_half, out_half);
}

/*
 * Eq. 8 with an optional shift (Eq. 6):
 *   out_e = (m^2 + sigma) in_e - D_eo ( D_oe in_e )
 */
int oracle_mdagm_bf(const int N[4], int antiperiodic_t, const cplx *U, const double *theta, double mass,
                    double sigma, const cplx *in_e, cplx *out_e)
{
    size_t Vh = vol(N) / 2;
    cplx *tmp_o = (cplx *)malloc(Vh * 3 * sizeof(cplx));
    if (!tmp_o) return -1;
    int rc = oracle_dslash_half_bf(N, antiperiodic_t, U, theta, 1, in_e, tmp_o);      /* D_oe in_e   */
    if (!rc) rc = oracle_dslash_half_bf(N, antiperiodic_t, U, theta, 0, tmp_o, out_e); /* D_eo (...) */
    if (!rc)
        for (size_t i = 0; i < Vh * 3; ++i) out_e[i] = (mass * mass + sigma) * in_e[i] - out_e[i];
    free(tmp_o);
    return rc;
}

int oracle_mdagm(const int N[4], int antiperiodic_t, const cplx *U, double mass, double sigma,
                 const cplx *in_e, cplx *out_e)
{
    return oracle_mdagm_bf(N, antiperiodic_t, U, NULL, mass, sigma, in_e, out_e);
}

/*
 * Third-row reconstruction: r2 = (r0 ^ r1)^*  (reading R8):
 *   r2[k] = conj( eps_{kij} r0[i] r1[j] )
 * u points at one row-major 3x3 matrix; rows 0,1 are read, row 2 is overwritten.
 */
void oracle_reconstruct_row3(cplx *u)
{
    const cplx *r0 = u, *r1 = u + 3;
    u[6] = conj(r0[1] * r1[2] - r0[2] * r1[1]);
    u[7] = conj(r0[2] * r1[0] - r0[0] * r1[2]);
    u[8] = conj(r0[0] * r1[1] - r0[1] * r1[0]);
}

/* n matrices in place. */
void oracle_reconstruct_row3_field(cplx *U, size_t n)
{
    for (size_t i = 0; i < n; ++i) oracle_reconstruct_row3(U + i * 9);
}

/* Re<a,b> = Re sum conj(a_i) b_i, plain serial loop (reading R13). */
static double re_dot(const cplx *a, const cplx *b, size_t n)
{
    double s = 0.0;
    for (size_t i = 0; i < n; ++i) s += creal(a[i]) * creal(b[i]) + cimag(a[i]) * cimag(b[i]);
    return s;
}

/* ---------------------------------------------------------------------------------------
 * Conjugate gradient for A x = b, A = m^2 - D_eo D_oe, reading R10:
 * textbook CG, x0 = 0, stop on the recursive residual ||r|| <= tol ||b||.
 *
 *   x = 0, r = p = b, rho = <r,r>
 *   loop:  q = A p;  alpha = rho / Re<p,q>;  x += alpha p;  r -= alpha q;  rho' = <r,r>
 *          stop if sqrt(rho') <= tol ||b||
 *          beta = rho'/rho;  p = r + beta p;  rho = rho'
 *
 * hist_alpha / hist_beta / hist_rnorm (each hist_len doubles, may be NULL) receive
 * alpha_k, beta_k and ||r_{k+1}|| of the first hist_len iterations.
 * true_relres = || b - A x || / || b || recomputed at exit.
 * Returns 0 converged, 1 hit max_iter, -1 allocation failure.
 * ------------------------------------------------------------------------------------- */
int oracle_cg_bf(const int N[4], int antiperiodic_t, const cplx *U, const double *theta, double mass,
                 const cplx *b, cplx *x, double tol, int max_iter,
                 int *iters, double *true_relres,
                 double *hist_alpha, double *hist_beta, double *hist_rnorm, int hist_len)
{
    size_t n = vol(N) / 2 * 3;
    cplx *r = (cplx *)malloc(n * sizeof(cplx));
    cplx *p = (cplx *)malloc(n * sizeof(cplx));
    cplx *q = (cplx *)malloc(n * sizeof(cplx));
    if (!r || !p || !q) { free(r); free(p); free(q); return -1; }
    int rc = 1, k = 0;
    for (size_t i = 0; i < n; ++i) { x[i] = 0.0; r[i] = b[i]; p[i] = b[i]; }
    double rho = re_dot(r, r, n);
    double bnorm = sqrt(rho);
    if (bnorm == 0.0) { rc = 0; goto done; }
    for (k = 0; k < max_iter; ++k) {
        if (oracle_mdagm_bf(N, antiperiodic_t, U, theta, mass, 0.0, p, q)) { rc = -1; goto done; }
        double alpha = rho / re_dot(p, q, n);
        for (size_t i = 0; i < n; ++i) x[i] += alpha * p[i];
        for (size_t i = 0; i < n; ++i) r[i] -= alpha * q[i];
        double rho_new = re_dot(r, r, n);
        if (k < hist_len) {
            if (hist_alpha) hist_alpha[k] = alpha;
            if (hist_rnorm) hist_rnorm[k] = sqrt(rho_new);
        }
        if (sqrt(rho_new) <= tol * bnorm) { ++k; rc = 0; break; }
        double beta = rho_new / rho;
        if (k < hist_len && hist_beta) hist_beta[k] = beta;
        for (size_t i = 0; i < n; ++i) p[i] = r[i] + beta * p[i];
        rho = rho_new;
    }
done:
    if (iters) *iters = k;
    if (true_relres) {
        if (bnorm == 0.0 || rc < 0) *true_relres = 0.0;
        else {
            oracle_mdagm_bf(N, antiperiodic_t, U, theta, mass, 0.0, x, q);
            for (size_t i = 0; i < n; ++i) q[i] = b[i] - q[i];
            *true_relres = sqrt(re_dot(q, q, n)) / bnorm;
        }
    }
    free(r); free(p); free(q);
    return rc;
}

int oracle_cg(const int N[4], int antiperiodic_t, const cplx *U, double mass,
              const cplx *b, cplx *x, double tol, int max_iter,
              int *iters, double *true_relres,
              double *hist_alpha, double *hist_beta, double *hist_rnorm, int hist_len)
{
    return oracle_cg_bf(N, antiperiodic_t, U, NULL, mass, b, x, tol, max_iter, iters, true_relres,
                        hist_alpha, hist_beta, hist_rnorm, hist_len);
}

/* ---------------------------------------------------------------------------------------
 * Multi-shift CG for (A + sigma_i) x_i = b, i = 0..nshift-1 (Eq. 6: "solve
 * all the equations at the same time, using at each iteration only one matrix-vector
 * product", refs 39,40).  The recurrences are not in the paper; reading R11:
 *
 *   base system A_b = A + sigma_min, delta_i = sigma_i - sigma_min >= 0
 *   x_i = 0, p_i = p = r = b, zeta_i^old = zeta_i = 1, alpha_prev = 1, beta_prev = 0, rho = <b,b>
 *   loop n = 0,1,...
 *     q = A_b p ;  alpha = rho / Re<p,q>
 *     for each i:  zeta_i^new = zeta_i zeta_i^old alpha_prev /
 *                      ( alpha beta_prev (zeta_i^old - zeta_i) + zeta_i^old alpha_prev (1 + delta_i alpha) )
 *                  alpha_i = alpha zeta_i^new / zeta_i
 *                  if active_i:  x_i += alpha_i p_i
 *     r -= alpha q ;  rho' = <r,r> ;  beta = rho'/rho ;  p = r + beta p
 *     for each i:  beta_i = beta (zeta_i^new / zeta_i)^2
 *                  if active_i:  p_i = zeta_i^new r + beta_i p_i
 *     (zeta_i^old, zeta_i) = (zeta_i, zeta_i^new); alpha_prev = alpha; beta_prev = beta; rho = rho'
 *     active_i = active_i AND ( |zeta_i| sqrt(rho) > tol ||b|| )          -- sticky
 *     stop when no shift is active
 *
 * The residual of system i is zeta_i r (never formed).
 *
 * x:            nshift vectors, contiguous, x[i*n .. (i+1)*n)
 * conv_iter[i]: iteration count at which shift i froze (or the final count)
 * true_relres:  || b - (A + sigma_i) x_i || / ||b|| at exit, per shift
 * zeta_out[i]:  zeta_i at exit;  r_out: r at exit (either may be NULL)
 * Returns 0 all converged, 1 hit max_iter, -1 allocation failure, -2 bad shifts.
 * ------------------------------------------------------------------------------------- */
int oracle_cg_multishift_bf(const int N[4], int antiperiodic_t, const cplx *U, const double *theta, double mass,
                            int nshift, const double *sigma, const cplx *b, cplx *x,
                            double tol, int max_iter,
                            int *iters, int *conv_iter, double *true_relres,
                            double *zeta_out, cplx *r_out,
                            double *hist_alpha, double *hist_beta, double *hist_rnorm, int hist_len)
{
    if (nshift < 1) return -2;
    size_t n = vol(N) / 2 * 3;
    double sigma_min = sigma[0];
    for (int i = 0; i < nshift; ++i) {
        if (sigma[i] < 0.0) return -2;
        if (sigma[i] < sigma_min) sigma_min = sigma[i];
    }
    cplx *r = (cplx *)malloc(n * sizeof(cplx));
    cplx *p = (cplx *)malloc(n * sizeof(cplx));
    cplx *q = (cplx *)malloc(n * sizeof(cplx));
    cplx *ps = (cplx *)malloc(n * (size_t)nshift * sizeof(cplx));
    double *sc = (double *)malloc((size_t)nshift * 5 * sizeof(double));
    int *active = (int *)malloc((size_t)nshift * sizeof(int));
    if (!r || !p || !q || !ps || !sc || !active) {
        free(r); free(p); free(q); free(ps); free(sc); free(active);
        return -1;
    }
    double *delta = sc, *zeta = sc + nshift, *zeta_old = sc + 2 * nshift,
           *zeta_new = sc + 3 * nshift, *alpha_i = sc + 4 * nshift;
    int rc = 1, k = 0;

    for (size_t j = 0; j < n; ++j) { r[j] = b[j]; p[j] = b[j]; }
    for (int i = 0; i < nshift; ++i) {
        delta[i] = sigma[i] - sigma_min;
        zeta[i] = zeta_old[i] = 1.0;
        active[i] = 1;
        if (conv_iter) conv_iter[i] = 0;
        for (size_t j = 0; j < n; ++j) { x[(size_t)i * n + j] = 0.0; ps[(size_t)i * n + j] = b[j]; }
    }
    double alpha_prev = 1.0, beta_prev = 0.0;
    double rho = re_dot(b, b, n);
    double bnorm = sqrt(rho);
    if (bnorm == 0.0) { rc = 0; goto done; }

    for (k = 0; k < max_iter; ++k) {
        if (oracle_mdagm_bf(N, antiperiodic_t, U, theta, mass, sigma_min, p, q)) { rc = -1; goto done; }
        double alpha = rho / re_dot(p, q, n);
        for (int i = 0; i < nshift; ++i) {
            zeta_new[i] = zeta[i] * zeta_old[i] * alpha_prev /
                          (alpha * beta_prev * (zeta_old[i] - zeta[i]) +
                           zeta_old[i] * alpha_prev * (1.0 + delta[i] * alpha));
            alpha_i[i] = alpha * zeta_new[i] / zeta[i];
            if (active[i])
                for (size_t j = 0; j < n; ++j) x[(size_t)i * n + j] += alpha_i[i] * ps[(size_t)i * n + j];
        }
        for (size_t j = 0; j < n; ++j) r[j] -= alpha * q[j];
        double rho_new = re_dot(r, r, n);
        double beta = rho_new / rho;
        for (size_t j = 0; j < n; ++j) p[j] = r[j] + beta * p[j];
        for (int i = 0; i < nshift; ++i) {
            double ratio = zeta_new[i] / zeta[i];
            double beta_i = beta * ratio * ratio;
            if (active[i])
                for (size_t j = 0; j < n; ++j)
                    ps[(size_t)i * n + j] = zeta_new[i] * r[j] + beta_i * ps[(size_t)i * n + j];
        }
        if (k < hist_len) {
            if (hist_alpha) hist_alpha[k] = alpha;
            if (hist_beta) hist_beta[k] = beta;
            if (hist_rnorm) hist_rnorm[k] = sqrt(rho_new);
        }
        int n_active = 0;
        for (int i = 0; i < nshift; ++i) {
            zeta_old[i] = zeta[i];
            zeta[i] = zeta_new[i];
            if (active[i]) {
                if (fabs(zeta[i]) * sqrt(rho_new) > tol * bnorm) ++n_active;
                else { active[i] = 0; if (conv_iter) conv_iter[i] = k + 1; }
            }
        }
        alpha_prev = alpha; beta_prev = beta; rho = rho_new;
        if (n_active == 0) { ++k; rc = 0; break; }
    }
done:
    if (iters) *iters = k;
    for (int i = 0; i < nshift; ++i) {
        if (conv_iter && active[i]) conv_iter[i] = k;
        if (zeta_out) zeta_out[i] = zeta[i];
        if (true_relres) {
            if (bnorm == 0.0 || rc < 0) true_relres[i] = 0.0;
            else {
                oracle_mdagm_bf(N, antiperiodic_t, U, theta, mass, sigma[i], x + (size_t)i * n, q);
                for (size_t j = 0; j < n; ++j) q[j] = b[j] - q[j];
                true_relres[i] = sqrt(re_dot(q, q, n)) / bnorm;
            }
        }
    }
    if (r_out) memcpy(r_out, r, n * sizeof(cplx));
    free(r); free(p); free(q); free(ps); free(sc); free(active);
    return rc;
}

int oracle_cg_multishift(const int N[4], int antiperiodic_t, const cplx *U, double mass,
                         int nshift, const double *sigma, const cplx *b, cplx *x,
                         double tol, int max_iter,
                         int *iters, int *conv_iter, double *true_relres,
                         double *zeta_out, cplx *r_out,
                         double *hist_alpha, double *hist_beta, double *hist_rnorm, int hist_len)
{
    return oracle_cg_multishift_bf(N, antiperiodic_t, U, NULL, mass, nshift, sigma, b, x, tol, max_iter, iters,
                                   conv_iter, true_relres, zeta_out, r_out, hist_alpha, hist_beta, hist_rnorm, hist_len);
}

/* ---------------------------------------------------------------------------------------
 * Rational function of A = m^2 - D_eo D_oe applied to a vector:
 *
 *   y = c0 b + sum_{i=1..r} c_i x_i ,     (A + sigma_i) x_i = b                      (Eq. 6)
 *
 * PAPER.md:133 "the algebraic matrix function appearing in Eq. (3) is approximated to machine
 * precision by a rational function" whose poles are the sigma_i of Eq. 6;
 * this partial-fraction sum is what the pseudofermion heatbath and the action evaluation
 * (Algorithm 1 steps 3 and 6: "function calls to the multishift inverter")
 * do with the solutions.  The paper prints neither c_i nor sigma_i: both are inputs.
 * Written as the definition: solve with the multi-shift CG above, then add the r+1 terms in
 * the order of the formula.  (The CUDA path accumulates y inside its vector-update kernel
 * and never stores x_i; that is a reordering of this sum, not a different quantity.)
 * Pins: dense (c0 + sum c_i (A+sigma_i)^-1) b by numpy.linalg.solve; the partial-fraction
 * identity 1/((A+s1)(A+s2)) = [1/(A+s1) - 1/(A+s2)]/(s2-s1) checked by applying both factors;
 * free-field plane wave b: y = (c0 + sum c_i/(lambda+sigma_i)) b.
 * Returns as oracle_cg_multishift.
 * ------------------------------------------------------------------------------------- */
int oracle_rational_apply(const int N[4], int antiperiodic_t, const cplx *U, double mass,
                          int nshift, const double *sigma, double c0, const double *c,
                          const cplx *b, cplx *y, double tol, int max_iter,
                          int *iters, int *conv_iter)
{
    size_t n = vol(N) / 2 * 3;
    cplx *x = (cplx *)malloc(n * (size_t)(nshift > 0 ? nshift : 1) * sizeof(cplx));
    if (!x) return -1;
    int rc = oracle_cg_multishift(N, antiperiodic_t, U, mass, nshift, sigma, b, x, tol, max_iter,
                                  iters, conv_iter, NULL, NULL, NULL, NULL, NULL, NULL, 0);
    if (rc >= 0) {
        for (size_t j = 0; j < n; ++j) y[j] = c0 * b[j];
        for (int i = 0; i < nshift; ++i)
            for (size_t j = 0; j < n; ++j) y[j] += c[i] * x[(size_t)i * n + j];
    }
    free(x);
    return rc;
}

/* ---------------------------------------------------------------------------------------
 * Fermion-force outer products ("the fermion force
 * calculation step ... a large fraction of the execution time is spent in ... deo and doe").
 * The paper gives no formula (it follows its ref. 33); reading R21 of DESIGN.md derives it:
 *
 *   S = phi^dagger r(A) phi,  r(A) = c0 + sum_i c_i (A + sigma_i)^-1,  A = m^2 - D_eo D_oe  (Eq. 3, 6, 8)
 *   x_i = (A + sigma_i)^-1 phi (even sites),  y_i = D_oe x_i (odd sites),
 *   w_i = x_i on even sites, y_i on odd sites.
 *   Under U_mu(x) -> exp(i eps T) U_mu(x)  (T Hermitian traceless):
 *       dS/d eps = 2 Re Tr[ i T F_mu(x) ],
 *   F_mu(x) = TA[ U_mu(x) Q_mu(x) ],
 *   Q_mu(x) = 1/2 eta_mu(x) s+_mu(x) (-1)^{p(x)} sum_i c_i  w_i(x+mu) w_i(x)^dagger      (3x3 outer product)
 *   TA[M]   = (M - M^dagger)/2 - Tr(M - M^dagger)/6                     (traceless anti-Hermitian part)
 * (both places where U_mu(x) enters D -- the forward hop out of x and the backward hop out of
 * x+mu -- are included; they are complex conjugates of each other, hence the "2 Re").
 * Pin: central finite differences of S computed with DENSE numpy solves, for random links,
 * directions and generators, both parities, across the antiperiodic boundary, and N_mu = 2.
 *
 * x: nshift even half vectors, contiguous.  F: [V][4][3][3], row-major.  Returns 0, or -1.
 * ------------------------------------------------------------------------------------- */
/* With the optional backfield theta (NULL: none; reading R6): the links of D are e^{i theta} U, a left
 * multiplication exp(i eps T) U commutes with the phase, so F_mu(x) = TA[ e^{i theta_mu(x)} U_mu(x) Q_mu(x) ] with the
 * y_i = D_oe x_i of the phased operator. */
int oracle_fermion_force_bf(const int N[4], int antiperiodic_t, const cplx *U, const double *theta, int nshift,
                            const double *c, const cplx *x, cplx *F)
{
    size_t V = vol(N), nh = V / 2 * 3;
    cplx *w = (cplx *)malloc(V * 3 * (size_t)nshift * sizeof(cplx));
    cplx *y = (cplx *)malloc(nh * sizeof(cplx));
    cplx *full = (cplx *)malloc(V * 3 * sizeof(cplx));
    if (!w || !y || !full) { free(w); free(y); free(full); return -1; }
    for (int i = 0; i < nshift; ++i) {
        cplx *wi = w + (size_t)i * V * 3;
        if (oracle_dslash_half_bf(N, antiperiodic_t, U, theta, 1, x + (size_t)i * nh, y)) { free(w); free(y); free(full); return -1; }
        oracle_half_to_full(N, 0, x + (size_t)i * nh, wi);        /* even sites: x_i, odd: 0 */
        oracle_half_to_full(N, 1, y, full);                        /* odd sites: y_i, even: 0 */
        for (size_t j = 0; j < V * 3; ++j) wi[j] += full[j];
    }
    for (size_t lex = 0; lex < V; ++lex) {
        int xc[4];
        coords_of(N, lex, xc);
        double sp = parity_of(xc) ? -1.0 : 1.0;
        for (int mu = 0; mu < 4; ++mu) {
            int xf[4] = { xc[0], xc[1], xc[2], xc[3] };
            xf[mu] = (xc[mu] + 1) % N[mu];
            size_t lf = lex_of(N, xf);
            double e = 0.5 * eta(mu, xc) * sp;
            if (antiperiodic_t && mu == 3 && xc[3] == N[3] - 1) e = -e;
            cplx Q[3][3], M[3][3];
            for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) Q[a][b] = 0.0;
            for (int i = 0; i < nshift; ++i) {
                const cplx *wi = w + (size_t)i * V * 3;
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b) Q[a][b] += c[i] * wi[lf * 3 + a] * conj(wi[lex * 3 + b]);
            }
            const cplx *u = U + (lex * 4 + (size_t)mu) * 9;
            const cplx ph = theta ? cexp(I * theta[lex * 4 + (size_t)mu]) : 1.0;
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b) {
                    cplx t = 0.0;
                    for (int k = 0; k < 3; ++k) t += u[a * 3 + k] * (e * Q[k][b]);
                    M[a][b] = theta ? ph * t : t;
                }
            cplx tr = 0.0;
            for (int a = 0; a < 3; ++a) tr += M[a][a] - conj(M[a][a]);
            cplx *f = F + (lex * 4 + (size_t)mu) * 9;
            for (int a = 0; a < 3; ++a)
                for (int b = 0; b < 3; ++b)
                    f[a * 3 + b] = 0.5 * (M[a][b] - conj(M[b][a])) - (a == b ? tr / 6.0 : 0.0);
        }
    }
    free(w); free(y); free(full);
    return 0;
}

int oracle_fermion_force(const int N[4], int antiperiodic_t, const cplx *U, int nshift,
                         const double *c, const cplx *x, cplx *F)
{
    return oracle_fermion_force_bf(N, antiperiodic_t, U, NULL, nshift, c, x, F);
}

/* ---------------------------------------------------------------------------------------
 * Gauge staples of the tree-level Symanzik improved action.
 * PAPER.md:105 names the action; PAPER.md:365 says the staples are "products of 3 and 5 SU(3)
 * matrices representing links on C-shaped paths" (Listing 3, shows only the loop
 * nest).  The paths and coefficients are not printed; reading R22 of DESIGN.md:
 *
 *   W[U] = sum_x sum_{mu<nu} { c0 Re Tr P_{mu nu}(x) + c1 [ Re Tr R_{mu nu}(x) + Re Tr R_{nu mu}(x) ] },
 *   c0 = 5/3, c1 = -1/12   (S_g = -(beta/3) W; P the 1x1 plaquette, R_{mu nu} the 2x1 rectangle, 2 along mu)
 *   staple S_mu(x) = sum over the loops of W through U_mu(x) of coefficient x (the remaining links,
 *   ordered from x+mu back to x), so that  W = ... + Re Tr[ U_mu(x) S_mu(x) ] + (terms without U_mu(x)).
 *
 * Per nu != mu that is 2 three-link paths (plaquette, above and below) and 6 five-link paths
 * (the link as first or second long side of a 2x1 rectangle, or as the short side of a 1x2 one;
 * each above and below).  A path is walked from x+mu: a step +d from y multiplies by U_d(y),
 * a step -d by U_d(y-d)^dagger.  Gauge links are periodic in all directions (no fermion phases).
 * Pins: the finite-difference derivative of W (computed by an independent numpy routine),
 * sum_{x,mu} Re Tr[U S] = 4 c0 sum P + 6 c1 sum R, unit links, gauge covariance.
 * ------------------------------------------------------------------------------------- */
static void mat_mul(const cplx *a, const cplx *b, cplx *o)
{
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            cplx t = 0.0;
            for (int k = 0; k < 3; ++k) t += a[i * 3 + k] * b[k * 3 + j];
            o[i * 3 + j] = t;
        }
}

/* out += coef * (product of the links along `steps` starting at site y); step = +-(d+1) */
static void add_path(const int N[4], const cplx *U, const int start[4], const int *steps, int nsteps,
                     double coef, cplx *out)
{
    cplx M[9] = { 1, 0, 0, 0, 1, 0, 0, 0, 1 }, L[9], T[9];
    int y[4] = { start[0], start[1], start[2], start[3] };
    for (int s = 0; s < nsteps; ++s) {
        int d = abs(steps[s]) - 1;
        if (steps[s] > 0) {
            const cplx *u = U + (lex_of(N, y) * 4 + (size_t)d) * 9;
            for (int k = 0; k < 9; ++k) L[k] = u[k];
            y[d] = (y[d] + 1) % N[d];
        } else {
            y[d] = (y[d] + N[d] - 1) % N[d];
            const cplx *u = U + (lex_of(N, y) * 4 + (size_t)d) * 9;
            for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) L[i * 3 + j] = conj(u[j * 3 + i]);
        }
        mat_mul(M, L, T);
        memcpy(M, T, sizeof(M));
    }
    for (int k = 0; k < 9; ++k) out[k] += coef * M[k];
}

/* S: [V][4][3][3].  c0, c1 are arguments so that tests can look at the two families separately. */
void oracle_gauge_staples(const int N[4], const cplx *U, double c0, double c1, cplx *S)
{
    size_t V = vol(N);
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (long long l = 0; l < (long long)V; ++l) {
        int x[4];
        coords_of(N, (size_t)l, x);
        for (int mu = 0; mu < 4; ++mu) {
            cplx *out = S + ((size_t)l * 4 + (size_t)mu) * 9;
            for (int k = 0; k < 9; ++k) out[k] = 0.0;
            int xm[4] = { x[0], x[1], x[2], x[3] };
            xm[mu] = (x[mu] + 1) % N[mu];
            int m = mu + 1;
            for (int nu = 0; nu < 4; ++nu) {
                if (nu == mu) continue;
                int n = nu + 1;
                const int pl_up[3] = { n, -m, -n }, pl_dn[3] = { -n, -m, n };
                const int ra_up[5] = { m, n, -m, -m, -n }, ra_dn[5] = { m, -n, -m, -m, n };
                const int rb_up[5] = { n, -m, -m, -n, m }, rb_dn[5] = { -n, -m, -m, n, m };
                const int rc_up[5] = { n, n, -m, -n, -n }, rc_dn[5] = { -n, -n, -m, n, n };
                add_path(N, U, xm, pl_up, 3, c0, out);
                add_path(N, U, xm, pl_dn, 3, c0, out);
                add_path(N, U, xm, ra_up, 5, c1, out);
                add_path(N, U, xm, ra_dn, 5, c1, out);
                add_path(N, U, xm, rb_up, 5, c1, out);
                add_path(N, U, xm, rb_dn, 5, c1, out);
                add_path(N, U, xm, rc_up, 5, c1, out);
                add_path(N, U, xm, rc_dn, 5, c1, out);
            }
        }
    }
}

/* Number of OpenMP threads the site loop uses (for bench.py's "cores" field). */
#ifdef _OPENMP
#include <omp.h>
int oracle_num_threads(void) { return omp_get_max_threads(); }
void oracle_set_num_threads(int n) { if (n > 0) omp_set_num_threads(n); }
#else
int oracle_num_threads(void) { return 1; }
void oracle_set_num_threads(int n) { (void)n; }
#endif

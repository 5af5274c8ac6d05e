/*
 * lqcd_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of what the hot path of arXiv 1311.2719
 * computes: the staggered and Wilson hopping terms ("fmv"/"fmtv", PAPER.md:48,
 * :83-88), the normal operator the conjugate gradient inverts, and the conjugate
 * gradient itself (subroutine congrad).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call it.  It shares no code, header, table or constant with the CUDA library
 * under paper_1311_2719_b200/csrc/.
 *
 * The paper's section-3 listing (the operator) is missing from the extraction
 * (PAPER.md:46-48 jumps from "Below we list the differences" to the discussion
 * of present(u,ud,v,w,iup,idn)), so the operators are the textbook definitions
 * fixed in SURVEY.md section 8(c.2)/(c.3) and DESIGN.md "Readings"; each function
 * below cites the passage it follows.  Pins (tests/test_oracle_pins.py): free
 * field spectra in closed form, anti-hermiticity, hermiticity and positivity of
 * M^+M, gauge covariance, gamma5-hermiticity, dense inversion on 2^4, table
 * permutation properties.  Unpinned by anything but declaration: the choice among
 * equivalent eta-phase conventions, the sign convention of the gamma matrices and
 * the even-first site ordering ("parity unpinned" for those choices only).
 *
 * Layouts (little-endian fp64, complex = (re,im) adjacent):
 *   site index   g = parity*Vh + e, e = floor(s/2), s = x0 + L0*(x1 + L1*(x2 + L2*x3)),
 *                parity = (x0+x1+x2+x3) mod 2  (even block first: the paper's l=1..mvd2)
 *   gauge        u[g][mu][row][col]          U_mu(x) stored at the site it leaves from
 *   staggered    v[c][e]  c=0..2             (the paper's p(l,ic)), one parity
 *   Wilson       v[spin][c][g]               full lattice
 *   tables       iup[mu][g], idn[mu][g]      g-index of x+mu, x-mu (periodic wrap, no signs)
 *
 * No blocking, fusion or reordering beyond the definitions: every output site
 * sums mu = 0..3, forward hop then backward hop.  OpenMP only distributes output
 * sites (and the fixed blocks of the dot product) over threads; results do not
 * depend on the thread count.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cd;

enum { ORACLE_STAGGERED = 0, ORACLE_WILSON = 1 };

typedef struct {
    int L[4];
    long V, Vh;
} geom_t;

static int geom_init(geom_t *G, const int *L)
{
    G->V = 1;
    for (int mu = 0; mu < 4; ++mu) {
        if (L[mu] < 2 || (L[mu] & 1)) return -1; /* A16: odd extents are an error */
        G->L[mu] = L[mu];
        G->V *= L[mu];
    }
    G->Vh = G->V / 2;
    return 0;
}

/* (parity, e) -> coordinates.  SURVEY 8(c.1). */
static void site_coords(const geom_t *G, int parity, long e, int x[4])
{
    const long L0 = G->L[0], L1 = G->L[1], L2 = G->L[2];
    long s = 2 * e;
    x[1] = (int)((s / L0) % L1);
    x[2] = (int)((s / (L0 * L1)) % L2);
    x[3] = (int)(s / (L0 * L1 * L2));
    x[0] = (int)(s % L0) + ((x[1] + x[2] + x[3] + parity) & 1);
}

/* coordinates -> g.  SURVEY 8(b). */
static long site_index(const geom_t *G, const int x[4])
{
    long s = x[0] + (long)G->L[0] * (x[1] + (long)G->L[1] * (x[2] + (long)G->L[2] * x[3]));
    int parity = (x[0] + x[1] + x[2] + x[3]) & 1;
    return parity * G->Vh + s / 2;
}

/* g-index of x + dir*mu_hat with periodic wrap in every direction. */
static long neighbour(const geom_t *G, const int x[4], int mu, int dir)
{
    int y[4] = { x[0], x[1], x[2], x[3] };
    y[mu] = (x[mu] + dir + G->L[mu]) % G->L[mu];
    return site_index(G, y);
}

/* Antiperiodic time boundary (BASELINE.json configs; reading A4): a hop that
 * crosses x3 = L3-1 <-> 0 carries a minus sign, in both directions. */
static double bc_forward(const geom_t *G, const int x[4], int mu)
{
    return (mu == 3 && x[3] == G->L[3] - 1) ? -1.0 : 1.0;
}
static double bc_backward(const geom_t *G, const int x[4], int mu)
{
    return (mu == 3 && x[3] == 0) ? -1.0 : 1.0;
}

/* Staggered phases eta_mu(x) (reading A3): eta_0 = 1, eta_1 = (-1)^x0,
 * eta_2 = (-1)^(x0+x1), eta_3 = (-1)^(x0+x1+x2). */
static double eta_phase(const int x[4], int mu)
{
    int s = 0;
    for (int nu = 0; nu < mu; ++nu) s += x[nu];
    return (s & 1) ? -1.0 : 1.0;
}

/* ------------------------------------------------------------------ tables */

/* iup/idn/lex2eo of SURVEY 8(b) (the paper's iup, idn: PAPER.md:48, :64). */
int oracle_tables(const int *L, int32_t *iup, int32_t *idn, int32_t *lex2eo)
{
    geom_t G;
    if (geom_init(&G, L)) return -1;
    for (int parity = 0; parity < 2; ++parity)
        for (long e = 0; e < G.Vh; ++e) {
            int x[4];
            site_coords(&G, parity, e, x);
            long g = parity * G.Vh + e;
            for (int mu = 0; mu < 4; ++mu) {
                iup[mu * G.V + g] = (int32_t)neighbour(&G, x, mu, +1);
                idn[mu * G.V + g] = (int32_t)neighbour(&G, x, mu, -1);
            }
            long s = x[0] + (long)G.L[0] * (x[1] + (long)G.L[1] * (x[2] + (long)G.L[2] * x[3]));
            lex2eo[s] = (int32_t)g;
        }
    return 0;
}

/* coordinates of site g, for the tests' own plane waves and gauge transformations */
int oracle_coords(const int *L, int32_t *x_out /* [V][4] */)
{
    geom_t G;
    if (geom_init(&G, L)) return -1;
    for (int parity = 0; parity < 2; ++parity)
        for (long e = 0; e < G.Vh; ++e) {
            int x[4];
            site_coords(&G, parity, e, x);
            long g = parity * G.Vh + e;
            for (int mu = 0; mu < 4; ++mu) x_out[g * 4 + mu] = x[mu];
        }
    return 0;
}

/* ------------------------------------------------------- staggered operator */

/* One output site of the staggered hopping term, SURVEY 8(c.2):
 *   (D chi)(x) = 1/2 sum_mu eta_mu(x) [ b+_mu(x) U_mu(x) chi(x+mu) - b-_mu(x) U_mu(x-mu)^+ chi(x-mu) ]
 * x has parity `parity`; `in` lives on the opposite parity, layout in[c][e]. */
static void stag_site(const geom_t *G, const cd *u, int parity, long e, const cd *in, cd out[3])
{
    int x[4];
    site_coords(G, parity, e, x);
    const long g = parity * G->Vh + e;
    const long other = (1 - parity) * G->Vh;
    cd acc[3] = { 0, 0, 0 };
    for (int mu = 0; mu < 4; ++mu) {
        const double eta = eta_phase(x, mu);
        /* forward hop: U_mu(x) chi(x+mu) */
        {
            const long ef = neighbour(G, x, mu, +1) - other;
            const cd *U = u + (g * 4 + mu) * 9;
            const double sgn = eta * bc_forward(G, x, mu);
            for (int a = 0; a < 3; ++a) {
                cd s = 0;
                for (int b = 0; b < 3; ++b) s += U[a * 3 + b] * in[b * G->Vh + ef];
                acc[a] += sgn * s;
            }
        }
        /* backward hop: U_mu(x-mu)^+ chi(x-mu) */
        {
            const long gb = neighbour(G, x, mu, -1);
            const long eb = gb - other;
            const cd *W = u + (gb * 4 + mu) * 9;
            const double sgn = eta * bc_backward(G, x, mu);
            for (int a = 0; a < 3; ++a) {
                cd s = 0;
                for (int b = 0; b < 3; ++b) s += conj(W[b * 3 + a]) * in[b * G->Vh + eb];
                acc[a] -= sgn * s;
            }
        }
    }
    for (int a = 0; a < 3; ++a) out[a] = 0.5 * acc[a];
}

static void stag_dslash(const geom_t *G, const cd *u, int out_parity, const cd *in, cd *out)
{
#pragma omp parallel for schedule(static)
    for (long e = 0; e < G->Vh; ++e) {
        cd r[3];
        stag_site(G, u, out_parity, e, in, r);
        for (int a = 0; a < 3; ++a) out[a * G->Vh + e] = r[a];
    }
}

/* --------------------------------------------------------- Wilson operator */

/* DeGrand-Rossi basis; rows top to bottom.  Hermitian,
 * {gamma_mu, gamma_nu} = 2 delta, gamma5 = g0 g1 g2 g3 = diag(1,1,-1,-1). */
static const cd GAMMA[4][4][4] = {
    { { 0, 0, 0, I }, { 0, 0, I, 0 }, { 0, -I, 0, 0 }, { -I, 0, 0, 0 } },
    { { 0, 0, 0, -1 }, { 0, 0, 1, 0 }, { 0, 1, 0, 0 }, { -1, 0, 0, 0 } },
    { { 0, 0, I, 0 }, { 0, 0, 0, -I }, { -I, 0, 0, 0 }, { 0, I, 0, 0 } },
    { { 0, 0, 1, 0 }, { 0, 0, 0, 1 }, { 1, 0, 0, 0 }, { 0, 1, 0, 0 } },
};
static const double GAMMA5[4] = { 1.0, 1.0, -1.0, -1.0 };

/* One output site of the Wilson hopping term, SURVEY 8(a) row W1 / 8(c.3):
 *   (D_W psi)(x) = sum_mu [ (1-gamma_mu) b+ U_mu(x) psi(x+mu) + (1+gamma_mu) b- U_mu(x-mu)^+ psi(x-mu) ]
 * full-lattice layout in[spin][c][g]. */
static void wilson_site(const geom_t *G, const cd *u, int parity, long e, const cd *in, cd out[4][3])
{
    int x[4];
    site_coords(G, parity, e, x);
    const long g = parity * G->Vh + e;
    const long V = G->V;
    cd acc[4][3];
    memset(acc, 0, sizeof acc);
    for (int mu = 0; mu < 4; ++mu) {
        cd h[4][3];
        /* forward */
        {
            const long gf = neighbour(G, x, mu, +1);
            const cd *U = u + (g * 4 + mu) * 9;
            const double sgn = bc_forward(G, x, mu);
            for (int s = 0; s < 4; ++s)
                for (int a = 0; a < 3; ++a) {
                    cd t = 0;
                    for (int b = 0; b < 3; ++b) t += U[a * 3 + b] * in[(s * 3 + b) * V + gf];
                    h[s][a] = t;
                }
            for (int s = 0; s < 4; ++s)
                for (int a = 0; a < 3; ++a) {
                    cd t = h[s][a];
                    for (int sp = 0; sp < 4; ++sp) t -= GAMMA[mu][s][sp] * h[sp][a];
                    acc[s][a] += sgn * t;
                }
        }
        /* backward */
        {
            const long gb = neighbour(G, x, mu, -1);
            const cd *W = u + (gb * 4 + mu) * 9;
            const double sgn = bc_backward(G, x, mu);
            for (int s = 0; s < 4; ++s)
                for (int a = 0; a < 3; ++a) {
                    cd t = 0;
                    for (int b = 0; b < 3; ++b) t += conj(W[b * 3 + a]) * in[(s * 3 + b) * V + gb];
                    h[s][a] = t;
                }
            for (int s = 0; s < 4; ++s)
                for (int a = 0; a < 3; ++a) {
                    cd t = h[s][a];
                    for (int sp = 0; sp < 4; ++sp) t += GAMMA[mu][s][sp] * h[sp][a];
                    acc[s][a] += sgn * t;
                }
        }
    }
    for (int s = 0; s < 4; ++s)
        for (int a = 0; a < 3; ++a) out[s][a] = acc[s][a];
}

/* writes the out_parity half of `out`, reads the other half of `in` */
static void wilson_dslash(const geom_t *G, const cd *u, int out_parity, const cd *in, cd *out)
{
#pragma omp parallel for schedule(static)
    for (long e = 0; e < G->Vh; ++e) {
        cd r[4][3];
        wilson_site(G, u, out_parity, e, in, r);
        const long g = out_parity * G->Vh + e;
        for (int s = 0; s < 4; ++s)
            for (int a = 0; a < 3; ++a) out[(s * 3 + a) * G->V + g] = r[s][a];
    }
}

/* M psi = psi - kappa D_W psi on the full lattice (row W2). */
static void wilson_M(const geom_t *G, const cd *u, double kappa, const cd *in, cd *out)
{
    wilson_dslash(G, u, 0, in, out);
    wilson_dslash(G, u, 1, in, out);
    const long n = 12 * G->V;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; ++i) out[i] = in[i] - kappa * out[i];
}

static void gamma5_mul(const geom_t *G, const cd *in, cd *out)
{
    const long V = G->V;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < 12 * V; ++i) out[i] = GAMMA5[i / (3 * V)] * in[i];
}

/* ------------------------------------------------------- the CG's operator */

typedef struct {
    geom_t G;
    const cd *u;
    int fermion;
    double param; /* mass (staggered) or kappa (Wilson) */
    long n;       /* complex length of a CG vector */
    cd *t1, *t2, *t3; /* scratch */
} op_t;

/* internal operator type: Schur complement of the Wilson matrix on the even sites (8(f) row 4) */
#define ORACLE_WILSON_EO 2

static int op_init(op_t *op, const int *L, int fermion, const cd *u, double param)
{
    if (geom_init(&op->G, L)) return -1;
    if (fermion != ORACLE_STAGGERED && fermion != ORACLE_WILSON && fermion != ORACLE_WILSON_EO) return -2;
    op->u = u;
    op->fermion = fermion;
    op->param = param;
    op->n = fermion == ORACLE_STAGGERED ? 3 * op->G.Vh : 12 * op->G.V;
    op->t1 = malloc(sizeof(cd) * op->n);
    op->t2 = malloc(sizeof(cd) * op->n);
    op->t3 = malloc(sizeof(cd) * op->n);
    return (op->t1 && op->t2 && op->t3) ? 0 : -3;
}
static void op_free(op_t *op)
{
    free(op->t1);
    free(op->t2);
    free(op->t3);
}

/* Even-odd (Schur) preconditioned Wilson matrix, SURVEY 8(f) row 4.  In even/odd blocks
 * M = 1 - kappa D_W = [[1, -kappa D_eo], [-kappa D_oe, 1]], whose Schur complement on the even
 * sites is  Mhat = 1 - kappa^2 D_eo D_oe.  Vectors are full-lattice arrays of which only the even
 * half (g < Vh) carries data: out_e = in_e - kappa^2 D_eo D_oe in_e, out_o = 0. */
static void wilson_Mhat(const geom_t *G, const cd *u, double kappa, const cd *in, cd *out, cd *scratch)
{
    wilson_dslash(G, u, 1, in, scratch); /* scratch_o = D_oe in_e */
    wilson_dslash(G, u, 0, scratch, out); /* out_e = D_eo scratch_o */
    const long V = G->V, Vh = G->Vh;
#pragma omp parallel for schedule(static)
    for (long e = 0; e < Vh; ++e)
        for (int k = 0; k < 12; ++k) {
            out[k * V + e] = in[k * V + e] - kappa * kappa * out[k * V + e];
            out[k * V + Vh + e] = 0;
        }
}

/* A = (M^+ M)_ee = m^2 - D_eo D_oe on even-site vectors (staggered);
 * A = M^+ M = gamma5 M gamma5 M on the full lattice (Wilson, 8(c.3)). */
static void apply_A(const op_t *op, const cd *in, cd *out)
{
    const geom_t *G = &op->G;
    if (op->fermion == ORACLE_STAGGERED) {
        const double m2 = op->param * op->param;
        stag_dslash(G, op->u, 1, in, op->t1);      /* t1_o = D_oe in_e */
        stag_dslash(G, op->u, 0, op->t1, op->t2);  /* t2_e = D_eo t1_o */
#pragma omp parallel for schedule(static)
        for (long i = 0; i < op->n; ++i) out[i] = m2 * in[i] - op->t2[i];
    } else if (op->fermion == ORACLE_WILSON) {
        wilson_M(G, op->u, op->param, in, op->t1);
        gamma5_mul(G, op->t1, op->t2);
        wilson_M(G, op->u, op->param, op->t2, op->t1);
        gamma5_mul(G, op->t1, out);
    } else { /* ORACLE_WILSON_EO: Mhat^+ Mhat = gamma5 Mhat gamma5 Mhat (gamma5 is site-diagonal) */
        wilson_Mhat(G, op->u, op->param, in, op->t1, op->t3);
        gamma5_mul(G, op->t1, op->t2);
        wilson_Mhat(G, op->u, op->param, op->t2, op->t1, op->t3);
        gamma5_mul(G, op->t1, out);
    }
}

/* Re<a,b> = Re sum conj(a_i) b_i (reading A9: only real parts are used), summed
 * in fixed blocks so the value does not depend on the thread count. */
#define DOT_BLOCK 4096
static double dot_re(const cd *a, const cd *b, long n)
{
    const long nb = (n + DOT_BLOCK - 1) / DOT_BLOCK;
    double *part = malloc(sizeof(double) * (nb > 0 ? nb : 1));
#pragma omp parallel for schedule(static)
    for (long k = 0; k < nb; ++k) {
        const long lo = k * DOT_BLOCK, hi = lo + DOT_BLOCK < n ? lo + DOT_BLOCK : n;
        double s = 0.0;
        for (long i = lo; i < hi; ++i) s += creal(a[i]) * creal(b[i]) + cimag(a[i]) * cimag(b[i]);
        part[k] = s;
    }
    double s = 0.0;
    for (long k = 0; k < nb; ++k) s += part[k];
    free(part);
    return s;
}

/* ------------------------------------------------------------ entry points */

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* Bare hopping term, no mass/kappa (SURVEY 8(b) lqcd_dslash).  Staggered: in/out
 * are half-lattice vectors [3][Vh]; Wilson: full-lattice vectors [4][3][V], only
 * the out_parity half of `out` is written. */
int oracle_dslash(const int *L, int fermion, const double *u, int out_parity, const double *in, double *out)
{
    geom_t G;
    if (geom_init(&G, L)) return -1;
    if (out_parity != 0 && out_parity != 1) return -2;
    if (fermion == ORACLE_STAGGERED)
        stag_dslash(&G, (const cd *)u, out_parity, (const cd *)in, (cd *)out);
    else if (fermion == ORACLE_WILSON)
        wilson_dslash(&G, (const cd *)u, out_parity, (const cd *)in, (cd *)out);
    else
        return -2;
    return 0;
}

/* The same, for a list of output sites only: out[k][component] for e = e_list[k].
 * Lets the full-size GPU tests check sampled outputs one by one. */
int oracle_dslash_sites(const int *L, int fermion, const double *u, int out_parity, const double *in, long nsites,
                        const int64_t *e_list, double *out)
{
    geom_t G;
    if (geom_init(&G, L)) return -1;
    if (out_parity != 0 && out_parity != 1) return -2;
    cd *o = (cd *)out;
    for (long k = 0; k < nsites; ++k) {
        if (e_list[k] < 0 || e_list[k] >= G.Vh) return -2;
        if (fermion == ORACLE_STAGGERED)
            stag_site(&G, (const cd *)u, out_parity, e_list[k], (const cd *)in, o + 3 * k);
        else
            wilson_site(&G, (const cd *)u, out_parity, e_list[k], (const cd *)in, (cd(*)[3])(o + 12 * k));
    }
    return 0;
}

int oracle_wilson_M(const int *L, const double *u, double kappa, const double *in, double *out)
{
    geom_t G;
    if (geom_init(&G, L)) return -1;
    wilson_M(&G, (const cd *)u, kappa, (const cd *)in, (cd *)out);
    return 0;
}

int oracle_apply_MdagM(const int *L, int fermion, const double *u, double param, const double *in, double *out)
{
    op_t op;
    int rc = op_init(&op, L, fermion, (const cd *)u, param);
    if (rc) return rc;
    apply_A(&op, (const cd *)in, (cd *)out);
    op_free(&op);
    return 0;
}

double oracle_dot_re(const double *a, const double *b, long n_complex)
{
    return dot_re((const cd *)a, (const cd *)b, n_complex);
}

/* Conjugate gradient on A x = b, following PAPER.md:68-96 line by
 * line: x=0, p=r=b, betan=<r,r> (:68-74); exit test on <r,r> (:75-76, :91-93;
 * relative form, reading A6); alpha = <r,r>/<p,Ap> (:85; plain dot product here);
 * x += alpha p (:86); r -= alpha Ap (:89); beta = betan/betad (:96);
 * p = r + beta p (missing from the truncated listing; reading A7).
 * Returns 0 = converged, 1 = maxiter reached (outputs valid), <0 = error.
 * rr_hist, if not NULL, receives <r,r> after k iterations at index k (0..iters). */
static int cg_core(op_t *opp, double tol, int maxiter, const double *b_, double *x_, int *iters, double *true_res,
                   double *rr_hist)
{
#define op (*opp)
    const long n = op.n;
    const cd *b = (const cd *)b_;
    cd *x = (cd *)x_;
    cd *r = malloc(sizeof(cd) * n), *p = malloc(sizeof(cd) * n), *Ap = malloc(sizeof(cd) * n);
    if (!r || !p || !Ap) return -3;

    for (long i = 0; i < n; ++i) {
        x[i] = 0;
        r[i] = b[i];
        p[i] = b[i];
    }
    double rr = dot_re(r, r, n);
    const double bb = rr;
    int status = 1, k = 0;
    if (rr_hist) rr_hist[0] = rr;
    if (bb == 0.0) { /* reading A11 */
        *iters = 0;
        *true_res = 0.0;
        status = 0;
        goto done;
    }
    for (k = 1; k <= maxiter; ++k) {
        apply_A(&op, p, Ap);
        const double pAp = dot_re(p, Ap, n);
        const double alpha = rr / pAp;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; ++i) {
            x[i] += alpha * p[i];
            r[i] -= alpha * Ap[i];
        }
        const double rr_new = dot_re(r, r, n);
        if (rr_hist) rr_hist[k] = rr_new;
        if (rr_new <= tol * tol * bb) {
            status = 0;
            break;
        }
        const double beta = rr_new / rr;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; ++i) p[i] = r[i] + beta * p[i];
        rr = rr_new;
    }
    *iters = status == 0 ? k : maxiter;
    /* true residual with a fresh application of A (row S7) */
    apply_A(&op, x, Ap);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; ++i) Ap[i] = b[i] - Ap[i];
    *true_res = sqrt(dot_re(Ap, Ap, n) / bb);
done:
    free(r);
    free(p);
    free(Ap);
    return status;
#undef op
}

int oracle_cg(const int *L, int fermion, const double *u_, double param, double tol, int maxiter, const double *b_,
              double *x_, int *iters, double *true_res, double *rr_hist)
{
    op_t op;
    if (fermion != ORACLE_STAGGERED && fermion != ORACLE_WILSON) return -2;
    int rc = op_init(&op, L, fermion, (const cd *)u_, param);
    if (rc) return rc;
    rc = cg_core(&op, tol, maxiter, b_, x_, iters, true_res, rr_hist);
    op_free(&op);
    return rc;
}

/* ------------------------------------------------ full-system staggered solve */

/* M = m + D on a full-lattice staggered vector given as its even and odd halves
 * ("M = m + D, M^+ = m - D"): out_e = m in_e + D_eo in_o,
 * out_o = m in_o + D_oe in_e. */
int oracle_stag_M(const int *L, const double *u, double mass, const double *in_e, const double *in_o, double *out_e,
                  double *out_o)
{
    geom_t G;
    if (geom_init(&G, L)) return -1;
    const long n = 3 * G.Vh;
    const cd *ie = (const cd *)in_e, *io = (const cd *)in_o;
    cd *oe = (cd *)out_e, *oo = (cd *)out_o;
    stag_dslash(&G, (const cd *)u, 0, io, oe); /* D_eo in_o */
    stag_dslash(&G, (const cd *)u, 1, ie, oo); /* D_oe in_e */
    for (long i = 0; i < n; ++i) {
        oe[i] = mass * ie[i] + oe[i];
        oo[i] = mass * io[i] + oo[i];
    }
    return 0;
}

/* Solve M x = b on the full lattice, the way the hybrid molecular dynamics needs it
 * (the paper's congrad has two outputs, copyout(x,y)).
 * Written out in even/odd blocks, M x = b reads
 *     m x_e + D_eo x_o = b_e,      m x_o + D_oe x_e = b_o,
 * so   x_o = (b_o - D_oe x_e)/m   and   (m^2 - D_eo D_oe) x_e = m b_e - D_eo b_o.
 * Steps, in this order:
 *   1. b' = m b_e - D_eo b_o                      (source preparation)
 *   2. CG on A x_e = b', A = m^2 - D_eo D_oe      (oracle_cg above, tol relative to |b'|)
 *   3. x_o = (b_o - D_oe x_e)/m                   (reconstruction)
 *   4. true_res = |b - M x| / |b| over the full lattice, with M applied afresh
 * Returns the CG's status (0 converged, 1 maxiter); mass = 0 is an error (-2).
 * b = 0 gives x = 0, iters = 0, true_res = 0. */
int oracle_stag_solve_full(const int *L, const double *u_, double mass, double tol, int maxiter, const double *b_e_,
                           const double *b_o_, double *x_e_, double *x_o_, int *iters, double *true_res)
{
    geom_t G;
    if (geom_init(&G, L)) return -1;
    if (mass == 0.0) return -2;
    const long n = 3 * G.Vh;
    const cd *u = (const cd *)u_, *be = (const cd *)b_e_, *bo = (const cd *)b_o_;
    cd *xe = (cd *)x_e_, *xo = (cd *)x_o_;
    cd *bp = malloc(sizeof(cd) * n), *t = malloc(sizeof(cd) * n), *me = malloc(sizeof(cd) * n), *mo = malloc(sizeof(cd) * n);
    if (!bp || !t || !me || !mo) return -3;
    /* 1 */
    stag_dslash(&G, u, 0, bo, t);
    for (long i = 0; i < n; ++i) bp[i] = mass * be[i] - t[i];
    /* 2 */
    double cg_res = 0.0;
    const int status = oracle_cg(L, ORACLE_STAGGERED, u_, mass, tol, maxiter, (const double *)bp, x_e_, iters, &cg_res, NULL);
    if (status < 0) return status;
    /* 3 */
    stag_dslash(&G, u, 1, xe, t);
    for (long i = 0; i < n; ++i) xo[i] = (bo[i] - t[i]) / mass;
    /* 4 */
    oracle_stag_M(L, u_, mass, x_e_, x_o_, (double *)me, (double *)mo);
    for (long i = 0; i < n; ++i) {
        me[i] = be[i] - me[i];
        mo[i] = bo[i] - mo[i];
    }
    const double bb = dot_re(be, be, n) + dot_re(bo, bo, n);
    *true_res = bb > 0.0 ? sqrt((dot_re(me, me, n) + dot_re(mo, mo, n)) / bb) : 0.0;
    free(bp);
    free(t);
    free(me);
    free(mo);
    return status;
}

/* ------------------------------------------- mixed-precision CG (fp32 inner) */

/* the technique of the paper's reference [2] (Clark et al.,
 * "Solving Lattice QCD systems of equations using mixed precision solvers on GPUs"): the CG
 * iteration runs on fp32 copies of the links and vectors ("sloppy" precision) and is tied to the
 * fp64 problem by RELIABLE UPDATES: whenever the iterated residual has dropped by the factor
 * delta below the largest residual seen since the last update (or claims convergence), the
 * partial solution is added to the fp64 solution, the residual is recomputed in fp64 from its
 * definition b - A x, and the iteration continues from it keeping its search direction.
 *
 * What is fp32 and what is fp64 (DESIGN.md "Mixed precision" states the same contract):
 *   - links uf = fl32(u), vectors xs, rs, ps, ts stored in fp32;
 *   - the hopping term D^ is evaluated in fp32 arithmetic (stag_site_f below);
 *   - every inner product is accumulated in fp64 from the fp32 values;
 *   - the vector updates are evaluated in fp64 from the fp32 values and rounded on store;
 *   - the scalars alpha, beta, <r,r>, the update test and the exit test are fp64;
 *   - the reliable update (x, b - A x, its norm) is entirely fp64 with the fp64 operator. */
typedef float complex cf;

/* stag_site in fp32 arithmetic: same sum, same order. */
static void stag_site_f(const geom_t *G, const cf *u, int parity, long e, const cf *in, cf out[3])
{
    int x[4];
    site_coords(G, parity, e, x);
    const long g = parity * G->Vh + e;
    const long other = (1 - parity) * G->Vh;
    cf acc[3] = { 0, 0, 0 };
    for (int mu = 0; mu < 4; ++mu) {
        const float eta = (float)eta_phase(x, mu);
        {
            const long ef = neighbour(G, x, mu, +1) - other;
            const cf *U = u + (g * 4 + mu) * 9;
            const float sgn = eta * (float)bc_forward(G, x, mu);
            for (int a = 0; a < 3; ++a) {
                cf s = 0;
                for (int b = 0; b < 3; ++b) s += U[a * 3 + b] * in[b * G->Vh + ef];
                acc[a] += sgn * s;
            }
        }
        {
            const long gb = neighbour(G, x, mu, -1);
            const long eb = gb - other;
            const cf *W = u + (gb * 4 + mu) * 9;
            const float sgn = eta * (float)bc_backward(G, x, mu);
            for (int a = 0; a < 3; ++a) {
                cf s = 0;
                for (int b = 0; b < 3; ++b) s += conjf(W[b * 3 + a]) * in[b * G->Vh + eb];
                acc[a] -= sgn * s;
            }
        }
    }
    for (int a = 0; a < 3; ++a) out[a] = 0.5f * acc[a];
}

static void stag_dslash_f(const geom_t *G, const cf *u, int out_parity, const cf *in, cf *out)
{
#pragma omp parallel for schedule(static)
    for (long e = 0; e < G->Vh; ++e) {
        cf r[3];
        stag_site_f(G, u, out_parity, e, in, r);
        for (int a = 0; a < 3; ++a) out[a * G->Vh + e] = r[a];
    }
}

/* Re<a,b> of fp32 vectors accumulated in fp64, fixed blocks as dot_re. */
static double dot_re_f(const cf *a, const cf *b, long n)
{
    const long nb = (n + DOT_BLOCK - 1) / DOT_BLOCK;
    double *part = malloc(sizeof(double) * (nb > 0 ? nb : 1));
#pragma omp parallel for schedule(static)
    for (long k = 0; k < nb; ++k) {
        const long lo = k * DOT_BLOCK, hi = lo + DOT_BLOCK < n ? lo + DOT_BLOCK : n;
        double s = 0.0;
        for (long i = lo; i < hi; ++i)
            s += (double)crealf(a[i]) * (double)crealf(b[i]) + (double)cimagf(a[i]) * (double)cimagf(b[i]);
        part[k] = s;
    }
    double s = 0.0;
    for (long k = 0; k < nb; ++k) s += part[k];
    free(part);
    return s;
}

/* dot_re_f through the C interface, for its own pin (tests/test_oracle_mixed.py): the fp64 arguments are
 * rounded to fp32 and handed to dot_re_f as the mixed-precision CG hands it rs, ps, ts.  No arithmetic of
 * its own.  Returns NaN if the two temporaries cannot be allocated. */
double oracle_dot_re_f(const double *a_, const double *b_, long n_complex)
{
    const cd *a = (const cd *)a_, *b = (const cd *)b_;
    const long n = n_complex > 0 ? n_complex : 0;
    cf *af = malloc(sizeof(cf) * (n > 0 ? n : 1)), *bf = malloc(sizeof(cf) * (n > 0 ? n : 1));
    if (!af || !bf) {
        free(af);
        free(bf);
        return NAN;
    }
    for (long i = 0; i < n; ++i) {
        af[i] = (cf)a[i];
        bf[i] = (cf)b[i];
    }
    const double s = dot_re_f(af, bf, n);
    free(af);
    free(bf);
    return s;
}

/* The fp32 hopping term through the C interface (for its own pin against the fp64 one). */
int oracle_stag_dslash_f32(const int *L, const double *u_, int out_parity, const double *in_, double *out_)
{
    geom_t G;
    if (geom_init(&G, L)) return -1;
    if (out_parity != 0 && out_parity != 1) return -2;
    const long n = 3 * G.Vh, nu = G.V * 36;
    const cd *u = (const cd *)u_, *in = (const cd *)in_;
    cd *out = (cd *)out_;
    cf *uf = malloc(sizeof(cf) * nu), *inf = malloc(sizeof(cf) * n), *of = malloc(sizeof(cf) * n);
    if (!uf || !inf || !of) return -3;
    for (long i = 0; i < nu; ++i) uf[i] = (cf)u[i];
    for (long i = 0; i < n; ++i) inf[i] = (cf)in[i];
    stag_dslash_f(&G, uf, out_parity, inf, of);
    for (long i = 0; i < n; ++i) out[i] = (cd)of[i];
    free(uf);
    free(inf);
    free(of);
    return 0;
}

/* Mixed-precision conjugate gradient with reliable updates on A x = b, A = m^2 - D_eo D_oe
 * (staggered, even sites).  Step by step (k counts applications of the fp32 operator):
 *
 *   x = 0 (fp64); bb = <b,b>; rr = bb; rs = ps = fl32(b); xs = 0; rmax = sqrt(rr)
 *   for k = 1..maxiter:
 *       ts = D^_oe ps;  qs = D^_eo ts                              (fp32 hopping terms)
 *       alpha = rr / (m^2 <ps,ps> + <ts,ts>)                       (<p,Ap> from norms)
 *       xs = fl32(xs + alpha ps);  rs = fl32(rs - alpha (m^2 ps - qs));  rr' = <rs,rs>
 *       update = sqrt(rr') < delta*rmax  or  rr' <= tol^2 bb;      rmax = max(rmax, sqrt(rr'))
 *       if update:                                                  (reliable update, all fp64)
 *           x += xs; xs = 0;  r = b - A x;  rr' = <r,r>;  rs = fl32(r);  rmax = sqrt(rr')
 *           if rr' <= tol^2 bb: converged, stop
 *       beta = rr'/rr;  ps = fl32(rs + beta ps);  rr = rr'
 *   if not converged: x += xs
 *   true_res = |b - A x| / |b| with a fresh fp64 A
 *
 * So convergence is only ever declared on a residual computed in fp64 from its definition.
 * Returns 0 converged / 1 maxiter; *nupdates = number of reliable updates; rr_hist[k] = rr' after
 * iteration k (the fp64 value where an update took place). */
int oracle_cg_mixed(const int *L, const double *u_, double mass, double tol, double delta, int maxiter,
                    const double *b_, double *x_, int *iters, int *nupdates, double *true_res, double *rr_hist)
{
    op_t op;
    int rc = op_init(&op, L, ORACLE_STAGGERED, (const cd *)u_, mass);
    if (rc) return rc;
    if (!(delta > 0.0 && delta < 1.0)) return -2;
    const geom_t *G = &op.G;
    const long n = op.n, nu = G->V * 36;
    const double m2 = mass * mass;
    const cd *b = (const cd *)b_, *u = (const cd *)u_;
    cd *x = (cd *)x_;
    cd *r = malloc(sizeof(cd) * n);
    cf *uf = malloc(sizeof(cf) * nu), *xs = malloc(sizeof(cf) * n), *rs = malloc(sizeof(cf) * n);
    cf *ps = malloc(sizeof(cf) * n), *ts = malloc(sizeof(cf) * n), *qs = malloc(sizeof(cf) * n);
    if (!r || !uf || !xs || !rs || !ps || !ts || !qs) return -3;
    for (long i = 0; i < nu; ++i) uf[i] = (cf)u[i];
    for (long i = 0; i < n; ++i) {
        x[i] = 0;
        xs[i] = 0;
        rs[i] = (cf)b[i];
        ps[i] = rs[i];
    }
    double rr = dot_re(b, b, n);
    const double bb = rr;
    double rmax = sqrt(rr);
    int status = 1, k = 0, nupd = 0;
    if (rr_hist) rr_hist[0] = rr;
    if (bb == 0.0) {
        *iters = 0;
        *nupdates = 0;
        *true_res = 0.0;
        status = 0;
        goto done;
    }
    for (k = 1; k <= maxiter; ++k) {
        stag_dslash_f(G, uf, 1, ps, ts);
        stag_dslash_f(G, uf, 0, ts, qs);
        const double alpha = rr / (m2 * dot_re_f(ps, ps, n) + dot_re_f(ts, ts, n));
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; ++i) {
            const cd pv = (cd)ps[i];
            const cd ap = m2 * pv - (cd)qs[i];
            xs[i] = (cf)((cd)xs[i] + alpha * pv);
            rs[i] = (cf)((cd)rs[i] - alpha * ap);
        }
        double rr_new = dot_re_f(rs, rs, n);
        const double rn = sqrt(rr_new);
        const int update = (rn < delta * rmax) || (rr_new <= tol * tol * bb);
        if (rn > rmax) rmax = rn;
        if (update) {
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) {
                x[i] += (cd)xs[i];
                xs[i] = 0;
            }
            apply_A(&op, x, r);
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) {
                r[i] = b[i] - r[i];
                rs[i] = (cf)r[i];
            }
            rr_new = dot_re(r, r, n);
            rmax = sqrt(rr_new);
            ++nupd;
        }
        if (rr_hist) rr_hist[k] = rr_new;
        if (update && rr_new <= tol * tol * bb) {
            status = 0;
            break;
        }
        const double beta = rr_new / rr;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; ++i) ps[i] = (cf)((cd)rs[i] + beta * (cd)ps[i]);
        rr = rr_new;
    }
    *iters = status == 0 ? k : maxiter;
    *nupdates = nupd;
    if (status != 0) {
        for (long i = 0; i < n; ++i) x[i] += (cd)xs[i];
    }
    apply_A(&op, x, r);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; ++i) r[i] = b[i] - r[i];
    *true_res = sqrt(dot_re(r, r, n) / bb);
done:
    free(r);
    free(uf);
    free(xs);
    free(rs);
    free(ps);
    free(ts);
    free(qs);
    op_free(&op);
    return status;
}

/* ------------------------------------- even-odd preconditioned Wilson solve */

/* Mhat (dagger = 0) or Mhat^+ = gamma5 Mhat gamma5 (dagger = 1) on the even half of a
 * full-lattice vector; the odd half of `out` is zero. */
int oracle_wilson_Mhat(const int *L, const double *u, double kappa, int dagger, const double *in, double *out)
{
    op_t op;
    int rc = op_init(&op, L, ORACLE_WILSON_EO, (const cd *)u, kappa);
    if (rc) return rc;
    if (!dagger) {
        wilson_Mhat(&op.G, op.u, kappa, (const cd *)in, (cd *)out, op.t3);
    } else {
        gamma5_mul(&op.G, (const cd *)in, op.t2);
        wilson_Mhat(&op.G, op.u, kappa, op.t2, op.t1, op.t3);
        gamma5_mul(&op.G, op.t1, (cd *)out);
    }
    op_free(&op);
    return 0;
}

/* Solve M x = b, M = 1 - kappa D_W, on the full lattice through the Schur complement on the
 * even sites.  From  x_e - kappa D_eo x_o = b_e,  x_o - kappa D_oe x_e = b_o:
 *     x_o = b_o + kappa D_oe x_e,      Mhat x_e = b_e + kappa D_eo b_o,   Mhat = 1 - kappa^2 D_eo D_oe.
 * Mhat is not hermitian, so the CG runs on its normal equations (as BASELINE.json config 4 does for M).
 * Steps, in this order:
 *   1. bh = b_e + kappa D_eo b_o                          (source preparation, even sites)
 *   2. c  = Mhat^+ bh = gamma5 Mhat gamma5 bh
 *   3. CG on (Mhat^+ Mhat) x_e = c, 8(c.4) exactly, tol relative to |c|
 *   4. x_o = b_o + kappa D_oe x_e                         (reconstruction)
 *   5. true_res = |b - M x| / |b| over the full lattice with M applied afresh
 * b and x are full-lattice Wilson vectors [4][3][V].  Returns the CG's status. */
int oracle_wilson_solve_eo(const int *L, const double *u_, double kappa, double tol, int maxiter, const double *b_,
                           double *x_, int *iters, double *true_res)
{
    op_t op;
    int rc = op_init(&op, L, ORACLE_WILSON_EO, (const cd *)u_, kappa);
    if (rc) return rc;
    const geom_t *G = &op.G;
    const long V = G->V, Vh = G->Vh, n = 12 * V;
    const cd *u = (const cd *)u_, *b = (const cd *)b_;
    cd *x = (cd *)x_;
    cd *bh = malloc(sizeof(cd) * n), *c = malloc(sizeof(cd) * n), *w = malloc(sizeof(cd) * n);
    if (!bh || !c || !w) return -3;
    /* 1 */
    wilson_dslash(G, u, 0, b, w); /* w_e = D_eo b_o */
    for (int k = 0; k < 12; ++k)
        for (long e = 0; e < Vh; ++e) {
            bh[k * V + e] = b[k * V + e] + kappa * w[k * V + e];
            bh[k * V + Vh + e] = 0;
        }
    /* 2 */
    gamma5_mul(G, bh, w);
    wilson_Mhat(G, u, kappa, w, c, op.t3);
    gamma5_mul(G, c, w);
    memcpy(c, w, sizeof(cd) * n);
    /* 3: x_e in the even half of x (odd half zero) */
    double cg_res = 0.0;
    const int status = cg_core(&op, tol, maxiter, (const double *)c, x_, iters, &cg_res, NULL);
    /* 4 */
    wilson_dslash(G, u, 1, x, w); /* w_o = D_oe x_e */
    for (int k = 0; k < 12; ++k)
        for (long e = 0; e < Vh; ++e) x[k * V + Vh + e] = b[k * V + Vh + e] + kappa * w[k * V + Vh + e];
    /* 5 */
    wilson_M(G, u, kappa, x, w);
    for (long i = 0; i < n; ++i) w[i] = b[i] - w[i];
    const double bb = dot_re(b, b, n);
    *true_res = bb > 0.0 ? sqrt(dot_re(w, w, n) / bb) : 0.0;
    free(bh);
    free(c);
    free(w);
    op_free(&op);
    return status;
}

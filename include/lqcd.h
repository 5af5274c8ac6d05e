/*
 * lqcd.h -- C-ABI boundary of the B200-native conjugate-gradient fermion solver of
 * arXiv 1311.2719 ("Lattice Simulations using OpenACC compilers").
 *
 * The calls are those BASELINE.json `north_star` (a) lists and SURVEY.md 8(b) shapes
 * after the paper's `congrad(nitcg)`, `fmv(offset,len,out,in)`
 * and `fmtv(out,in)`.  Plain pointers and sizes only; no
 * exception crosses this boundary.  Every step runs in hand-written sm_100a kernels;
 * there is no CPU fallback: without a CUDA device every compute call returns
 * LQCD_ECUDA.
 *
 * Pointer suffixes: *_dev = device memory, *_host = host memory.  The caller
 * (PyTorch in the Python binding) allocates every device buffer and owns the CUDA
 * stream; the library keeps no user pointer past a call except the workspace, in
 * which it places its internal gauge copy, the CG vectors, the reduction scratch and
 * the staging buffers of the *_host entry points.  All calls enqueue on the one
 * stream given to lqcd_set_workspace; calls that return values to the host
 * (get_tables, cg_solve, *_host) synchronise that stream before returning.
 *
 * Canonical layouts (little-endian fp64, complex = (re,im) adjacent; V = L0*L1*L2*L3,
 * Vh = V/2; direction mu = 0,1,2,3 <-> x,y,z,t; time is mu = 3):
 *   site index  g = parity*Vh + e,  e = floor(s/2),  s = x0 + L0*(x1 + L1*(x2 + L2*x3)),
 *               parity = (x0+x1+x2+x3) mod 2   (even block first, the paper's l = 1..mvd2,
 *               PAPER.md:69, :83)
 *   gauge       u[g][mu][row][col]    9 complex per link, U_mu(x) stored at the site it leaves
 *   staggered   v[c][e]               c = 0..2, one parity (the paper's p(l,ic))
 *   Wilson      v[spin][c][g]         spin = 0..3, full lattice
 *   tables      iup[mu][g], idn[mu][g] = g-index of x+mu^, x-mu^ (periodic wrap; signs are
 *               not in the tables);  lex2eo[s] = g
 *
 * Operators (the paper's section-3 listing is missing from
 * PAPER.md:46-48):
 *   staggered  (D chi)(x) = 1/2 sum_mu eta_mu(x) [ b+ U_mu(x) chi(x+mu^) - b- U_mu(x-mu^)^+ chi(x-mu^) ],
 *              eta_0 = 1, eta_1 = (-1)^x0, eta_2 = (-1)^(x0+x1), eta_3 = (-1)^(x0+x1+x2);
 *              b+- = -1 on hops across x3 = L3-1 <-> 0 (antiperiodic time), else +1.
 *              A = (M^+ M)_ee = m^2 - D_eo D_oe on even-site vectors.
 *   Wilson     (D_W psi)(x) = sum_mu [ (1-gamma_mu) b+ U_mu(x) psi(x+mu^) + (1+gamma_mu) b- U_mu(x-mu^)^+ psi(x-mu^) ],
 *              DeGrand-Rossi gamma matrices, M = 1 - kappa D_W, A = M^+ M = gamma5 M gamma5 M, full lattice.
 *
 * Return codes: 0 = ok; LQCD_MAXITER (=1) only from the CG calls (outputs still valid);
 * negative = error, message available from lqcd_last_error().
 */
#ifndef LQCD_H
#define LQCD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lqcd_ctx lqcd_ctx; /* opaque; owns no user memory */

enum { LQCD_STAGGERED = 0, LQCD_WILSON = 1 };
enum { LQCD_EVEN = 0, LQCD_ODD = 1 };
enum {
    LQCD_OK = 0,
    LQCD_MAXITER = 1, /* CG stopped at maxiter; x, iters, true_residual are valid */
    LQCD_EDIM = -1,   /* an extent is odd or < 2, or the volume overflows the index type */
    LQCD_EARG = -2,   /* null pointer, bad enum, bad parity, tol < 0, maxiter < 0 */
    LQCD_ESTATE = -3, /* workspace not set or gauge field not loaded */
    LQCD_ECUDA = -4,  /* a CUDA call failed (including: no device) */
    LQCD_ENOMEM = -5  /* workspace too small */
};

/* Solver variants of lqcd_set_option(LQCD_OPT_CG_MODE): all run the same arithmetic in the
 * same order and give bit-identical iterates; they differ only in how the host learns of
 * convergence ("update host(betan)"). */
enum {
    LQCD_CG_SYNC = 0,  /* the paper's scheme: one 8-byte D2H + host test per iteration */
    LQCD_CG_ASYNC = 1, /* kernels of later iterations are enqueued while the scalar is in flight;
                          a device-side flag turns iterations after convergence into no-ops */
    LQCD_CG_GRAPH = 2  /* ASYNC with each batch of iterations replayed from one CUDA graph */
};
enum {
    LQCD_OPT_CG_MODE = 0,
    LQCD_OPT_CG_CHECK_EVERY = 1, /* iterations enqueued per convergence read-back, 1..1024 */
    /* 18 (default): all nine complex entries of a link are stored and read (144 B per link).
     * 12: only the first two rows are stored; the third is rebuilt in registers as the
     * conjugated cross product (PAPER.md:132 names this "two-column link compression" as the
     * optimisation its code does not use): 96 B per link, 864 instead of
     * 1248 B per staggered Dslash site.  Exact for SU(3) links up to rounding (1e-16).
     * Changing it invalidates the loaded gauge field: call lqcd_load_gauge again. */
    LQCD_OPT_RECONSTRUCT = 2,
    /* 64 (default): lqcd_congrad_host solves with lqcd_cg_solve.  32: with lqcd_cg_solve_mixed
     * (delta = 0.1; staggered contexts only). */
    LQCD_OPT_CONGRAD_PRECISION = 3,
    /* 1 (default): the fp32 kernels of lqcd_cg_solve_mixed give each thread two neighbouring sites and
     * read them with 128-bit loads (lattices with L0 % 4 == 0; others use the one-site kernels).
     * 0: one site per thread.  The vectors are bit-identical either way; the partial sums are
     * grouped differently, so scalars differ in the last bits. */
    LQCD_OPT_F32_PAIRS = 4,
    /* The iteration loop of lqcd_cg_solve as ONE cooperative kernel (staggered contexts; grid-wide barriers
     * between the three phases of an iteration, no host round trip and no kernel boundary inside the loop:
     * PAPER.md:100 "the entire conjugate gradient routine runs on the GPU").  -1 (default): automatic --
     * used where the three-kernel iteration is bounded by its kernel boundaries, i.e. on lattices whose
     * links fit the L2 cache (4^4, 16^4); 0: never; 1: always.  The iterates are bit-identical to the
     * other modes run with 32-thread blocks (same arithmetic, same summation order: a warp of the
     * cooperative kernel is one 32-thread block of the three-kernel path; 32 is what LQCD_OPT_STAG_BLOCK's
     * automatic choice gives on those lattices); LQCD_OPT_CG_MODE / _CHECK_EVERY do not apply while it is
     * in use (the exit test runs on the device every iteration).  The automatic choice never overrides an
     * explicit lqcd_set_option(LQCD_OPT_CG_MODE, LQCD_CG_SYNC): a caller who asked for the paper's loop with
     * its host-side exit test gets it on every lattice.  lqcd_last_cg_path() tells which one ran.  A solve
     * longer than 2^20 iterations continues in further launches of the same kernel (same iterates). */
    LQCD_OPT_PERSISTENT = 5,
    /* Threads per block of the fp64 staggered kernels: 0 (default) = by lattice size (32 / 64 / 128: small
     * lattices are latency-bound and gain from more, smaller blocks), or 32, 64, 128.  Changes how the
     * per-block partial sums are grouped, hence the last bits of the inner products -- nothing else. */
    LQCD_OPT_STAG_BLOCK = 6,
    /* Iterations one launch of the LQCD_OPT_PERSISTENT kernel may run, 1..1048576 (default 1048576 = 2^20: the
     * kernel's grid barrier counts arrivals in 32 bits from zero at launch, three per iteration and block).  A
     * solve that needs more continues in the next launch from the scalars the last one left on the device,
     * with one 128-byte read-back in between: same iterates, bit for bit. */
    LQCD_OPT_PERSISTENT_CHUNK = 7
};

/* Create a context for an L0 x L1 x L2 x L3 lattice (every extent even and >= 2; L = 2 is
 * legal: forward and backward neighbour coincide).  Host-only; touches no device. */
int lqcd_create(lqcd_ctx **out, int L0, int L1, int L2, int L3, int fermion_type);
int lqcd_destroy(lqcd_ctx *ctx);

/* Bytes of device scratch the caller must provide (256-byte aligned), and the hand-over.
 * `cuda_stream` is a cudaStream_t (NULL = the legacy default stream).  The workspace must
 * outlive the context or be replaced by another lqcd_set_workspace call. */
size_t lqcd_workspace_bytes(const lqcd_ctx *ctx);
int lqcd_set_workspace(lqcd_ctx *ctx, void *workspace_dev, size_t bytes, void *cuda_stream);

/* Integer options (above).  Returns LQCD_EARG for an unknown option or value. */
int lqcd_set_option(lqcd_ctx *ctx, int option, int value);

/* Convert the canonical gauge field u_dev[V][4][3][3] (complex) into the library's
 * structure-of-arrays copy inside the workspace (the paper's
 * copyin(u) + linkc_acc).  u_dev is not referenced after the call returns
 * control to the stream (stream-ordered). */
int lqcd_load_gauge(lqcd_ctx *ctx, const double *u_dev);

/* Neighbour and index tables (the paper's iup, idn), built on the device
 * by the same index arithmetic the Dslash kernels use and copied to host arrays
 * iup_host[4][V], idn_host[4][V], lex2eo_host[V].  Any of the three may be NULL. */
int lqcd_get_tables(lqcd_ctx *ctx, int32_t *iup_host, int32_t *idn_host, int32_t *lex2eo_host);

/* Bare hopping term, no mass / kappa (the paper's fmv / fmtv).
 * Staggered: in_dev[3][Vh] lives on parity 1-out_parity, out_dev[3][Vh] on out_parity.
 * Wilson: in_dev and out_dev are full-lattice vectors [4][3][V]; the half of in_dev on parity
 * 1-out_parity is read and only the out_parity half of out_dev is written.
 * in_dev and out_dev must not alias. */
int lqcd_dslash(lqcd_ctx *ctx, int out_parity, const double *in_dev, double *out_dev);

/* Throughput sweep of the bare hopping term (BASELINE.json config 5 "Dslash throughput sweep"): `reps`
 * back-to-back launches enqueued natively, ping-pong between the two vectors -- launch k computes
 * parity (first_out_parity + k) mod 2 from the vector launch k-1 wrote (launch 0 reads a_dev and
 * writes b_dev).  For timing only: no host round trip between launches, so lattices whose kernel
 * is shorter than a ctypes call are still measured on the device.  Vectors as lqcd_dslash. */
int lqcd_dslash_sweep(lqcd_ctx *ctx, int first_out_parity, double *a_dev, double *b_dev, int reps);

/* out = A in.  Staggered: even-site vectors, A = mass^2 - D_eo D_oe.  Wilson: full-lattice
 * vectors, A = gamma5 M gamma5 M with M = 1 - kappa D_W.  No aliasing. */
int lqcd_apply_MdagM(lqcd_ctx *ctx, double mass_or_kappa, const double *in_dev, double *out_dev);

/* Conjugate gradient on A x = b from x = 0 (the paper's congrad; steps
 * S1-S7 of SURVEY.md 8(a)): stops when <r,r> <= tol^2 <b,b> (tol = 0: run exactly maxiter
 * iterations) or after maxiter iterations (returns LQCD_MAXITER).  *iters = number of
 * applications of A inside the loop; *true_residual = |b - A x| / |b| from a fresh A.
 * The status is decided by the RECURSION residual, as in the paper (betan.lt.delit):
 * LQCD_OK means <r,r> of the iterated r met the rule; *true_residual is reported beside it and can
 * exceed tol by rounding on ill-conditioned systems (32^4, m = 0.01: 9.94e-11 at tol 1e-10) -- a caller
 * that needs the bound on the true residual compares *true_residual itself (the full-system, even-odd
 * and slab solvers follow the same rule; lqcd_cg_solve_mixed decides on an fp64 true residual).
 * b = 0 gives x = 0, iters = 0, true_residual = 0.  b_dev and x_dev must not alias. */
int lqcd_cg_solve(lqcd_ctx *ctx, double mass_or_kappa, double tol, int maxiter, const double *b_dev, double *x_dev,
                  int *iters, double *true_residual);

/* Mixed-precision conjugate gradient with reliable updates on the same system as lqcd_cg_solve
 * (staggered contexts; the technique of the paper's reference [2],
 * PAPER.md:151).  The iteration (S1-S5) runs on fp32 copies of the links and of x, r, p, t -- half
 * the bytes per iteration -- and is tied to the fp64 problem by reliable updates: when the iterated
 * |r| has fallen below delta times the largest |r| since the last update, or claims convergence,
 * x_dev += xs in fp64, r = b - A x is recomputed in fp64 from its definition with the fp64 links,
 * and the iteration resumes from fl32(r) keeping its search direction.  Convergence
 * (<r,r> <= tol^2 <b,b>) is only ever declared on such an fp64 residual, so *true_residual <= tol
 * holds as for lqcd_cg_solve.  fp32/fp64 split: hopping terms in fp32; inner products accumulated in
 * fp64; vector updates evaluated in fp64 and rounded on store; all scalars and tests fp64.
 * delta in (0,1), typically 0.1.  *iters = fp32 iterations, *reliable_updates = fp64 updates.
 * Contract: the solution agrees with lqcd_cg_solve's within 2 tol |b| / (m^2 |x|);
 * iteration counts are NOT comparable to +-2 (fp32 rounding changes the trajectory). */
int lqcd_cg_solve_mixed(lqcd_ctx *ctx, double mass, double tol, int maxiter, double delta, const double *b_dev,
                        double *x_dev, int *iters, int *reliable_updates, double *true_residual);

/* Full-system staggered solve M x = b, M = m + D, on the whole lattice (
 * what the hybrid molecular dynamics around the paper's congrad needs, whose data region has two
 * outputs, copyout(x,y)).  Even-odd reduction, every step in the CUDA kernels:
 *   b' = m b_e - D_eo b_o;   CG on (m^2 - D_eo D_oe) x_e = b' (tol relative to |b'|, as lqcd_cg_solve);
 *   x_o = (b_o - D_oe x_e)/m;   *true_residual = |b - M x| / |b| over both parities, M applied afresh.
 * The four vectors are staggered half-lattice vectors [3][Vh] (even / odd sites); none may alias.
 * *iters = CG iterations.  mass = 0 and a Wilson context are LQCD_EARG.  b = 0 gives x = 0. */
int lqcd_stag_solve_full(lqcd_ctx *ctx, double mass, double tol, int maxiter, const double *b_even_dev,
                         const double *b_odd_dev, double *x_even_dev, double *x_odd_dev, int *iters,
                         double *true_residual);

/* Even-odd (Schur) preconditioned Wilson solver (Wilson contexts).  In even/odd
 * blocks M = 1 - kappa D_W = [[1, -kappa D_eo], [-kappa D_oe, 1]]; its Schur complement on the even sites is
 * Mhat = 1 - kappa^2 D_eo D_oe, with Mhat^+ = gamma5 Mhat gamma5.  Vectors are full-lattice Wilson
 * vectors [4][3][V]; "even half" = the entries with site index g < Vh.
 *
 * lqcd_wilson_eo_MdagM: even half of out = Mhat^+ Mhat applied to the even half of in; the odd halves
 * are neither read nor written.  No aliasing.
 *
 * lqcd_wilson_solve_eo: solves M x = b on the full lattice:  bh = b_e + kappa D_eo b_o;  c = Mhat^+ bh;
 * CG (as lqcd_cg_solve, tol relative to |c|) on Mhat^+ Mhat x_e = c;  x_o = b_o + kappa D_oe x_e;
 * *true_residual = |b - M x| / |b| over the full lattice with M applied afresh.  *iters = CG iterations
 * (each costs the same four one-parity hopping terms as an iteration of lqcd_cg_solve, on a better
 * conditioned matrix).  b = 0 gives x = 0. */
int lqcd_wilson_eo_MdagM(lqcd_ctx *ctx, double kappa, const double *in_dev, double *out_dev);
int lqcd_wilson_solve_eo(lqcd_ctx *ctx, double kappa, double tol, int maxiter, const double *b_dev, double *x_dev,
                         int *iters, double *true_residual);

/* The paper's congrad with its data region (copyin(u,r) ... copyout(x)):
 * HOST buffers in the canonical layouts (pinned memory makes the copies asynchronous).
 * Copies u and b to the device, converts the gauge field, solves, copies x back. */
int lqcd_congrad_host(lqcd_ctx *ctx, const double *u_host, double mass_or_kappa, double tol, int maxiter,
                      const double *b_host, double *x_host, int *iters, double *true_residual);

/* Host-buffer form of lqcd_dslash (copies in_host up, out_host down; gauge must be loaded). */
int lqcd_dslash_host(lqcd_ctx *ctx, int out_parity, const double *in_host, double *out_host);

/* Residual history of the last CG call: <r,r> after iteration k at index k (index 0 = <b,b>),
 * for k <= min(iters, 65535).  Copies at most `capacity` values to rr_host and returns the
 * number copied (negative = error). */
int lqcd_cg_history(lqcd_ctx *ctx, double *rr_host, int capacity);

/* Which iteration loop the last CG call on this context ran (lqcd_cg_solve, lqcd_cg_solve_mixed,
 * lqcd_stag_solve_full, lqcd_wilson_solve_eo, lqcd_congrad_host): the host loop in the LQCD_OPT_CG_MODE
 * form, or the one cooperative kernel of LQCD_OPT_PERSISTENT (where LQCD_OPT_CG_MODE / _CHECK_EVERY played no
 * part).  LQCD_PATH_NONE before the first solve; LQCD_EARG for a null context.  Host-only. */
enum { LQCD_PATH_NONE = 0, LQCD_PATH_HOST_LOOP = 1, LQCD_PATH_PERSISTENT = 2 };
int lqcd_last_cg_path(const lqcd_ctx *ctx);

/* Number of kernels launched by this context since creation (for bench.py's gpu_launches). */
long long lqcd_kernel_launches(const lqcd_ctx *ctx);

/* Text of the last error on this context ("" if none).  Valid until the next call on ctx. */
const char *lqcd_last_error(const lqcd_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* LQCD_H */

/*
 * lqcd_slab.h -- time-slab decomposition of the staggered conjugate-gradient solver over several
 * GPUs (the paper's own multi-GPU scheme is PAPER.md:106-136).
 *
 * One rank (one process, one GPU) owns T = L3/nranks consecutive time-slices, both parities, and the
 * links that leave from them.  The operator, the layouts and the CG are those of lqcd.h applied to
 * the global lattice; a slab object works on the rank's part of every array:
 *   local lattice      L0 x L1 x L2 x T (T even, >= 2), time-slices t0 .. t0+T-1 with t0 = rank*T;
 *                      because t0 is even, local parity = global parity and a local vector is the
 *                      contiguous range [t0*sh, (t0+T)*sh) of every colour of the global vector,
 *                      sh = L0*L1*L2/2 sites of one parity per time-slice;
 *   vectors            v[c][e_local], c = 0..2, one parity, as lqcd.h;
 *   gauge              u_local[g_local][mu][3][3] = the canonical layout of lqcd.h on the local
 *                      lattice, plus u3_below[parity][f][3][3], f = 0..sh-1: the links U_3 that leave
 *                      from the time-slice below the slab (global slice t0-1, periodic), which the
 *                      backward time hop of the first local slice needs.
 * Antiperiodic time boundary: on the GLOBAL hop L3-1 <-> 0, wherever the slab boundaries fall.
 *
 * Exchange (what replaces the paper's host-staged MPI_ALLGATHER of the whole vector per iteration,
 * PAPER.md:110-124): per Dslash a rank needs one time-slice of the input vector from each
 * neighbour (sh*48 bytes per face).  The kernel that PRODUCES a vector stores its two boundary
 * slices straight into the neighbours' ghost faces through peer memory (NVLink); inner products
 * travel as one partial per rank into every rank's mailbox -- two 64-bit words, each tagged with the
 * number of the synchronisation point, so that no fence has to order "data" before "flag" -- and are
 * added in rank order, so every rank holds bit-identical scalars.  A synchronisation point (signal, bounded wait, combine) runs in
 * the last block of the producing kernel when a rank drives its own slab, or as two tiny kernels in
 * the *_group calls; nothing goes through the host.  All of that memory is the rank's MAILBOX.
 *
 * Collective semantics: every rank must make the same sequence of lqcd_slab_* compute calls with the
 * same scalar arguments.  A peer that never arrives makes the call fail with LQCD_ECOMM after the
 * wait timeout (default 20 s) instead of hanging the device.
 *
 * Two ways to drive it, one implementation:
 *   - one process per GPU: each rank calls lqcd_slab_dslash / _apply_MdagM / _cg_solve on its own slab;
 *     mailboxes of the other ranks are mapped with the lqcd_slab_ipc_* helpers (CUDA IPC);
 *   - *_group calls: one host thread drives n slabs phase by phase (all producers, then all signals,
 *     then all waits).  With the slabs on one device and one stream this is how the whole path is
 *     tested on a single GPU -- stream order then guarantees that no kernel ever waits for another
 *     (B200_PROFILING.md: kernels that wait on one another must not share a GPU); with the slabs on
 *     several devices of one process (peer access enabled) it is a single-process multi-GPU solver.
 *
 * VALIDATION STATUS: every call is parity-tested against the oracle of the undivided lattice with all
 * slabs on ONE GPU (the *_group calls, and the nranks = 1 ring through the one-rank-per-process calls),
 * where system-scope and device-scope fences behave alike.  The one-rank-per-process path with
 * nranks > 1 (IPC-mapped mailboxes, peer stores over NVLink) has not yet run on more than one GPU:
 * tests/test_gpu_slab.py holds a parity test that runs only where torch.cuda.device_count() >= 2.
 *
 * Pointer suffixes, return codes, error text: as lqcd.h.  No CPU fallback.
 */
#ifndef LQCD_SLAB_H
#define LQCD_SLAB_H

#include "lqcd.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lqcd_slab lqcd_slab; /* opaque; owns no user memory */

enum { LQCD_ECOMM = -6 }; /* a peer did not reach a synchronisation point within the timeout */
enum { LQCD_SLAB_MAX_RANKS = 16 };
enum {
    LQCD_SLAB_OPT_RECONSTRUCT = 0,  /* 18 or 12, as LQCD_OPT_RECONSTRUCT; invalidates the loaded links */
    LQCD_SLAB_OPT_CHECK_EVERY = 1,  /* iterations enqueued per convergence read-back, 1..1024 (default 8) */
    LQCD_SLAB_OPT_TIMEOUT_MS = 2,   /* wait timeout of a synchronisation point, 1..600000 (default 20000) */
    LQCD_SLAB_OPT_GRAPH = 3,        /* 1 (default): when every slab of the call runs on one stream, each batch of
                                       CG iterations is replayed from one CUDA graph (an odd check_every is
                                       rounded up to even); 0: kernel-by-kernel launches.  Same iterates. */
    LQCD_SLAB_OPT_FUSE_SYNC = 4,    /* one-rank-per-process calls only.  1: the last block of every kernel that ends
                                       in a sum (the Dslash kernels of the CG, the p-update, the init) also
                                       signals, waits and combines, so an iteration is three launches and the
                                       exchange costs no kernel boundary; 0: a separate small launch per
                                       synchronisation point, as the *_group calls always do.  Same iterates.
                                       Default: 1 for nranks = 1, 0 for nranks > 1 -- the fused tail has only
                                       ever synchronised with itself (one GPU per box so far); switch it on
                                       explicitly once the separate-launch form has run on real peers. */
    LQCD_SLAB_OPT_ACQUIRE = 5       /* ordering of a synchronisation point against the ghost faces in the PTX memory
                                       model.  1: the thread that sends the tagged words first fences at system scope
                                       (a release of the face stores it learnt of through the ticket chain), and a
                                       receiver that has seen its words fences at system scope before it goes on (an
                                       acquire: the next kernel's ghost-face loads cannot see older data).  0: relaxed
                                       stores and polls only -- enough when every mailbox is in this GPU's memory,
                                       whose L2 is the point of coherence.  -1 (default): 1 if lqcd_slab_connect found
                                       a peer mailbox on another device, else 0.  Same iterates; costs two fences
                                       (microseconds) per synchronisation point, in one block. */
};

/* Slab of rank `rank` of `nranks` for the global L0 x L1 x L2 x L3 staggered lattice.  L3/nranks must be
 * an even integer >= 2 (LQCD_EDIM otherwise); nranks <= LQCD_SLAB_MAX_RANKS.  Host-only. */
int lqcd_slab_create(lqcd_slab **out, int L0, int L1, int L2, int L3, int rank, int nranks);
int lqcd_slab_destroy(lqcd_slab *s);

/* Device memory the caller provides (both 256-byte aligned): the private workspace (links, r, p, t,
 * reduction scratch) and the mailbox (tagged words, ghost faces) the peers store into.  The call zeroes
 * the mailbox words; every rank must have done so before any rank's first compute call (a host
 * barrier in the caller).  cuda_stream as in lqcd_set_workspace. */
size_t lqcd_slab_workspace_bytes(const lqcd_slab *s);
size_t lqcd_slab_mailbox_bytes(const lqcd_slab *s);
int lqcd_slab_set_memory(lqcd_slab *s, void *workspace_dev, size_t workspace_bytes, void *mailbox_dev,
                         size_t mailbox_bytes, void *cuda_stream);

/* peer_mailboxes[r], r = 0..nranks-1: rank r's mailbox as a device pointer this device can store to
 * (the same process: the pointer itself, with peer access enabled across devices; another process:
 * what lqcd_slab_ipc_open returned).  peer_mailboxes[rank] must be the own mailbox. */
int lqcd_slab_connect(lqcd_slab *s, void *const *peer_mailboxes);

int lqcd_slab_set_option(lqcd_slab *s, int option, int value);

/* Links of the slab (layout above), device pointers, converted into the structure-of-arrays copy. */
int lqcd_slab_load_gauge(lqcd_slab *s, const double *u_local_dev, const double *u3_below_dev);

/* out = D in on the slab (bare hopping term as lqcd_dslash): pushes the faces of `in` to the
 * neighbours, synchronises, applies the hopping term.  in/out: local vectors [3][T*sh]. */
int lqcd_slab_dslash(lqcd_slab *s, int out_parity, const double *in_dev, double *out_dev);
/* out = (mass^2 - D_eo D_oe) in on even-site vectors. */
int lqcd_slab_apply_MdagM(lqcd_slab *s, double mass, const double *in_dev, double *out_dev);
/* The conjugate gradient of lqcd_cg_solve on the global system; b and x are the local parts.
 * *iters and *true_residual are global (identical on every rank). */
int lqcd_slab_cg_solve(lqcd_slab *s, double mass, double tol, int maxiter, const double *b_dev, double *x_dev,
                       int *iters, double *true_residual);
/* The mixed-precision conjugate gradient of lqcd_cg_solve_mixed (fp32 iterations on fp32 copies of the links and
 * of x, r, p, t; fp64 reliable updates; PAPER.md:151 ref. [2]) on the global system.
 * The fp32 vectors travel as fp32 faces (sh*24 bytes per face), the x of a reliable update as fp64 faces; every
 * inner product is combined in rank order, so the pause / resume / exit decisions are identical on every rank.
 * One small launch per synchronisation point (no fused tails, no graph replay: the host loop has to see the
 * pause).  Arguments and contract as lqcd_cg_solve_mixed; *iters, *reliable_updates, *true_residual are global. */
int lqcd_slab_cg_solve_mixed(lqcd_slab *s, double mass, double tol, int maxiter, double delta, const double *b_dev,
                             double *x_dev, int *iters, int *reliable_updates, double *true_residual);

/* The same three operations on n slabs driven by the calling thread (n = nranks of every slab, slabs[r]
 * of rank r, all connected to each other).  in/out/b/x: arrays of n device pointers. */
int lqcd_slab_dslash_group(lqcd_slab *const *slabs, int n, int out_parity, const double *const *in_dev,
                           double *const *out_dev);
int lqcd_slab_apply_MdagM_group(lqcd_slab *const *slabs, int n, double mass, const double *const *in_dev,
                                double *const *out_dev);
int lqcd_slab_cg_solve_group(lqcd_slab *const *slabs, int n, double mass, double tol, int maxiter,
                             const double *const *b_dev, double *const *x_dev, int *iters, double *true_residual);
int lqcd_slab_cg_solve_mixed_group(lqcd_slab *const *slabs, int n, double mass, double tol, int maxiter, double delta,
                                   const double *const *b_dev, double *const *x_dev, int *iters, int *reliable_updates,
                                   double *true_residual);

/* CUDA IPC plumbing for one process per GPU: export the own mailbox as a 64-byte handle plus the
 * offset of the mailbox inside the allocation the handle names; open / close a peer's. */
int lqcd_slab_ipc_export(lqcd_slab *s, unsigned char handle[64], size_t *offset);
int lqcd_slab_ipc_open(lqcd_slab *s, const unsigned char handle[64], size_t offset, void **peer_mailbox);
int lqcd_slab_ipc_close(lqcd_slab *s, void *peer_mailbox, size_t offset);

/* Synchronisation points passed since lqcd_slab_connect and kernels launched since creation. */
long long lqcd_slab_sync_points(const lqcd_slab *s);
long long lqcd_slab_kernel_launches(const lqcd_slab *s);
const char *lqcd_slab_last_error(const lqcd_slab *s);

#ifdef __cplusplus
}
#endif
#endif /* LQCD_SLAB_H */

/*
 * lqcd_noalloc.h -- one entry point of liblqcd_b200.so for callers that cannot allocate device memory.
 *
 * Who this is for.  Everything in include/lqcd.h runs on a workspace the CALLER allocates
 * (lqcd_workspace_bytes / lqcd_set_workspace), and its context pins a few host bytes with cudaHostAlloc.
 * Some programs that embed a solver cannot do either at the point where they need a kernel:
 *   - a simulation that sized its fields to fill the card at start-up (the paper picks its lattices by what
 *     fits a 6 GB GPU): a later cudaMalloc can fail, or succeed only by fragmenting what was
 *     carefully packed;
 *   - a plug-in running under a host framework whose own allocator owns all device memory and forbids raw
 *     cudaMalloc / cudaFree in extension code;
 *   - code in the middle of a molecular-dynamics trajectory with several streams in flight: cudaMalloc and
 *     cudaFree synchronise the whole device, so one allocation stalls every stream.
 * For them the scratch memory of the kernel below (per-block partial sums and the ticket counter of the
 * deterministic reduction, csrc/reduce.cuh) lives in a fixed array compiled into the library instead of in
 * a workspace.  No context, no workspace, no cudaMalloc / cudaFree / cudaHostAlloc, no allocating library
 * routine, on the first call or any later one.
 *
 * The price, and the limit.  The array is LQCD_NOALLOC_SCRATCH_BYTES (64 KiB + 256 B) of device memory on
 * EVERY GPU on which the process has loaded this library, held until the process exits whether or not the entry point is
 * ever called.  It has room for LQCD_NOALLOC_MAX_TILES partial sums, one per tile of
 * LQCD_NOALLOC_TILE complex numbers, so a vector may have at most LQCD_NOALLOC_MAX_COMPLEX =
 * 33 554 432 complex numbers (512 MiB; twice the CG vector of the 48^3 x 96 lattice).  Longer vectors are
 * refused with LQCD_ENOMEM and nothing is launched.
 *
 * Sharing.  There is ONE array per GPU and every call on that GPU uses it.  It keeps whatever the previous call
 * left: the entry point clears the ticket counter on the caller's stream before each launch (the partial sums
 * need no clearing, every slot that is read is written first by the same launch).  Two calls that can run
 * on the GPU at the same time -- different streams without an event between them, or two host threads --
 * race on the array and give wrong sums.  Put calls on one stream, or order them yourself.
 *
 * First call on a device.  The first call made while a given device is current looks up the device address
 * of the array (cudaGetSymbolAddress; the array's name is only a placeholder on the host side) and remembers
 * it for that device.  Make that first call at set-up time, on each device you will use, with that device
 * current and BEFORE any stream capture is begun.  Later calls do no set-up.
 */
#ifndef LQCD_NOALLOC_H
#define LQCD_NOALLOC_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LQCD_NOALLOC_TILE 4096u                 /* complex numbers summed by one block          */
#define LQCD_NOALLOC_MAX_TILES 8192u            /* partial-sum slots in the static array        */
#define LQCD_NOALLOC_MAX_COMPLEX ((size_t)LQCD_NOALLOC_TILE * LQCD_NOALLOC_MAX_TILES) /* 33 554 432 */
#define LQCD_NOALLOC_SCRATCH_BYTES (256u + 8u * LQCD_NOALLOC_MAX_TILES)               /* 65 792     */

/* First fused loop of the paper's congrad in one pass over the
 * source:   p = r = b,   x = 0,   *bb_dev = <b,b> = sum |b_i|^2   (the paper's betan before the loop).
 * It computes what the S6 kernel of lqcd_cg_solve computes, with the reduction scratch in the static array.
 *
 *   b_dev                  in   n_complex complex fp64 numbers ((re,im) adjacent), device memory, any CG-vector
 *                               layout of include/lqcd.h -- the operation is elementwise
 *   x_dev, r_dev, p_dev    out  n_complex complex fp64 each, device memory; must not overlap b_dev or each other
 *   bb_dev                 out  one fp64 in device memory (stays on the device: the value is stream-ordered like
 *                               the vectors; copy it back yourself if the host needs it)
 *   cuda_stream                 a cudaStream_t of the CURRENT device (NULL = the legacy default stream)
 *
 * All five pointers must be 16-byte aligned except bb_dev (8).  The caller owns every buffer; the library keeps
 * no pointer after the call.  The call only enqueues (one 256-byte memset + one kernel) and returns; it does
 * not synchronise.  n_complex = 0 is legal: nothing is written but *bb_dev = 0.
 * The sum is deterministic: tile partials are added in a fixed order, no floating-point atomics.  It groups the
 * terms differently from lqcd_cg_solve's kernel, so the two agree to rounding (1e-15 relative), not bit for bit.
 *
 * Returns LQCD_OK (0);  LQCD_EARG (-2): a null or misaligned pointer;  LQCD_ENOMEM (-5): n_complex >
 * LQCD_NOALLOC_MAX_COMPLEX;  LQCD_ECUDA (-4): no device, the address look-up, the memset or the launch failed.
 * The text of the last error of the calling thread is in lqcd_noalloc_last_error(). */
int lqcd_cg_init_noalloc(const double *b_dev, double *x_dev, double *r_dev, double *p_dev, size_t n_complex,
                         double *bb_dev, void *cuda_stream);

/* LQCD_NOALLOC_MAX_COMPLEX as the loaded library was compiled (for bindings that cannot read the macro). */
size_t lqcd_noalloc_max_complex(void);

/* Message of the last failed lqcd_cg_init_noalloc call made by this host thread ("" if none).  Host-only. */
const char *lqcd_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LQCD_NOALLOC_H */

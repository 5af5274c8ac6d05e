// lqcd_noalloc.cu -- the one entry point of include/lqcd_noalloc.h: the S6 pass of the conjugate gradient
// (p = r = b, x = 0, <b,b>) for callers that must not allocate device memory (a code whose
// fields already fill the card, a plug-in under a framework that owns the allocator, a trajectory that cannot
// afford cudaMalloc's device-wide synchronisation -- see the header).
//
// Every other kernel of the library that reduces takes its scratch (one partial sum per block + a ticket
// counter, reduce.cuh) from the workspace the caller allocated.  Here that scratch is the file-scope array
// below: part of the library's image, present on every GPU that loads it, shared by all calls.
//
// Nothing in this file calls cudaMalloc, cudaFree, cudaHostAlloc or a library routine that allocates.
#include <cuda_runtime.h>
#include <stdarg.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "../../include/lqcd.h"
#include "../../include/lqcd_noalloc.h"
#include "reduce.cuh"

using namespace lqcd;

namespace {

constexpr int kBlock = 256;                              // threads per block
constexpr unsigned int kTile = LQCD_NOALLOC_TILE;        // complex numbers per block: 16 per thread
constexpr unsigned int kMaxTiles = LQCD_NOALLOC_MAX_TILES;
constexpr size_t kTicketBytes = 256;                     // the ticket counter has the first 256 bytes to itself
constexpr size_t kScratchBytes = LQCD_NOALLOC_SCRATCH_BYTES;
static_assert(kScratchBytes == kTicketBytes + sizeof(double) * kMaxTiles, "layout of the static scratch");
static_assert(kTile % kBlock == 0, "a tile is a whole number of elements per thread");

// The scratch itself: [0, 256) the ticket counter of grid_sum (must be zero when a kernel starts),
// [256, 256 + 8 * kMaxTiles) one partial sum per block.
//
// On the HOST side the name `noalloc_scratch` is only a handle for the runtime's symbol look-up -- it is not a device
// address, and a kernel handed `noalloc_scratch` (or &noalloc_scratch[0]) from host code would fault, or scribble over whatever
// host memory the GPU can reach.  Host code below therefore asks cudaGetSymbolAddress for the real address,
// once per device, and passes THAT to the kernel.
static __device__ __align__(256) unsigned char noalloc_scratch[kScratchBytes];

// Device address of noalloc_scratch on each device, filled in by the first call made with that device current.
constexpr int kMaxDevices = 64;
void* g_scratch_addr[kMaxDevices];   // zero-initialised: "not looked up yet"
std::mutex g_setup_lock;

thread_local char t_err[320] = "";

int fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof t_err, fmt, ap);
    va_end(ap);
    return code;
}

// Set-up, once per device, with that device current: device address of the static scratch.
int scratch_for_current_device(unsigned char** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(LQCD_ECUDA, "cudaGetDevice failed: %s (no CUDA device?)", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return fail(LQCD_ECUDA, "device ordinal %d is outside 0..%d", dev, kMaxDevices - 1);
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (!g_scratch_addr[dev]) {
        void* ptr = nullptr;
        e = cudaGetSymbolAddress((void**)&ptr, noalloc_scratch);
        if (e != cudaSuccess || !ptr)
            return fail(LQCD_ECUDA, "cudaGetSymbolAddress(noalloc_scratch) failed on device %d: %s", dev, cudaGetErrorString(e));
        g_scratch_addr[dev] = ptr;
    }
    *out = (unsigned char*)g_scratch_addr[dev];
    return LQCD_OK;
}

// S6 with one TILE of the vector per block (no grid-stride loop: the number of blocks, hence of partial sums,
// is what the fixed scratch bounds).  Otherwise cg_init_kernel (cg_kernels.cuh) without the CG bookkeeping:
// the only scalar that leaves is <b,b>.
__global__ void __launch_bounds__(kBlock) cg_init_noalloc_kernel(const cplx* __restrict__ b, cplx* __restrict__ x,
                                                                 cplx* __restrict__ r, cplx* __restrict__ p, size_t n,
                                                                 double* __restrict__ bb, ReduceScratch rs)
{
    const size_t base = (size_t)blockIdx.x * kTile;
    double local = 0.0;
#pragma unroll 4
    for (unsigned int k = threadIdx.x; k < kTile; k += kBlock) {
        const size_t i = base + k;
        if (i < n) {
            const cplx v = b[i];
            r[i] = v;
            p[i] = v;
            x[i] = cmake(0.0, 0.0);
            local += cnorm2(v);
        }
    }
    grid_sum<kBlock>(local, rs, [bb](double total) { *bb = total; });
}

bool misaligned(const void* p, uintptr_t a) { return ((uintptr_t)p & (a - 1)) != 0; }

}  // namespace

extern "C" {

int lqcd_cg_init_noalloc(const double* b_dev, double* x_dev, double* r_dev, double* p_dev, size_t n_complex,
                         double* bb_dev, void* cuda_stream)
{
    if (!bb_dev || misaligned(bb_dev, 8)) return fail(LQCD_EARG, "bb_dev is null or not 8-byte aligned");
    if (n_complex > 0 && (!b_dev || !x_dev || !r_dev || !p_dev)) return fail(LQCD_EARG, "null vector pointer");
    if (misaligned(b_dev, 16) || misaligned(x_dev, 16) || misaligned(r_dev, 16) || misaligned(p_dev, 16))
        return fail(LQCD_EARG, "vector pointers must be 16-byte aligned (complex fp64)");
    if (n_complex > LQCD_NOALLOC_MAX_COMPLEX)
        return fail(LQCD_ENOMEM,
                    "n_complex = %zu exceeds LQCD_NOALLOC_MAX_COMPLEX = %zu: the static scratch holds %u partial sums, one per "
                    "%u-element tile; use lqcd_cg_solve with a caller-allocated workspace for longer vectors",
                    n_complex, (size_t)LQCD_NOALLOC_MAX_COMPLEX, kMaxTiles, kTile);

    unsigned char* scratch = nullptr;
    const int rc = scratch_for_current_device(&scratch);
    if (rc) return rc;
    ReduceScratch rs;
    rs.ticket = (unsigned int*)scratch;
    rs.partials = (double*)(scratch + kTicketBytes);

    cudaStream_t stream = (cudaStream_t)cuda_stream;
    // The array keeps what the last call left.  grid_sum needs the ticket at zero; it puts it back to zero itself,
    // but a launch that died half-way would not have, so it is cleared here every time (a memset, not an allocation).
    cudaError_t e = cudaMemsetAsync(scratch, 0, kTicketBytes, stream);
    if (e != cudaSuccess) return fail(LQCD_ECUDA, "cudaMemsetAsync of the ticket counter failed: %s", cudaGetErrorString(e));

    size_t tiles = (n_complex + kTile - 1) / kTile;
    if (tiles < 1) tiles = 1;   // n = 0 still has to write *bb_dev = 0
    cg_init_noalloc_kernel<<<(unsigned int)tiles, kBlock, 0, stream>>>((const cplx*)b_dev, (cplx*)x_dev, (cplx*)r_dev,
                                                                       (cplx*)p_dev, n_complex, bb_dev, rs);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(LQCD_ECUDA, "launch of cg_init_noalloc_kernel failed: %s", cudaGetErrorString(e));
    return LQCD_OK;
}

size_t lqcd_noalloc_max_complex(void) { return LQCD_NOALLOC_MAX_COMPLEX; }

const char* lqcd_noalloc_last_error(void) { return t_err; }

}  // extern "C"

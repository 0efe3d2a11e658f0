// static_scratch.cu -- rcg_eri_batch_static: the hot path for callers that may not allocate (code under CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc).  It is rcg_eri_batch for the classes whose kernels need SCRATCH -- the block-tier
// classes with side kernels (gen/emit_heavy.py: every class with a g shell and the light-ket (fd|xx), (ff|xx) classes), whose
// evaluation kernel hands H[quartet][ket target][bra target] and the half-transformed block to the two Phase-2 side kernels through
// a workspace (the paper's Tier-2 buffer) -- with that workspace in a file-scope device array instead of a
// caller-provided allocation.  The array has a fixed, modest size (RCG_STATIC_SCRATCH_BYTES = 32 MiB); every GPU that loads the library
// holds it until the process exits.
//
// Nothing here, and nothing it calls for these classes, calls cudaMalloc, cudaFree or an allocating library routine: the launchers of
// these classes only raise a kernel's shared-memory limit once per device (cudaFuncSetAttribute) and launch.  (The light classes'
// launchers may take two statistics words from the library's memory pool, and the table-driven global tier uploads its tables on
// first use; neither is reachable from this entry point, which refuses classes that need no scratch -- call rcg_eri_batch with a
// NULL workspace for those.)
//
// All calls share the one array, and it keeps the last call's contents.  Nothing in it has to start at zero: the evaluation kernel
// writes every element of H it later reads and the bra side kernel every element of the half-transformed block, so no clearing is
// needed.  Two calls that overlap on the GPU (different streams, or different host threads without an ordering between their
// streams) RACE on the array; calls on one stream are ordered and safe.
#include <atomic>
#include "rcg_internal.h"

#define RCG_STATIC_SCRATCH_DOUBLES (RCG_STATIC_SCRATCH_BYTES / 8)
static __device__ __align__(256) double rcg_static_scratch[RCG_STATIC_SCRATCH_DOUBLES];

// In host code `rcg_static_scratch` is a host-side stand-in, not a device address: the address the kernels can use comes from
// cudaGetSymbolAddress, once per device, with that device current.
static std::atomic<double *> scratch_of[64];

static cudaError_t static_scratch_ptr(double **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    double *p = scratch_of[dev].load(std::memory_order_acquire);
    if (!p) {
        void *q = nullptr;
        if ((e = cudaGetSymbolAddress(&q, rcg_static_scratch)) != cudaSuccess) return e;     // a lost race repeats an idempotent call
        p = (double *)q;
        scratch_of[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return cudaSuccess;
}

extern "C" rcg_status rcg_eri_batch_static_max_quartets(const rcg_basis *b, int la, int lb, int lc, int ld, int64_t *max_quartets)
{
    if (!b || !max_quartets) return RCG_ERR_INVALID_ARG;
    size_t one = 0;
    rcg_status s = rcg_eri_workspace_bytes(b, la, lb, lc, ld, 1, &one);
    if (s != RCG_OK) return s;
    if (one == 0) return RCG_ERR_UNSUPPORTED_CLASS;          // the class uses no scratch: rcg_eri_batch with a NULL workspace allocates nothing either
    *max_quartets = (int64_t)(RCG_STATIC_SCRATCH_BYTES / one);       // scratch of a launch = bytes per quartet x quartets (up to one chunk)
    return RCG_OK;
}

extern "C" rcg_status rcg_eri_batch_static(const rcg_basis *b, int la, int lb, int lc, int ld, const int32_t *quartets,
                                           int64_t nquartet, double *out, void *stream)
{
    if (!b || nquartet < 0) return RCG_ERR_INVALID_ARG;
    size_t one = 0, need = 0;
    rcg_status s = rcg_eri_workspace_bytes(b, la, lb, lc, ld, 1, &one);
    if (s != RCG_OK) return s;
    if (one == 0) return RCG_ERR_UNSUPPORTED_CLASS;
    if (nquartet == 0) return RCG_OK;
    if ((s = rcg_eri_workspace_bytes(b, la, lb, lc, ld, nquartet, &need)) != RCG_OK) return s;
    if (need > (size_t)RCG_STATIC_SCRATCH_BYTES) return RCG_ERR_STATIC_SCRATCH_LIMIT;
    double *ws = nullptr;
    const cudaError_t e = static_scratch_ptr(&ws);
    if (e != cudaSuccess) return rcg_cuda_fail(e);
    return rcg_eri_batch(b, la, lb, lc, ld, quartets, nquartet, out, ws, (size_t)RCG_STATIC_SCRATCH_BYTES, stream);
}

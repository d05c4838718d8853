// dmrg_stack_dots_noalloc: the RDM accumulation kernel for few right-hand sides (E = S M^T; kernels in
// vec_kernels.cu) for callers that cannot call cudaMalloc - code under CUDA graph capture, tight serving loops, harnesses
// that forbid allocation.  The span partial sums, which dmrg_stack_dots puts into a cudaMalloc'ed buffer per call, live
// here in ONE file-scope device array of a fixed, modest size (every GPU that loads the library holds these 8 MiB until
// exit).  In host code the array's name is only a host-side stand-in for the symbol, not a device address: its device
// address is fetched with cudaGetSymbolAddress in this file, once per device, with that device current, and that pointer
// is what the kernels receive.
//
// Sharing: every call on a device uses the same array.  The kernels overwrite every partial sum they later read (nothing
// has to start at zero, stale contents of the previous call are never read), but two calls that overlap on the GPU (two
// streams, or two host threads) race on it - calls must be ordered on one stream, or otherwise not overlap.
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>

#include "../../include/dmrg_b200.h"
#include "kernels.hpp"

namespace {

constexpr int64_t SCRATCH_DOUBLES = DMRG_STACK_DOTS_NOALLOC_MAX_SCRATCH;      // 2^20 doubles = 8 MiB
static __device__ __align__(256) double g_stack_dots_scratch[SCRATCH_DOUBLES];

// keeps the symbol in the device image whatever the toolchain decides about device variables only the host names
__global__ void stack_dots_scratch_anchor(double* out) { if (out) out[0] = g_stack_dots_scratch[0]; }

constexpr int MAX_DEV = 64;
std::atomic<double*> g_scratch_ptr[MAX_DEV];                                  // device address of the array, per device

// device address of the scratch array on the CURRENT device (looked up once per device); nullptr on failure
double* scratch_address() {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEV) return nullptr;
    double* p = g_scratch_ptr[dev].load(std::memory_order_acquire);
    if (p) return p;
    void* q = nullptr;
    if (cudaGetSymbolAddress(&q, g_stack_dots_scratch) != cudaSuccess || !q) { cudaGetLastError(); return nullptr; }
    g_scratch_ptr[dev].store((double*)q, std::memory_order_release);
    return (double*)q;
}

}  // namespace

extern "C" int dmrg_stack_dots_noalloc(const double* S, int64_t lds, int nrows, const double* M, int64_t ldm, int nc,
                                       int64_t K, double* E, int ldE, void* cuda_stream) {
    if (!S || !M || !E || nrows < 1 || nc < 1 || nc > 8 || K < 0 || (lds & 1) || (ldm & 1) || ldE < nc) return DMRG_EINVAL;
    if ((((uintptr_t)S) & 15) || (((uintptr_t)M) & 15)) return DMRG_EINVAL;
    if (dmrg::stack_dots_scratch(nrows, nc, K) > SCRATCH_DOUBLES) return DMRG_ENOMEM;   // beyond the static scratch: use dmrg_stack_dots
    double* scratch = scratch_address();
    if (!scratch) return DMRG_ECUDA;
    dmrg::launch_stack_dots(S, lds, nrows, M, ldm, nc, K, E, ldE, scratch, (cudaStream_t)cuda_stream);
    return cudaGetLastError() == cudaSuccess ? DMRG_OK : DMRG_ECUDA;
}

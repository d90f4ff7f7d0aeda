// carve_noalloc.cu -- carve_fwd_bwd_static: training forward + backward with NO caller workspace and no allocation.
//
// carve_fwd (training) and carve_bwd exchange a workspace -- the chunk records the forward leaves for the reverse
// kernel, the per-chain weight-gradient partials, the progress flags (carve_tc.cuh Rec, TcWsLayout; the SIMT family's
// checkpoints) -- that the caller normally allocates (carve_workspace_bytes).  Some callers cannot call cudaMalloc:
// code under CUDA graph capture, tight serving loops, harnesses that forbid it.  For them this file holds that
// workspace in a file-scope __device__ array of CARVE_STATIC_SCRATCH_BYTES; the entry point runs the same two calls
// on it.  The kernels, their launch configuration and their results are those of carve_fwd + carve_bwd.
//
//  * Every GPU that loads the library holds the array until the process exits (16 MiB).
//  * Problems whose carve_workspace_bytes() exceeds it are rejected with CARVE_ERR_STATIC_LIMIT; nothing is launched.
//  * Nothing here or below calls cudaMalloc / cudaFree or an allocating library routine.
//  * All calls share the array and it keeps the last call's contents.  Nothing in it has to start at zero except the
//    tensor path's per-chain progress flags, which carve_bwd clears itself (cudaMemsetAsync on the caller's stream)
//    before the reverse kernel; every other region is written before it is read within one call.
//  * Calls that overlap on the GPU (different streams, or different host threads on one device) RACE on the array:
//    keep calls to this entry point on one stream per device, or order them with events.
#include <cuda_runtime.h>

#include <mutex>

#include "carve.h"

namespace {

// In host code this name is a host-side stand-in for the device array, not a device address: the address the kernels
// get is looked up per device with cudaGetSymbolAddress below.
static __device__ __align__(256) unsigned char g_carve_static_scratch[CARVE_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_scratch_ptr[kMaxDevices];   // device address of the array on device i (0: not looked up yet)

// Device address of the scratch array on the CURRENT device; looked up once per device, with that device current.
cudaError_t scratch_on_current_device(void** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {
        void* ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_carve_static_scratch);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        g_scratch_ptr[dev] = ptr;
    }
    *out = g_scratch_ptr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" {

size_t carve_static_scratch_bytes(void) { return (size_t)CARVE_STATIC_SCRATCH_BYTES; }

carve_status_t carve_fwd_bwd_static(const carve_params_t* p, const void* q, const void* k, const void* v, const void* f,
                                    const void* bx, const void* wx, const void* beta, const float* A, const float* tau,
                                    const float* Ub, const float* Uw, const float* Vb, const float* Vw, const float* S0,
                                    void* O, float* S_final, const void* dO, const float* dS_final, void* dq, void* dk,
                                    void* dv, void* df, void* dbx, void* dwx, void* dbeta, float* dA, float* dtau,
                                    float* dUb, float* dUw, float* dVb, float* dVw, float* dS0, void* cuda_stream)
{
    if (!p) return CARVE_ERR_NULL;
    // Pre-flight: carve_bwd without a workspace validates the parameters, the NULL rules, the alignment and the shape
    // and then stops at CARVE_ERR_WORKSPACE before any launch; any other status is the caller's error, reported as is.
    const carve_status_t pre = carve_bwd(p, q, k, v, f, bx, wx, beta, A, tau, Ub, Uw, Vb, Vw, S0, dO, dS_final, dq, dk, dv, df,
                                         dbx, dwx, dbeta, dA, dtau, dUb, dUw, dVb, dVw, dS0, nullptr, 0, cuda_stream);
    if (pre != CARVE_ERR_WORKSPACE) return pre == CARVE_OK ? CARVE_ERR_SHAPE : pre;
    if (!O || !S_final) return CARVE_ERR_NULL;
    if (carve_workspace_bytes(p, 1) > (size_t)CARVE_STATIC_SCRATCH_BYTES) return CARVE_ERR_STATIC_LIMIT;
    void* ws = nullptr;
    if (scratch_on_current_device(&ws) != cudaSuccess) return CARVE_ERR_CUDA;
    carve_status_t s = carve_fwd(p, q, k, v, f, bx, wx, beta, A, tau, Ub, Uw, Vb, Vw, S0, O, S_final, ws,
                                 (size_t)CARVE_STATIC_SCRATCH_BYTES, cuda_stream);
    if (s != CARVE_OK) return s;
    return carve_bwd(p, q, k, v, f, bx, wx, beta, A, tau, Ub, Uw, Vb, Vw, S0, dO, dS_final, dq, dk, dv, df, dbx, dwx, dbeta,
                     dA, dtau, dUb, dUw, dVb, dVw, dS0, ws, (size_t)CARVE_STATIC_SCRATCH_BYTES, cuda_stream);
}

}  // extern "C"

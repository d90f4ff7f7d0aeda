// carve_api.cu -- the C ABI of include/carve.h: host-side validation, workspace carve-up,
// kernel-family selection and the host-buffer entry point.  No arithmetic of the method here.
#include <cstdio>
#include <cstring>
#include <new>

#include "carve_internal.h"

namespace carve {
namespace {

constexpr size_t kMaxSmem = 227 * 1024;

bool one_of(int v, std::initializer_list<int> s)
{
    for (int x : s)
        if (x == v) return true;
    return false;
}

carve_status_t check_params(const carve_params_t* p, bool bwd)
{
    if (!p) return CARVE_ERR_NULL;
    if (p->dtype != CARVE_F32 && p->dtype != CARVE_BF16) return CARVE_ERR_DTYPE;
    if (p->B <= 0 || p->H <= 0 || p->T <= 0) return CARVE_ERR_SHAPE;
    if (!one_of(p->L, {16, 32, 64, 128}) || p->T % p->L != 0) return CARVE_ERR_SHAPE;
    if (!one_of(p->dk, {64, 128, 256}) || !one_of(p->dv, {64, 128, 256})) return CARVE_ERR_SHAPE;
    if (!one_of(p->r, {8, 16, 32})) return CARVE_ERR_SHAPE;
    if ((long long)p->dk * p->dv > 32768) return CARVE_ERR_SHAPE;
    if (p->path != CARVE_PATH_AUTO && p->path != CARVE_PATH_SIMT && p->path != CARVE_PATH_TENSOR)
        return CARVE_ERR_SHAPE;
    if (simt_fwd_smem_bytes(p->dk, p->dv, p->r) > kMaxSmem) return CARVE_ERR_SHAPE;
    if (bwd) {
        if ((long long)p->dk * p->dv > 16384) return CARVE_ERR_SHAPE;
        if (simt_bwd_smem_bytes(p->dk, p->dv, p->r) > kMaxSmem) return CARVE_ERR_SHAPE;
    }
    return CARVE_OK;
}

// Kernel family of a call.  `bwd` = the call is carve_bwd or a carve_fwd that saves for it: the two
// must agree because the workspace layouts differ.  An explicit CARVE_PATH_TENSOR request for a shape
// the tensor path does not cover is refused (no silent substitution).
int resolve_path(const carve_params_t* p, bool bwd)
{
    const bool tc_ok = bwd ? tc_bwd_supported(*p) : tc_fwd_supported(*p);
    if (p->path == CARVE_PATH_TENSOR) return tc_ok ? CARVE_PATH_TENSOR : -1;
    if (p->path == CARVE_PATH_SIMT) return CARVE_PATH_SIMT;
    return tc_ok ? CARVE_PATH_TENSOR : CARVE_PATH_SIMT;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// Scalar-write variant (carve.h): wx, Uw, Vw all NULL.  Returns false when only some of the three are NULL.
bool write_gate_args_ok(const void* wx, const float* Uw, const float* Vw)
{
    const int n = (wx == nullptr) + (Uw == nullptr) + (Vw == nullptr);
    return n == 0 || n == 3;
}

carve_status_t check_arch()
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return CARVE_ERR_CUDA;
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return CARVE_ERR_CUDA;
    return major == 10 ? CARVE_OK : CARVE_ERR_ARCH;
}

void fill_ws(Args& a, const carve_params_t& p, void* workspace)
{
    if (!workspace) {
        a.ws_states = a.ws_E = a.ws_tt = a.ws_G = a.ws_part = nullptr;
        a.part_stride = 0;
        return;
    }
    const WsLayout w = simt_ws_layout(p);
    float* base = static_cast<float*>(workspace);
    a.ws_states = base + w.states;
    a.ws_E = base + w.E;
    a.ws_tt = base + w.tt;
    a.ws_G = base + w.G;
    a.ws_part = base + w.part;
    a.part_stride = w.part_stride;
}

size_t elt(const carve_params_t* p) { return p->dtype == CARVE_BF16 ? 2 : 4; }

}  // namespace
}  // namespace carve

using namespace carve;

// out[i] = sum over slices s (ascending) of in[s * stride + i]   (carve_fwd_bwd_host: shared-weight gradients)
static __global__ void carve_sum_slices_kernel(float* __restrict__ out, const float* __restrict__ in, int n, int ns,
                                               size_t stride)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float acc = 0.f;
    for (int s = 0; s < ns; ++s) acc += in[s * stride + i];
    out[i] = acc;
}

extern "C" {

const char* carve_version(void) { return "carve-b200 0.1 (sm_100a)"; }

const char* carve_status_string(carve_status_t s)
{
    switch (s) {
        case CARVE_OK: return "ok";
        case CARVE_ERR_NULL: return "required pointer is NULL";
        case CARVE_ERR_SHAPE: return "unsupported shape";
        case CARVE_ERR_DTYPE: return "unsupported dtype";
        case CARVE_ERR_ALIGN: return "pointer not 16-byte aligned";
        case CARVE_ERR_WORKSPACE: return "workspace missing or too small";
        case CARVE_ERR_ARCH: return "device is not sm_100";
        case CARVE_ERR_CUDA: return "CUDA runtime error";
        case CARVE_ERR_STATIC_LIMIT: return "problem needs more scratch than the static no-allocation limit (CARVE_STATIC_SCRATCH_BYTES)";
    }
    return "unknown status";
}

size_t carve_workspace_bytes(const carve_params_t* p, int need_bwd)
{
    if (!need_bwd || check_params(p, true) != CARVE_OK) return 0;
    const int path = resolve_path(p, true);
    if (path < 0) return 0;
    return path == CARVE_PATH_TENSOR ? tc_ws_layout(*p).total_bytes : simt_ws_layout(*p).total_bytes;
}

int carve_resolved_path(const carve_params_t* p, int bwd)
{
    if (check_params(p, bwd != 0) != CARVE_OK) return -1;
    return resolve_path(p, bwd != 0);
}

int carve_num_launches(const carve_params_t* p, int bwd)
{
    if (check_params(p, bwd != 0) != CARVE_OK) return 0;
    if (!bwd) return 1;
    // SIMT: persistent reverse kernel + weight-gradient reduction; tensor path: reverse kernel, chunk-local
    // epilogue, dA/dtau chunk reduction, weight-gradient reduction
    return resolve_path(p, true) == CARVE_PATH_TENSOR ? 4 : 2;
}

carve_status_t carve_fwd(const carve_params_t* p, const void* q, const void* k, const void* v, const void* f,
                         const void* bx, const void* wx, const void* beta, const float* A, const float* tau,
                         const float* Ub, const float* Uw, const float* Vb, const float* Vw, const float* S0,
                         void* O, float* S_final, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    carve_status_t s = check_params(p, workspace != nullptr);
    if (s != CARVE_OK) return s;
    if (!q || !k || !v || !f || !bx || !beta || !Ub || !Vb || !O || !S_final || !write_gate_args_ok(wx, Uw, Vw)) return CARVE_ERR_NULL;
    for (const void* ptr : {q, k, v, f, bx, wx, beta, (const void*)A, (const void*)tau, (const void*)Ub,
                            (const void*)Uw, (const void*)Vb, (const void*)Vw, (const void*)S0, (const void*)O,
                            (const void*)S_final, (const void*)workspace})
        if (!aligned16(ptr)) return CARVE_ERR_ALIGN;
    const int path = resolve_path(p, workspace != nullptr);
    if (path < 0) return CARVE_ERR_SHAPE;
    if (workspace && workspace_bytes < carve_workspace_bytes(p, 1)) return CARVE_ERR_WORKSPACE;
    if ((s = check_arch()) != CARVE_OK) return s;

    Args a{};
    a.B = p->B; a.H = p->H; a.T = p->T; a.L = p->L; a.dk = p->dk; a.dv = p->dv; a.r = p->r;
    a.l2norm = p->qk_l2norm; a.scale = p->scale; a.eps = p->eps;
    a.q = q; a.k = k; a.v = v; a.f = f; a.bx = bx; a.wx = wx; a.beta = beta;
    a.A = A; a.tau = tau; a.Ub = Ub; a.Uw = Uw; a.Vb = Vb; a.Vw = Vw; a.S0 = S0;
    a.O = O; a.S_final = S_final;
    if (path == CARVE_PATH_TENSOR) {
        uint8_t* rec = nullptr;
        if (workspace) {
            const TcWsLayout w = tc_ws_layout(*p);
            rec = static_cast<uint8_t*>(workspace) + w.rec;
        }
        return tc_fwd_launch(a, rec, static_cast<cudaStream_t>(cuda_stream)) == cudaSuccess ? CARVE_OK : CARVE_ERR_CUDA;
    }
    fill_ws(a, *p, workspace);
    return simt_fwd_launch(a, p->dtype, static_cast<cudaStream_t>(cuda_stream)) == cudaSuccess ? CARVE_OK
                                                                                              : CARVE_ERR_CUDA;
}

static carve_status_t step_impl(const carve_params_t* p, const void* q, const void* k, const void* v, const void* f,
                                const void* bx, const void* wx, const void* beta, const float* A, const float* tau,
                                const float* Ub, const float* Uw, const float* Vb, const float* Vw, float* S, void* O,
                                const int* cu_seqlens, void* cuda_stream)
{
    if (!p) return CARVE_ERR_NULL;
    if (p->dtype != CARVE_F32 && p->dtype != CARVE_BF16) return CARVE_ERR_DTYPE;
    if (p->B <= 0 || p->H <= 0 || p->T < 1 || p->T > 16) return CARVE_ERR_SHAPE;
    if (!step_supported(p->dk, p->dv) || !one_of(p->r, {8, 16, 32})) return CARVE_ERR_SHAPE;
    if (!q || !k || !v || !f || !bx || !beta || !Ub || !Vb || !S || !O || !write_gate_args_ok(wx, Uw, Vw)) return CARVE_ERR_NULL;
    for (const void* ptr : {q, k, v, f, bx, wx, beta, (const void*)A, (const void*)tau, (const void*)Ub, (const void*)Uw,
                            (const void*)Vb, (const void*)Vw, (const void*)S, (const void*)O})
        if (!aligned16(ptr)) return CARVE_ERR_ALIGN;
    const carve_status_t s = check_arch();
    if (s != CARVE_OK) return s;
    return step_launch(*p, q, k, v, f, bx, wx, beta, A, tau, Ub, Uw, Vb, Vw, S, O, cu_seqlens,
                       static_cast<cudaStream_t>(cuda_stream)) == cudaSuccess
               ? CARVE_OK
               : CARVE_ERR_CUDA;
}

carve_status_t carve_step(const carve_params_t* p, const void* q, const void* k, const void* v, const void* f,
                          const void* bx, const void* wx, const void* beta, const float* A, const float* tau,
                          const float* Ub, const float* Uw, const float* Vb, const float* Vw, float* S, void* O,
                          void* cuda_stream)
{
    return step_impl(p, q, k, v, f, bx, wx, beta, A, tau, Ub, Uw, Vb, Vw, S, O, nullptr, cuda_stream);
}

carve_status_t carve_step_varlen(const carve_params_t* p, const void* q, const void* k, const void* v, const void* f,
                                 const void* bx, const void* wx, const void* beta, const float* A, const float* tau,
                                 const float* Ub, const float* Uw, const float* Vb, const float* Vw, float* S, void* O,
                                 const int* cu_seqlens, void* cuda_stream)
{
    if (!cu_seqlens) return CARVE_ERR_NULL;
    return step_impl(p, q, k, v, f, bx, wx, beta, A, tau, Ub, Uw, Vb, Vw, S, O, cu_seqlens, cuda_stream);
}

// carve_bwd; `epilogue_after`: the tensor path launches its chunk-local epilogue as a plain dependent kernel
// instead of overlapping it with the reverse kernel (see Args::epilogue_after).
static carve_status_t bwd_impl(const carve_params_t* p, const void* q, const void* k, const void* v, const void* f,
                               const void* bx, const void* wx, const void* beta, const float* A, const float* tau,
                               const float* Ub, const float* Uw, const float* Vb, const float* Vw, const float* S0,
                               const void* dO, const float* dS_final, void* dq, void* dk, void* dv, void* df, void* dbx,
                               void* dwx, void* dbeta, float* dA, float* dtau, float* dUb, float* dUw, float* dVb,
                               float* dVw, float* dS0, void* workspace, size_t workspace_bytes, void* cuda_stream,
                               bool epilogue_after)
{
    carve_status_t s = check_params(p, true);
    if (s != CARVE_OK) return s;
    if (!q || !k || !v || !f || !bx || !beta || !Ub || !Vb || !dO || !dq || !dk || !dv || !df || !dbx || !dbeta || !dUb ||
        !dVb || !dS0 || !write_gate_args_ok(wx, Uw, Vw))
        return CARVE_ERR_NULL;
    if (wx && (!dwx || !dUw || !dVw)) return CARVE_ERR_NULL;   // (scalar-write variant: dwx, dUw, dVw are not written)
    if (!wx) { dwx = nullptr; dUw = nullptr; dVw = nullptr; }
    for (const void* ptr : {q, k, v, f, bx, wx, beta, (const void*)A, (const void*)tau, (const void*)Ub,
                            (const void*)Uw, (const void*)Vb, (const void*)Vw, (const void*)S0, dO,
                            (const void*)dS_final, (const void*)dq, (const void*)dk, (const void*)dv,
                            (const void*)df, (const void*)dbx, (const void*)dwx, (const void*)dbeta,
                            (const void*)dA, (const void*)dtau, (const void*)dUb, (const void*)dUw,
                            (const void*)dVb, (const void*)dVw, (const void*)dS0, (const void*)workspace})
        if (!aligned16(ptr)) return CARVE_ERR_ALIGN;
    const int path = resolve_path(p, true);
    if (path < 0) return CARVE_ERR_SHAPE;
    if (!workspace || workspace_bytes < carve_workspace_bytes(p, 1)) return CARVE_ERR_WORKSPACE;
    if ((s = check_arch()) != CARVE_OK) return s;

    Args a{};
    a.B = p->B; a.H = p->H; a.T = p->T; a.L = p->L; a.dk = p->dk; a.dv = p->dv; a.r = p->r;
    a.l2norm = p->qk_l2norm; a.scale = p->scale; a.eps = p->eps;
    a.q = q; a.k = k; a.v = v; a.f = f; a.bx = bx; a.wx = wx; a.beta = beta;
    a.A = A; a.tau = tau; a.Ub = Ub; a.Uw = Uw; a.Vb = Vb; a.Vw = Vw; a.S0 = S0;
    a.dO = dO; a.dS_final = dS_final;
    a.dq = dq; a.dk_ = dk; a.dv_ = dv; a.df = df; a.dbx = dbx; a.dwx = dwx; a.dbeta = dbeta; a.dS0 = dS0;
    a.epilogue_after = epilogue_after;
    if (path == CARVE_PATH_TENSOR)
        return tc_bwd_launch(a, static_cast<uint8_t*>(workspace), tc_ws_layout(*p), dA, dtau, dUb, dUw, dVb, dVw,
                             static_cast<cudaStream_t>(cuda_stream)) == cudaSuccess
                   ? CARVE_OK
                   : CARVE_ERR_CUDA;
    fill_ws(a, *p, workspace);
    return simt_bwd_launch(a, p->dtype, dA, dtau, dUb, dUw, dVb, dVw, static_cast<cudaStream_t>(cuda_stream)) ==
                   cudaSuccess
               ? CARVE_OK
               : CARVE_ERR_CUDA;
}

carve_status_t carve_bwd(const carve_params_t* p, const void* q, const void* k, const void* v, const void* f,
                         const void* bx, const void* wx, const void* beta, const float* A, const float* tau,
                         const float* Ub, const float* Uw, const float* Vb, const float* Vw, const float* S0,
                         const void* dO, const float* dS_final, void* dq, void* dk, void* dv, void* df, void* dbx,
                         void* dwx, void* dbeta, float* dA, float* dtau, float* dUb, float* dUw, float* dVb,
                         float* dVw, float* dS0, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    return bwd_impl(p, q, k, v, f, bx, wx, beta, A, tau, Ub, Uw, Vb, Vw, S0, dO, dS_final, dq, dk, dv, df, dbx, dwx, dbeta,
                    dA, dtau, dUb, dUw, dVb, dVw, dS0, workspace, workspace_bytes, cuda_stream, false);
}

// ---- layer ends -----------------------------------------------------------------
static carve_status_t ends_params_ok(const carve_params_t* p)
{
    if (!p) return CARVE_ERR_NULL;
    if (p->dtype != CARVE_F32 && p->dtype != CARVE_BF16) return CARVE_ERR_DTYPE;
    if (p->B <= 0 || p->H <= 0 || p->T <= 0 || p->dk <= 0 || p->dv <= 0) return CARVE_ERR_SHAPE;
    const int per16 = p->dtype == CARVE_BF16 ? 8 : 4;
    if (p->dk % per16 || p->dv % per16) return CARVE_ERR_SHAPE;
    return CARVE_OK;
}

static carve_status_t silu_impl(const carve_params_t* p, const void* qx, const void* kx, const void* vx, void* q, void* k,
                                void* v, bool bwd, void* cuda_stream)
{
    carve_status_t s = ends_params_ok(p);
    if (s != CARVE_OK) return s;
    if ((qx == nullptr) != (q == nullptr) || (kx == nullptr) != (k == nullptr) || (vx == nullptr) != (v == nullptr))
        return CARVE_ERR_NULL;   // a tensor is skipped by passing NULL for both of its pointers
    for (const void* ptr : {qx, kx, vx, (const void*)q, (const void*)k, (const void*)v})
        if (!aligned16(ptr)) return CARVE_ERR_ALIGN;
    if ((s = check_arch()) != CARVE_OK) return s;
    return silu_qkv_launch(*p, qx, kx, vx, q, k, v, bwd, static_cast<cudaStream_t>(cuda_stream)) == cudaSuccess ? CARVE_OK
                                                                                                                  : CARVE_ERR_CUDA;
}

carve_status_t carve_silu_qkv_fwd(const carve_params_t* p, const void* qx, const void* kx, const void* vx, void* q, void* k,
                                  void* v, void* cuda_stream)
{
    return silu_impl(p, qx, kx, vx, q, k, v, false, cuda_stream);
}

carve_status_t carve_silu_qkv_bwd(const carve_params_t* p, const void* qx, const void* kx, const void* vx, void* dq, void* dk,
                                  void* dv, void* cuda_stream)
{
    return silu_impl(p, qx, kx, vx, dq, dk, dv, true, cuda_stream);
}

size_t carve_out_norm_workspace_bytes(const carve_params_t* p)
{
    if (ends_params_ok(p) != CARVE_OK || !out_norm_supported(*p)) return 0;
    return out_norm_ws_bytes(*p);
}

carve_status_t carve_out_norm_fwd(const carve_params_t* p, const void* o, const float* gain, float eps, void* y,
                                  void* cuda_stream)
{
    carve_status_t s = ends_params_ok(p);
    if (s != CARVE_OK) return s;
    if (!out_norm_supported(*p)) return CARVE_ERR_SHAPE;
    if (!o || !gain || !y) return CARVE_ERR_NULL;
    if (!aligned16(o) || !aligned16(gain) || !aligned16(y)) return CARVE_ERR_ALIGN;
    if ((s = check_arch()) != CARVE_OK) return s;
    return out_norm_launch(*p, false, o, gain, eps, nullptr, y, nullptr, nullptr, static_cast<cudaStream_t>(cuda_stream)) ==
                   cudaSuccess
               ? CARVE_OK
               : CARVE_ERR_CUDA;
}

carve_status_t carve_out_norm_bwd(const carve_params_t* p, const void* o, const float* gain, float eps, const void* dy,
                                  void* d_o, float* dgain, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    carve_status_t s = ends_params_ok(p);
    if (s != CARVE_OK) return s;
    if (!out_norm_supported(*p)) return CARVE_ERR_SHAPE;
    if (!o || !gain || !dy || !d_o || !dgain) return CARVE_ERR_NULL;
    for (const void* ptr : {o, (const void*)gain, dy, (const void*)d_o, (const void*)dgain, (const void*)workspace})
        if (!aligned16(ptr)) return CARVE_ERR_ALIGN;
    if (!workspace || workspace_bytes < out_norm_ws_bytes(*p)) return CARVE_ERR_WORKSPACE;
    if ((s = check_arch()) != CARVE_OK) return s;
    return out_norm_launch(*p, true, o, gain, eps, dy, d_o, static_cast<float*>(workspace), dgain,
                           static_cast<cudaStream_t>(cuda_stream)) == cudaSuccess
               ? CARVE_OK
               : CARVE_ERR_CUDA;
}

// ---- host-buffer entry point ---------------------------------------------------------------------
// The batch is cut into up to 8 slices (chains are independent; [B,T,H,d] makes a batch slice one
// contiguous slab of every token tensor).  Each slice runs copy-in -> carve_fwd -> carve_bwd -> copy-out on a
// stream of its own, so the host->device copies of slice i+1, the kernels of slice i and the device->host
// copies of slice i-1 overlap (PCIe is full duplex; the chains of all slices together still fill the SMs).
// The weight gradients of the slices are summed in a fixed order by one small kernel.
namespace {
struct HostPlan {
    size_t tok_k, tok_v, tok_1, st, w_u, w_vb, w_vw, w_a;  // byte sizes (token tensors and states: per slice)
};
HostPlan plan_of(const carve_params_t* p)
{
    HostPlan h{};
    const size_t tok = (size_t)p->B * p->T * p->H, e = elt(p);
    h.tok_k = tok * p->dk * e;
    h.tok_v = tok * p->dv * e;
    h.tok_1 = tok * e;
    h.st = (size_t)p->B * p->H * p->dv * p->dk * 4;
    h.w_u = (size_t)p->r * p->dv * 4;
    h.w_vb = (size_t)p->dk * p->r * 4;
    h.w_vw = (size_t)p->dv * p->r * 4;
    h.w_a = (size_t)p->H * p->dk * 4;
    return h;
}
size_t up256(size_t n) { return (n + 255) & ~(size_t)255; }
int host_slices(const carve_params_t* p)
{
    int n = 1;
    for (int d = 2; d <= 8; ++d)
        if (p->B % d == 0) n = d;
    return n;
}
size_t wgrad_floats(const carve_params_t* p) { return (size_t)2 * p->H * p->dk + 2 * p->r * p->dv + p->dk * p->r + p->dv * p->r; }
}  // namespace

size_t carve_host_arena_bytes(const carve_params_t* p, int with_bwd)
{
    if (check_params(p, with_bwd != 0) != CARVE_OK) return 0;
    const int ns = host_slices(p);
    carve_params_t ps = *p;
    ps.B = p->B / ns;
    const HostPlan h = plan_of(&ps);
    size_t n = 0, per = 0;
    n += 2 * up256(h.w_a) + 2 * up256(h.w_u) + up256(h.w_vb) + up256(h.w_vw);  // A,tau,Ub,Uw,Vb,Vw
    per += 4 * up256(h.tok_k) + 3 * up256(h.tok_v) + up256(h.tok_1);           // q,k,f,bx ; v,wx,O ; beta
    per += 2 * up256(h.st);                                                     // S0, S_final
    if (with_bwd) {
        per += up256(h.tok_v) + up256(h.st);                                    // dO, dS_final
        per += 4 * up256(h.tok_k) + 2 * up256(h.tok_v) + up256(h.tok_1);       // dq,dk,df,dbx ; dv,dwx ; dbeta
        per += up256(h.st) + up256(wgrad_floats(p) * 4);                        // dS0, weight gradients of the slice
        per += up256(carve_workspace_bytes(&ps, 1));
        n += up256(wgrad_floats(p) * 4);                                        // summed weight gradients
    }
    return n + per * ns;
}

struct carve_host_ctx {
    cudaStream_t side[8];
    cudaEvent_t fork, join[8], arrived[8];
};

static carve_status_t host_impl(carve_host_ctx* ctx, const carve_params_t* p, int with_bwd, const void* q, const void* k,
                                  const void* v, const void* f, const void* bx, const void* wx, const void* beta,
                                  const float* A, const float* tau, const float* Ub, const float* Uw,
                                  const float* Vb, const float* Vw, const float* S0, void* O, float* S_final,
                                  const void* dO, const float* dS_final, void* dq, void* dk, void* dv, void* df,
                                  void* dbx, void* dwx, void* dbeta, float* dA, float* dtau, float* dUb,
                                  float* dUw, float* dVb, float* dVw, float* dS0, void* device_arena,
                                  size_t arena_bytes, void* cuda_stream)
{
    carve_status_t s = check_params(p, with_bwd != 0);
    if (s != CARVE_OK) return s;
    if (!device_arena || arena_bytes < carve_host_arena_bytes(p, with_bwd)) return CARVE_ERR_WORKSPACE;
    if (!aligned16(device_arena)) return CARVE_ERR_ALIGN;
    if (!q || !k || !v || !f || !bx || !wx || !beta || !Ub || !Uw || !Vb || !Vw || !O || !S_final) return CARVE_ERR_NULL;   // (full write gate only)
    if (with_bwd && (!dO || !dq || !dk || !dv || !df || !dbx || !dwx || !dbeta || !dUb || !dUw || !dVb || !dVw || !dS0))
        return CARVE_ERR_NULL;
    if (resolve_path(p, with_bwd != 0) < 0) return CARVE_ERR_SHAPE;
    if ((s = check_arch()) != CARVE_OK) return s;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int ns = host_slices(p);
    carve_params_t ps = *p;
    ps.B = p->B / ns;
    const HostPlan h = plan_of(&ps);
    char* cur = static_cast<char*>(device_arena);
    bool ok = true;
    auto slot = [&](size_t bytes) -> void* { void* d = cur; cur += up256(bytes); return d; };
    auto up = [&](const void* src, size_t bytes, cudaStream_t on) -> void* {  // host -> device copy into the arena
        if (!src) return nullptr;
        void* d = slot(bytes);
        ok = ok && cudaMemcpyAsync(d, src, bytes, cudaMemcpyHostToDevice, on) == cudaSuccess;
        return d;
    };
    auto down = [&](void* dst, const void* src, size_t bytes, cudaStream_t on) {
        if (dst) ok = ok && cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, on) == cudaSuccess;
    };
    auto at = [](const void* base, size_t off) -> const char* { return base ? static_cast<const char*>(base) + off : nullptr; };
    auto atw = [](void* base, size_t off) -> char* { return base ? static_cast<char*>(base) + off : nullptr; };

    // shared weights, on the caller's stream, before the slices fork from it
    float *d_A = (float*)up(A, h.w_a, st), *d_tau = (float*)up(tau, h.w_a, st), *d_Ub = (float*)up(Ub, h.w_u, st),
          *d_Uw = (float*)up(Uw, h.w_u, st), *d_Vb = (float*)up(Vb, h.w_vb, st), *d_Vw = (float*)up(Vw, h.w_vw, st);
    const size_t nwg = wgrad_floats(p);
    float* d_wsum = with_bwd ? (float*)slot(nwg * 4) : nullptr;
    float* d_wpart = nullptr;  // first slice's weight-gradient block; the others follow at a fixed byte stride
    size_t wpart_stride = 0;

    cudaStream_t side[8] = {};
    cudaEvent_t fork = nullptr, join[8] = {}, arrived[8] = {};  // arrived[i]: slice i's host -> device copies done
    if (ctx) {   // caller-owned streams and events (carve_host_ctx_create): nothing is created or destroyed per call
        fork = ctx->fork;
        for (int i = 0; i < 8; ++i) { side[i] = ctx->side[i]; join[i] = ctx->join[i]; arrived[i] = ctx->arrived[i]; }
    } else {
        ok = ok && cudaEventCreateWithFlags(&fork, cudaEventDisableTiming) == cudaSuccess;
    }
    ok = ok && cudaEventRecord(fork, st) == cudaSuccess;
    for (int i = 0; i < ns && ok; ++i) {
        if (ns > 1) {
            if (!ctx) {
                ok = ok && cudaStreamCreateWithFlags(&side[i], cudaStreamNonBlocking) == cudaSuccess;
                ok = ok && cudaEventCreateWithFlags(&join[i], cudaEventDisableTiming) == cudaSuccess;
                ok = ok && cudaEventCreateWithFlags(&arrived[i], cudaEventDisableTiming) == cudaSuccess;
            }
            ok = ok && cudaStreamWaitEvent(side[i], fork, 0) == cudaSuccess;
        } else {
            side[i] = st;
        }
    }
    carve_status_t rs = CARVE_OK;
    for (int i = 0; i < ns && ok && rs == CARVE_OK; ++i) {
        cudaStream_t ss = side[i];
        // copies of different streams may run on different copy engines and share the link: keep the slices'
        // uploads in order, so that slice i is complete (and its kernels start) after (i+1)/ns of the transfer
        if (ns > 1 && i > 0) ok = ok && cudaStreamWaitEvent(ss, arrived[i - 1], 0) == cudaSuccess;
        const size_t okk = (size_t)i * h.tok_k, ov = (size_t)i * h.tok_v, o1 = (size_t)i * h.tok_1, os = (size_t)i * h.st;
        void *d_q = up(at(q, okk), h.tok_k, ss), *d_k = up(at(k, okk), h.tok_k, ss), *d_v = up(at(v, ov), h.tok_v, ss),
             *d_f = up(at(f, okk), h.tok_k, ss), *d_bx = up(at(bx, okk), h.tok_k, ss), *d_wx = up(at(wx, ov), h.tok_v, ss),
             *d_beta = up(at(beta, o1), h.tok_1, ss);
        float* d_S0 = (float*)up(at(S0, os), h.st, ss);
        // the cotangents go up with the inputs: queued behind the forward they would hold the copy engine's queue
        void* d_dO = with_bwd ? up(at(dO, ov), h.tok_v, ss) : nullptr;
        float* d_dSf = with_bwd ? (float*)up(at(dS_final, os), h.st, ss) : nullptr;
        if (ns > 1) ok = ok && cudaEventRecord(arrived[i], ss) == cudaSuccess;
        void* d_O = slot(h.tok_v);
        float* d_Sf = (float*)slot(h.st);
        void* d_ws = nullptr;
        size_t ws_bytes = 0;
        if (with_bwd) {
            ws_bytes = carve_workspace_bytes(&ps, 1);
            d_ws = slot(ws_bytes);
        }
        if (!ok) break;
        rs = carve_fwd(&ps, d_q, d_k, d_v, d_f, d_bx, d_wx, d_beta, d_A, d_tau, d_Ub, d_Uw, d_Vb, d_Vw, d_S0, d_O, d_Sf,
                       d_ws, ws_bytes, ss);
        if (rs != CARVE_OK) break;
        if (with_bwd) {
            void *d_dq = slot(h.tok_k), *d_dk = slot(h.tok_k), *d_df = slot(h.tok_k), *d_dbx = slot(h.tok_k),
                 *d_dv = slot(h.tok_v), *d_dwx = slot(h.tok_v), *d_dbeta = slot(h.tok_1);
            float* d_dS0 = (float*)slot(h.st);
            float* wp = (float*)slot(nwg * 4);
            float *d_dA = wp, *d_dtau = d_dA + (size_t)p->H * p->dk, *d_dUb = d_dtau + (size_t)p->H * p->dk,
                  *d_dUw = d_dUb + (size_t)p->r * p->dv, *d_dVb = d_dUw + (size_t)p->r * p->dv,
                  *d_dVw = d_dVb + (size_t)p->dk * p->r;
            if (!ok) break;
            rs = bwd_impl(&ps, d_q, d_k, d_v, d_f, d_bx, d_wx, d_beta, d_A, d_tau, d_Ub, d_Uw, d_Vb, d_Vw, d_S0, d_dO,
                          d_dSf, d_dq, d_dk, d_dv, d_df, d_dbx, d_dwx, d_dbeta, d_dA, d_dtau, d_dUb, d_dUw, d_dVb,
                          d_dVw, d_dS0, d_ws, ws_bytes, ss, ns > 1);
            if (rs != CARVE_OK) break;
            down(atw(dq, okk), d_dq, h.tok_k, ss); down(atw(dk, okk), d_dk, h.tok_k, ss);
            down(atw(df, okk), d_df, h.tok_k, ss); down(atw(dbx, okk), d_dbx, h.tok_k, ss);
            down(atw(dv, ov), d_dv, h.tok_v, ss); down(atw(dwx, ov), d_dwx, h.tok_v, ss);
            down(atw(dbeta, o1), d_dbeta, h.tok_1, ss); down(atw(dS0, os), d_dS0, h.st, ss);
            if (i == 0) d_wpart = wp;
            if (i == 1) wpart_stride = (size_t)((char*)wp - (char*)d_wpart) / 4;
        }
        // after the backward: a download between the two calls would make carve_bwd wait for the copy engine's queue
        down(atw(O, ov), d_O, h.tok_v, ss);
        down(atw(S_final, os), d_Sf, h.st, ss);
    }
    // join: the caller's stream continues after every slice has finished
    for (int i = 0; i < ns; ++i) {
        if (ns > 1 && side[i] && join[i]) {
            ok = cudaEventRecord(join[i], side[i]) == cudaSuccess && ok;
            ok = cudaStreamWaitEvent(st, join[i], 0) == cudaSuccess && ok;
        }
    }
    if (with_bwd && ok && rs == CARVE_OK) {
        carve_sum_slices_kernel<<<(unsigned)((nwg + 255) / 256), 256, 0, st>>>(d_wsum, d_wpart, (int)nwg, ns, wpart_stride);
        ok = ok && cudaGetLastError() == cudaSuccess;
        const float* w = d_wsum;
        down(dA, w, h.w_a, st); w += (size_t)p->H * p->dk;
        down(dtau, w, h.w_a, st); w += (size_t)p->H * p->dk;
        down(dUb, w, h.w_u, st); w += (size_t)p->r * p->dv;
        down(dUw, w, h.w_u, st); w += (size_t)p->r * p->dv;
        down(dVb, w, h.w_vb, st); w += (size_t)p->dk * p->r;
        down(dVw, w, h.w_vw, st);
    }
    // (without a context) streams and events are released by the runtime once the work enqueued on them has completed
    if (!ctx) {
        for (int i = 0; i < ns; ++i) {
            if (ns > 1 && side[i]) cudaStreamDestroy(side[i]);
            if (join[i]) cudaEventDestroy(join[i]);
            if (arrived[i]) cudaEventDestroy(arrived[i]);
        }
        if (fork) cudaEventDestroy(fork);
    }
    if (rs != CARVE_OK) return rs;
    return ok ? CARVE_OK : CARVE_ERR_CUDA;
}

carve_status_t carve_fwd_bwd_host(const carve_params_t* p, int with_bwd, const void* q, const void* k,
                                  const void* v, const void* f, const void* bx, const void* wx, const void* beta,
                                  const float* A, const float* tau, const float* Ub, const float* Uw,
                                  const float* Vb, const float* Vw, const float* S0, void* O, float* S_final,
                                  const void* dO, const float* dS_final, void* dq, void* dk, void* dv, void* df,
                                  void* dbx, void* dwx, void* dbeta, float* dA, float* dtau, float* dUb,
                                  float* dUw, float* dVb, float* dVw, float* dS0, void* device_arena,
                                  size_t arena_bytes, void* cuda_stream)
{
    return host_impl(nullptr, p, with_bwd, q, k, v, f, bx, wx, beta, A, tau, Ub, Uw, Vb, Vw, S0, O, S_final, dO, dS_final, dq, dk, dv, df, dbx, dwx, dbeta, dA, dtau, dUb, dUw, dVb, dVw, dS0, device_arena, arena_bytes, cuda_stream);
}

carve_status_t carve_host_ctx_create(carve_host_ctx_t** out)
{
    if (!out) return CARVE_ERR_NULL;
    *out = nullptr;
    carve_host_ctx* c = new (std::nothrow) carve_host_ctx();
    if (!c) return CARVE_ERR_CUDA;
    bool ok = cudaEventCreateWithFlags(&c->fork, cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; i < 8; ++i) {
        ok = ok && cudaStreamCreateWithFlags(&c->side[i], cudaStreamNonBlocking) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&c->join[i], cudaEventDisableTiming) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&c->arrived[i], cudaEventDisableTiming) == cudaSuccess;
    }
    if (!ok) { carve_host_ctx_destroy(c); return CARVE_ERR_CUDA; }
    *out = c;
    return CARVE_OK;
}

void carve_host_ctx_destroy(carve_host_ctx_t* c)
{
    if (!c) return;
    for (int i = 0; i < 8; ++i) {
        if (c->side[i]) cudaStreamDestroy(c->side[i]);
        if (c->join[i]) cudaEventDestroy(c->join[i]);
        if (c->arrived[i]) cudaEventDestroy(c->arrived[i]);
    }
    if (c->fork) cudaEventDestroy(c->fork);
    delete c;
}

carve_status_t carve_fwd_bwd_host_ctx(carve_host_ctx_t* ctx, const carve_params_t* p, int with_bwd, const void* q, const void* k,
                                  const void* v, const void* f, const void* bx, const void* wx, const void* beta,
                                  const float* A, const float* tau, const float* Ub, const float* Uw,
                                  const float* Vb, const float* Vw, const float* S0, void* O, float* S_final,
                                  const void* dO, const float* dS_final, void* dq, void* dk, void* dv, void* df,
                                  void* dbx, void* dwx, void* dbeta, float* dA, float* dtau, float* dUb,
                                  float* dUw, float* dVb, float* dVw, float* dS0, void* device_arena,
                                  size_t arena_bytes, void* cuda_stream)
{
    return host_impl(ctx, p, with_bwd, q, k, v, f, bx, wx, beta, A, tau, Ub, Uw, Vb, Vw, S0, O, S_final, dO, dS_final, dq, dk, dv, df, dbx, dwx, dbeta, dA, dtau, dUb, dUw, dVb, dVw, dS0, device_arena, arena_bytes, cuda_stream);
}

}  // extern "C"

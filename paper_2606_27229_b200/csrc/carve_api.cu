// carve_api.cu -- the C ABI of include/carve.h: host-side validation, workspace carve-up,
// kernel-family selection and the host-buffer entry point.  No arithmetic of the method here.
#include <cstdio>
#include <cstring>

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
    if (!q || !k || !v || !f || !bx || !wx || !beta || !Ub || !Uw || !Vb || !Vw || !O || !S_final) return CARVE_ERR_NULL;
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

carve_status_t carve_bwd(const carve_params_t* p, const void* q, const void* k, const void* v, const void* f,
                         const void* bx, const void* wx, const void* beta, const float* A, const float* tau,
                         const float* Ub, const float* Uw, const float* Vb, const float* Vw, const float* S0,
                         const void* dO, const float* dS_final, void* dq, void* dk, void* dv, void* df, void* dbx,
                         void* dwx, void* dbeta, float* dA, float* dtau, float* dUb, float* dUw, float* dVb,
                         float* dVw, float* dS0, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    carve_status_t s = check_params(p, true);
    if (s != CARVE_OK) return s;
    if (!q || !k || !v || !f || !bx || !wx || !beta || !Ub || !Uw || !Vb || !Vw || !dO || !dq || !dk || !dv || !df ||
        !dbx || !dwx || !dbeta || !dUb || !dUw || !dVb || !dVw || !dS0)
        return CARVE_ERR_NULL;
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

// ---- host-buffer entry point ---------------------------------------------------------------------
namespace {
struct HostPlan {
    size_t tok_k, tok_v, tok_1, st, w_u, w_vb, w_vw, w_a;  // byte sizes
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
}  // namespace

size_t carve_host_arena_bytes(const carve_params_t* p, int with_bwd)
{
    if (check_params(p, with_bwd != 0) != CARVE_OK) return 0;
    const HostPlan h = plan_of(p);
    size_t n = 0;
    n += 4 * up256(h.tok_k) + 3 * up256(h.tok_v) + up256(h.tok_1);              // q,k,f,bx ; v,wx,O ; beta
    n += 2 * up256(h.w_a) + 2 * up256(h.w_u) + up256(h.w_vb) + up256(h.w_vw);   // A,tau,Ub,Uw,Vb,Vw
    n += 2 * up256(h.st);                                                        // S0, S_final
    if (with_bwd) {
        n += up256(h.tok_v) + up256(h.st);                                       // dO, dS_final
        n += 4 * up256(h.tok_k) + 2 * up256(h.tok_v) + up256(h.tok_1);          // dq,dk,df,dbx ; dv,dwx ; dbeta
        n += 2 * up256(h.w_a) + 2 * up256(h.w_u) + up256(h.w_vb) + up256(h.w_vw) + up256(h.st);
        n += up256(carve_workspace_bytes(p, 1));
    }
    return n;
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
    carve_status_t s = check_params(p, with_bwd != 0);
    if (s != CARVE_OK) return s;
    if (!device_arena || arena_bytes < carve_host_arena_bytes(p, with_bwd)) return CARVE_ERR_WORKSPACE;
    if (!aligned16(device_arena)) return CARVE_ERR_ALIGN;
    if (!q || !k || !v || !f || !bx || !wx || !beta || !Ub || !Uw || !Vb || !Vw || !O || !S_final) return CARVE_ERR_NULL;
    if (with_bwd && (!dO || !dq || !dk || !dv || !df || !dbx || !dwx || !dbeta || !dUb || !dUw || !dVb || !dVw || !dS0))
        return CARVE_ERR_NULL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const HostPlan h = plan_of(p);
    char* cur = static_cast<char*>(device_arena);
    bool ok = true;
    auto up = [&](const void* src, size_t bytes) -> void* {  // host -> device copy into the arena
        if (!src) return nullptr;
        void* d = cur;
        cur += up256(bytes);
        ok = ok && cudaMemcpyAsync(d, src, bytes, cudaMemcpyHostToDevice, st) == cudaSuccess;
        return d;
    };
    auto slot = [&](size_t bytes) -> void* { void* d = cur; cur += up256(bytes); return d; };

    void *d_q = up(q, h.tok_k), *d_k = up(k, h.tok_k), *d_v = up(v, h.tok_v), *d_f = up(f, h.tok_k),
         *d_bx = up(bx, h.tok_k), *d_wx = up(wx, h.tok_v), *d_beta = up(beta, h.tok_1);
    float *d_A = (float*)up(A, h.w_a), *d_tau = (float*)up(tau, h.w_a), *d_Ub = (float*)up(Ub, h.w_u),
          *d_Uw = (float*)up(Uw, h.w_u), *d_Vb = (float*)up(Vb, h.w_vb), *d_Vw = (float*)up(Vw, h.w_vw),
          *d_S0 = (float*)up(S0, h.st);
    void* d_O = slot(h.tok_v);
    float* d_Sf = (float*)slot(h.st);
    void* d_ws = nullptr;
    size_t ws_bytes = 0;
    if (with_bwd) {
        ws_bytes = carve_workspace_bytes(p, 1);
        d_ws = slot(ws_bytes);
    }
    if (!ok) return CARVE_ERR_CUDA;
    s = carve_fwd(p, d_q, d_k, d_v, d_f, d_bx, d_wx, d_beta, d_A, d_tau, d_Ub, d_Uw, d_Vb, d_Vw, d_S0, d_O, d_Sf,
                  d_ws, ws_bytes, cuda_stream);
    if (s != CARVE_OK) return s;
    auto down = [&](void* dst, const void* src, size_t bytes) {
        if (dst) ok = ok && cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, st) == cudaSuccess;
    };
    down(O, d_O, h.tok_v);
    down(S_final, d_Sf, h.st);
    if (with_bwd) {
        void* d_dO = up(dO, h.tok_v);
        float* d_dSf = (float*)up(dS_final, h.st);
        void *d_dq = slot(h.tok_k), *d_dk = slot(h.tok_k), *d_df = slot(h.tok_k), *d_dbx = slot(h.tok_k),
             *d_dv = slot(h.tok_v), *d_dwx = slot(h.tok_v), *d_dbeta = slot(h.tok_1);
        float *d_dA = dA ? (float*)slot(h.w_a) : nullptr, *d_dtau = dtau ? (float*)slot(h.w_a) : nullptr;
        float *d_dUb = (float*)slot(h.w_u), *d_dUw = (float*)slot(h.w_u), *d_dVb = (float*)slot(h.w_vb),
              *d_dVw = (float*)slot(h.w_vw), *d_dS0 = (float*)slot(h.st);
        if (!ok) return CARVE_ERR_CUDA;
        s = carve_bwd(p, d_q, d_k, d_v, d_f, d_bx, d_wx, d_beta, d_A, d_tau, d_Ub, d_Uw, d_Vb, d_Vw, d_S0, d_dO,
                      d_dSf, d_dq, d_dk, d_dv, d_df, d_dbx, d_dwx, d_dbeta, d_dA, d_dtau, d_dUb, d_dUw, d_dVb,
                      d_dVw, d_dS0, d_ws, ws_bytes, cuda_stream);
        if (s != CARVE_OK) return s;
        down(dq, d_dq, h.tok_k); down(dk, d_dk, h.tok_k); down(df, d_df, h.tok_k); down(dbx, d_dbx, h.tok_k);
        down(dv, d_dv, h.tok_v); down(dwx, d_dwx, h.tok_v); down(dbeta, d_dbeta, h.tok_1);
        down(dA, d_dA, h.w_a); down(dtau, d_dtau, h.w_a); down(dUb, d_dUb, h.w_u); down(dUw, d_dUw, h.w_u);
        down(dVb, d_dVb, h.w_vb); down(dVw, d_dVw, h.w_vw); down(dS0, d_dS0, h.st);
    }
    return ok ? CARVE_OK : CARVE_ERR_CUDA;
}

}  // extern "C"

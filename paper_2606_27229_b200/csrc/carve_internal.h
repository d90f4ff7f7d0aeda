// Internal declarations shared by the translation units of libcarve.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stddef.h>
#include <stdint.h>

#include "carve.h"

namespace carve {

// Everything a kernel needs, passed by value.
struct Args {
    int B, H, T, L, dk, dv, r;
    int l2norm;
    // tensor path, backward: launch the chunk-local epilogue as a plain dependent kernel.  The overlapped form
    // (an early grid that polls per-chain progress flags) fills every idle SM, which starves the chains of other
    // calls running beside this one (the batch slices of carve_fwd_bwd_host).
    bool epilogue_after = false;
    float scale, eps;
    // forward inputs
    const void *q, *k, *v, *f, *bx, *wx, *beta;
    const float *A, *tau, *Ub, *Uw, *Vb, *Vw, *S0;
    // forward outputs
    void* O;
    float* S_final;
    // backward inputs / outputs
    const void* dO;
    const float* dS_final;
    void *dq, *dk_, *dv_, *df, *dbx, *dwx, *dbeta;
    float* dS0;
    // workspace views (nullptr in inference forward)
    float* ws_states;  // [chains][T/LS][dv][dk]   state entering every solve sub-chunk
    float* ws_E;       // [B,T,H,dv]               pre-beta error e_t (u_t = beta_t e_t)
    float* ws_tt;      // [B,T,H,2r]               tanh bottleneck
    float* ws_G;       // [chains][T/L][2r][dk]    folded readout of every gate chunk
    float* ws_part;    // [chains][part_stride]    per-chain partial weight gradients
    int part_stride;
};

// Workspace layout (in floats) for the SIMT path; `total` in bytes.
struct WsLayout {
    size_t states, E, tt, G, part, total_bytes;
    int part_stride;
};

constexpr int kSimtSub = 16;  // solve sub-chunk of the SIMT path (tokens)

inline int part_stride_of(int dk, int dv, int r) { return 2 * r * dv + dk * r + dv * r + 2 * dk; }

inline WsLayout simt_ws_layout(const carve_params_t& p)
{
    WsLayout w{};
    const size_t chains = (size_t)p.B * p.H, tok = chains * p.T;
    size_t off = 0;
    auto take = [&](size_t n) { size_t o = off; off += (n + 3) & ~(size_t)3; return o; };
    w.states = take(chains * (p.T / kSimtSub) * p.dv * p.dk);
    w.E = take(tok * p.dv);
    w.tt = take(tok * 2 * p.r);
    w.G = take(chains * (p.T / p.L) * 2 * p.r * p.dk);
    w.part_stride = part_stride_of(p.dk, p.dv, p.r);
    w.part = take(chains * (size_t)w.part_stride);
    w.total_bytes = off * sizeof(float);
    return w;
}

// SIMT path (carve_simt.cu).  Return cudaSuccess or the failing CUDA error.
size_t simt_fwd_smem_bytes(int dk, int dv, int r);
size_t simt_bwd_smem_bytes(int dk, int dv, int r);
cudaError_t simt_fwd_launch(const Args& a, int dtype, cudaStream_t st);
cudaError_t simt_bwd_launch(const Args& a, int dtype, float* dA, float* dtau, float* dUb, float* dUw,
                            float* dVb, float* dVw, cudaStream_t st);

// Tensor-core path (carve_tc_fwd.cu, carve_tc_bwd.cu): bf16 tokens, dk == dv in {64,128}, r <= 16.
bool tc_fwd_supported(const carve_params_t& p);
bool tc_bwd_supported(const carve_params_t& p);
size_t tc_state_tile_bytes(const carve_params_t& p);
size_t tc_record_bytes(const carve_params_t& p);

// Workspace of the tensor path (byte offsets): chunk records, per-chain weight-gradient
// partials (layout of part_stride_of) and per-chunk dA/dtau partials.
struct TcWsLayout {
    size_t rec, part, partAT, dgs, flags, total_bytes;
    int part_stride;
};
inline TcWsLayout tc_ws_layout(const carve_params_t& p)
{
    TcWsLayout w{};
    const size_t chains = (size_t)p.B * p.H;
    const int LC = p.L < 64 ? p.L : 64;
    const size_t nchunks = p.T / LC;
    size_t off = 0;
    auto take = [&](size_t n) { size_t o = off; off += (n + 1023) & ~(size_t)1023; return o; };
    w.rec = take(chains * nchunks * tc_record_bytes(p));
    w.part_stride = part_stride_of(p.dk, p.dv, p.r);
    w.part = take(chains * (size_t)w.part_stride * sizeof(float));
    w.partAT = take(chains * nchunks * 2 * p.dk * sizeof(float));
    w.dgs = take(chains * (size_t)p.dk * 32 * sizeof(float));
    w.flags = take(chains * sizeof(int));   // chunks finished per chain (reverse kernel -> overlapped epilogue)
    w.total_bytes = off;
    return w;
}

// rec / sfin: workspace views (nullptr for an inference forward).
cudaError_t tc_fwd_launch(const Args& a, uint8_t* rec, cudaStream_t st);
cudaError_t tc_bwd_launch(const Args& a, uint8_t* ws, const TcWsLayout& w, float* dA, float* dtau, float* dUb,
                          float* dUw, float* dVb, float* dVw, cudaStream_t st);

// Recurrent step (carve_step.cu): n <= 16 new tokens per chain, state in place.
bool step_supported(int dk, int dv);
// layer ends (carve_layer_ends.cu)
cudaError_t silu_qkv_launch(const carve_params_t& p, const void* qx, const void* kx, const void* vx, void* q, void* k, void* v,
                            bool bwd, cudaStream_t st);
bool out_norm_supported(const carve_params_t& p);
size_t out_norm_ws_bytes(const carve_params_t& p);
cudaError_t out_norm_launch(const carve_params_t& p, bool bwd, const void* o, const float* gain, float eps, const void* dy,
                            void* out, float* partial, float* dgain, cudaStream_t st);

cudaError_t step_launch(const carve_params_t& p, const void* q, const void* k, const void* v, const void* f, const void* bx,
                        const void* wx, const void* beta, const float* A, const float* tau, const float* Ub, const float* Uw,
                        const float* Vb, const float* Vw, float* S, void* O, const int* cu_seqlens, cudaStream_t st);

// Deterministic reduction of per-chain partials (carve_simt_bwd.cu), shared by both paths.
cudaError_t reduce_weights_launch(const float* part, int chains, int stride, int H, int dk, int dv, int r, float* dUb,
                                  float* dUw, float* dVb, float* dVw, float* dA, float* dtau, cudaStream_t st);

}  // namespace carve

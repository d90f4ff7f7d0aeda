// carve_step.cu -- the recurrent (decode) form of the CARVE layer operator: a few new tokens per sequence, state in
// and out (Table 1 l.432 "Infer/tok O(d_v d_k)", l.27; "chunk mode vs sequential at chunk size 1", l.450).
//
// The n <= 16 new tokens of a sequence form ONE gate chunk: the content gates read the incoming state once,
// G = [Ub;Uw] S (Eq. 7 l.134), and every token then applies Eq. 5 (l.108) in its per-token form with those gates:
//     a_t = exp(g_t) (1 - b_t),   e_t = w_t . v_t - S_{t-1} k^_t,   u_t = beta_t e_t,
//     S_t = S_{t-1} diag(a_t) + u_t k^_t^T,   o_t = scale S_t q^_t.
// With n = 1 this is exact per-token content gating.  It is the same function as carve_fwd with T = L = n (the chunked
// WY form equals this recurrence), evaluated without the solve because n is small.
//
// Ragged batches (carve_step_varlen): the token tensors are packed [total_tokens, H, d] and sequence b owns the rows
// cu_seqlens[b] .. cu_seqlens[b+1] (0..T tokens each; the variable-length batches of SURVEY 8(f) NEXT-1).
//
// One CTA per (batch, head) chain; the state makes one round trip HBM -> shared memory -> HBM per call, which is the
// algorithmic traffic of a decode step (2 x 4 d_v d_k bytes per chain).  fp32 arithmetic throughout, plain FFMA.
#include "simt_common.cuh"

namespace carve {
namespace {

struct StepArgs {
    int B, H, n, r, l2norm;
    float scale, eps;
    const void *q, *k, *v, *f, *bx, *wx, *beta;
    const float *A, *tau, *Ub, *Uw, *Vb, *Vw;
    float* S;
    void* O;
    const int* cu;   // ragged batch: tokens of sequence b are rows cu[b] .. cu[b+1] of the packed token tensors (else NULL)
};

template <typename T, int DK, int DV>
__global__ void __launch_bounds__(NT, 1) carve_step_kernel(const StepArgs a)
{
    extern __shared__ __align__(16) float smem[];
    constexpr int SP = DK + 4;
    const int r = a.r, R2 = 2 * r;
    float* sS = smem;                  // [DV][SP]
    float* sG = sS + DV * SP;          // [R2][SP]
    float* sQ = sG + R2 * SP;          // [DK] q^
    float* sK = sQ + DK;               // [DK] k^
    float* sA = sK + DK;               // [DK] a_t
    float* sU = sA + DK;               // [DV] u_t
    float* sW = sU + DV;               // [DV] w_t v_t
    float* sT = sW + DV;               // [R2] tanh bottleneck
    float* sRed = sT + 64;             // [2] 1/|q|, 1/|k|;  [2..3] the state load's mbarrier;  [4] beta of the token

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int chain = blockIdx.x, b = chain / a.H, h = chain % a.H;
    const T* gq = static_cast<const T*>(a.q);
    const T* gk = static_cast<const T*>(a.k);
    const T* gv = static_cast<const T*>(a.v);
    const T* gf = static_cast<const T*>(a.f);
    const T* gbx = static_cast<const T*>(a.bx);
    const T* gwx = static_cast<const T*>(a.wx);
    const T* gbeta = static_cast<const T*>(a.beta);
    T* gO = static_cast<T*>(a.O);
    float* gS = a.S + (size_t)chain * DV * DK;
    // tokens of this sequence: rows tok0 .. tok0 + n of the [tokens, H, d] tensors (ragged: from cu_seqlens, clamped to the
    // declared maximum; a sequence without new tokens leaves its state untouched)
    const int tok0 = a.cu ? __ldg(a.cu + b) : b * a.n;
    const int n = a.cu ? min(max(__ldg(a.cu + b + 1) - tok0, 0), a.n) : a.n;
    if (n == 0) return;

    // The state comes in by bulk copies, one per row (the rows are padded in shared memory), all in flight at once and
    // asynchronous: the staging of Ucat^T and of the first token's inputs below runs under them.  (As per-thread loads
    // the 64 KB cost a chain of load round trips per thread; ncu: 5.2 long-scoreboard stalls per issue, 11 % of the DRAM peak.)
    uint64_t* sbar = reinterpret_cast<uint64_t*>(sRed + 2);
    const uint32_t sbar_a = (uint32_t)__cvta_generic_to_shared(sbar);
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(sbar_a));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(sbar_a), "r"((uint32_t)(DV * DK * 4)) : "memory");
    }
    __syncthreads();
    for (int x = tid; x < DV; x += NT)
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"((uint32_t)__cvta_generic_to_shared(sS + x * SP)), "l"(gS + (size_t)x * DK), "r"((uint32_t)(DK * 4)), "r"(sbar_a)
                     : "memory");
    // fold: G[i][j] = sum_x Ucat[i][x] S[x][j]   (once per call: the gates of all n tokens read the incoming state).
    // Ucat^T is staged in shared memory ([x][i]); a thread owns one key channel j and 8 bottleneck rows, so that one
    // state read feeds 8 FMAs (the first version read the state once per FMA and was 2.2x slower end to end).
    float* sUt = sRed + 8;             // [DV][RP], RP = R2 + 4: the transposing stores below hit 8 banks instead of one
    const int RP = R2 + 4;
    // (16-byte loads, four in flight per thread: as one scalar load per loop trip this staging was 17 % of the kernel)
    for (int o0 = tid; o0 < R2 * DV / 4; o0 += 4 * NT) {
        float4 u4[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int o = o0 + u * NT, i = o / (DV / 4), x4 = o % (DV / 4);
            u4[u] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (o < R2 * DV / 4) {
                if (i < r) u4[u] = ldg4(a.Ub + (size_t)i * DV + 4 * x4);
                else if (a.Uw) u4[u] = ldg4(a.Uw + (size_t)(i - r) * DV + 4 * x4);
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int o = o0 + u * NT, i = o / (DV / 4), x4 = o % (DV / 4);
            if (o < R2 * DV / 4) {
                sUt[(4 * x4 + 0) * RP + i] = u4[u].x; sUt[(4 * x4 + 1) * RP + i] = u4[u].y;
                sUt[(4 * x4 + 2) * RP + i] = u4[u].z; sUt[(4 * x4 + 3) * RP + i] = u4[u].w;
            }
        }
    }
    // token inputs are staged in shared memory one token ahead of their use: all of a token's loads are in flight together
    // (q, k, f, bx: DK each; v, wx: DV each), instead of one exposed load round trip in each of the six phases of a token
    float* sIn = sUt + DV * RP;        // [4 DK + 2 DV]: q | k | f | bx | v | wx (raw)
    constexpr int NIN = (4 * DK + 2 * DV + NT - 1) / NT;   // staged values per thread
    float in_r[NIN], beta_r = 0.f;
    auto load_token = [&](int t2) {   // global loads of token t2 into registers (all in flight together)
        const size_t tok2 = ((size_t)tok0 + t2) * a.H + h;
#pragma unroll
        for (int u = 0; u < NIN; ++u) {
            const int j = tid + u * NT;
            float vv = 0.f;
            if (j < DK) vv = ldf<T>(gq, tok2 * DK + j);
            else if (j < 2 * DK) vv = ldf<T>(gk, tok2 * DK + (j - DK));
            else if (j < 3 * DK) vv = ldf<T>(gf, tok2 * DK + (j - 2 * DK));
            else if (j < 4 * DK) vv = ldf<T>(gbx, tok2 * DK + (j - 3 * DK));
            else if (j < 4 * DK + DV) vv = ldf<T>(gv, tok2 * DV + (j - 4 * DK));
            else if (j < 4 * DK + 2 * DV) vv = gwx ? ldf<T>(gwx, tok2 * DV + (j - 4 * DK - DV)) : 0.f;
            in_r[u] = vv;
        }
        if (tid == 0) beta_r = ldf<T>(gbeta, tok2);
    };
    auto store_token = [&]() {
#pragma unroll
        for (int u = 0; u < NIN; ++u) {
            const int j = tid + u * NT;
            if (j < 4 * DK + 2 * DV) sIn[j] = in_r[u];
        }
        if (tid == 0) sRed[4] = beta_r;
    };
    load_token(0);
    store_token();
    // wait for the state
    {
        uint32_t done = 0;
        while (!done)
            asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                         : "=r"(done) : "r"(sbar_a) : "memory");
    }
    __syncthreads();
    // a thread owns two key channels (j, j + DK/2) and 8 bottleneck rows: 16 FMAs per two state reads and two broadcast
    // 16-byte reads of Ucat^T (the loop is bound by shared-memory instructions, not by the FMA pipe)
    for (int o = tid; o < (DK / 2) * (R2 / 8); o += NT) {
        const int j = o % (DK / 2), i0 = 8 * (o / (DK / 2));
        float acc[2][8];
#pragma unroll
        for (int e = 0; e < 8; ++e) acc[0][e] = acc[1][e] = 0.f;
#pragma unroll 8
        for (int x = 0; x < DV; ++x) {
            const float s0 = sS[x * SP + j], s1 = sS[x * SP + j + DK / 2];
            const float4 u0 = ld4s(sUt + x * RP + i0), u1 = ld4s(sUt + x * RP + i0 + 4);
            const float uu[8] = {u0.x, u0.y, u0.z, u0.w, u1.x, u1.y, u1.z, u1.w};
#pragma unroll
            for (int e = 0; e < 8; ++e) { acc[0][e] = fmaf(uu[e], s0, acc[0][e]); acc[1][e] = fmaf(uu[e], s1, acc[1][e]); }
        }
#pragma unroll
        for (int e = 0; e < 8; ++e) { sG[(i0 + e) * SP + j] = acc[0][e]; sG[(i0 + e) * SP + j + DK / 2] = acc[1][e]; }
    }
    __syncthreads();

    for (int t = 0; t < n; ++t) {
        const size_t tok = ((size_t)tok0 + t) * a.H + h;
        const float *iq = sIn, *ik = sIn + DK, *if_ = sIn + 2 * DK, *ibx = sIn + 3 * DK, *iv = sIn + 4 * DK, *iwx = sIn + 4 * DK + DV;
        // q^, k^ (D1)
        if (warp < 2) {
            const float* src = warp == 0 ? iq : ik;
            float ss = 0.f;
            for (int j = lane; j < DK; j += 32) { const float x = src[j]; ss = fmaf(x, x, ss); }
            ss = warp_sum(ss);
            if (lane == 0) sRed[warp] = a.l2norm ? rsqrtf(ss + a.eps) : 1.f;
        }
        __syncthreads();
        for (int j = tid; j < 2 * DK; j += NT) {
            if (j < DK) sQ[j] = iq[j] * sRed[0];
            else sK[j - DK] = ik[j - DK] * sRed[1];
        }
        __syncthreads();
        // tt = tanh(G q^) (Eq. 7)
        for (int i = warp; i < R2; i += NT / 32) {
            float acc = 0.f;
            for (int j = lane; j < DK; j += 32) acc = fmaf(sG[i * SP + j], sQ[j], acc);
            acc = warp_sum(acc);
            if (lane == 0) sT[i] = tanhf(acc);
        }
        __syncthreads();
        // gates (Eq. 8-9): a_t = exp(g)(1 - b), w_t v_t
        for (int j = tid; j < DK + DV; j += NT) {
            if (j < DK) {
                float pre = ibx[j];
                for (int i = 0; i < r; ++i) pre = fmaf(__ldg(a.Vb + (size_t)j * r + i), sT[i], pre);
                const float eA = a.A ? expf(__ldg(a.A + h * DK + j)) : 1.f;
                const float ta = a.tau ? __ldg(a.tau + h * DK + j) : 0.f;
                const float g = -eA * softplusf(if_[j] + ta);
                sA[j] = expf(g - softplusf(pre));          // exp(g) (1 - sigmoid(pre)),  log(1 - sigmoid(x)) = -softplus(x)
            } else {
                const int x = j - DK;
                float w = 1.f;   // scalar-write variant (wx = NULL, P l.145)
                if (gwx) {
                    float pre = iwx[x];
                    for (int i = 0; i < r; ++i) pre = fmaf(__ldg(a.Vw + (size_t)x * r + i), sT[r + i], pre);
                    w = sigmoidf_(pre);
                }
                sW[x] = w * iv[x];
            }
        }
        __syncthreads();
        const float beta = sRed[4];
        if (t + 1 < n) load_token(t + 1);   // the next token's inputs: in flight under the two state phases below
        // u_t = beta (w v - S k^): two threads per state row, half of the key channels each
        for (int p = tid; p < 2 * DV; p += NT) {
            const int x = p >> 1, hf = p & 1;
            const float* srow = sS + x * SP + hf * (DK / 2);
            const float* kk = sK + hf * (DK / 2);
            float acc = 0.f;
#pragma unroll 4
            for (int j = 0; j < DK / 2; j += 4) acc += dot4(ld4s(srow + j), ld4s(kk + j));
            acc += __shfl_xor_sync(0xffffffffu, acc, 1);
            if (hf == 0) sU[x] = beta * (sW[x] - acc);
        }
        __syncthreads();
        // S_t = S diag(a) + u k^^T;  o_t = scale S_t q^
        for (int p = tid; p < 2 * DV; p += NT) {
            const int x = p >> 1, hf = p & 1;
            float* srow = sS + x * SP + hf * (DK / 2);
            const float* kk = sK + hf * (DK / 2);
            const float* qq = sQ + hf * (DK / 2);
            const float* aa = sA + hf * (DK / 2);
            const float u = sU[x];
            float acc = 0.f;
#pragma unroll 4
            for (int j = 0; j < DK / 2; j += 4) {
                float4 s4 = ld4s(srow + j);
                const float4 a4 = ld4s(aa + j), k4 = ld4s(kk + j);
                s4.x = fmaf(s4.x, a4.x, u * k4.x); s4.y = fmaf(s4.y, a4.y, u * k4.y);
                s4.z = fmaf(s4.z, a4.z, u * k4.z); s4.w = fmaf(s4.w, a4.w, u * k4.w);
                st4s(srow + j, s4);
                acc += dot4(s4, ld4s(qq + j));
            }
            acc += __shfl_xor_sync(0xffffffffu, acc, 1);
            if (hf == 0) stf<T>(gO, tok * DV + x, a.scale * acc);
        }
        if (t + 1 < n) store_token();
        __syncthreads();
    }
    for (int i = tid; i < DV * DK / 4; i += NT) {
        const int x = i / (DK / 4), j4 = i % (DK / 4);
        *reinterpret_cast<float4*>(gS + (size_t)i * 4) = ld4s(sS + x * SP + 4 * j4);
    }
}

template <typename T, int DK, int DV>
cudaError_t launch_step(const StepArgs& a, cudaStream_t st)
{
    const size_t smem = ((size_t)(DV + 2 * a.r) * (DK + 4) + 3 * DK + 2 * DV + 64 + 8 + (size_t)DV * (2 * a.r + 4) + 4 * DK + 2 * DV) * sizeof(float);
    auto kern = carve_step_kernel<T, DK, DV>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<a.B * a.H, NT, smem, st>>>(a);
    return cudaGetLastError();
}

template <typename T>
cudaError_t dispatch_step(const StepArgs& a, int dk, int dv, cudaStream_t st)
{
    if (dk == 64 && dv == 64) return launch_step<T, 64, 64>(a, st);
    if (dk == 128 && dv == 128) return launch_step<T, 128, 128>(a, st);
    if (dk == 64 && dv == 128) return launch_step<T, 64, 128>(a, st);
    if (dk == 128 && dv == 64) return launch_step<T, 128, 64>(a, st);
    if (dk == 128 && dv == 256) return launch_step<T, 128, 256>(a, st);
    return cudaErrorInvalidValue;
}

}  // namespace

bool step_supported(int dk, int dv)
{
    return (dk == 64 || dk == 128) && (dv == 64 || dv == 128 || (dk == 128 && dv == 256));
}

cudaError_t step_launch(const carve_params_t& p, const void* q, const void* k, const void* v, const void* f, const void* bx,
                        const void* wx, const void* beta, const float* A, const float* tau, const float* Ub, const float* Uw,
                        const float* Vb, const float* Vw, float* S, void* O, const int* cu_seqlens, cudaStream_t st)
{
    StepArgs a{};
    a.cu = cu_seqlens;
    a.B = p.B; a.H = p.H; a.n = p.T; a.r = p.r; a.l2norm = p.qk_l2norm; a.scale = p.scale; a.eps = p.eps;
    a.q = q; a.k = k; a.v = v; a.f = f; a.bx = bx; a.wx = wx; a.beta = beta;
    a.A = A; a.tau = tau; a.Ub = Ub; a.Uw = Uw; a.Vb = Vb; a.Vw = Vw; a.S = S; a.O = O;
    return p.dtype == CARVE_BF16 ? dispatch_step<__nv_bfloat16>(a, p.dk, p.dv, st) : dispatch_step<float>(a, p.dk, p.dv, st);
}

}  // namespace carve

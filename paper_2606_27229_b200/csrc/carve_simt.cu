// carve_simt.cu -- fp32 SIMT path of the CARVE layer operator (forward).
//
// One CTA per (batch, head) chain, persistent over the whole sequence; the d_v x d_k fp32 state
// lives in shared memory and never leaves the SM between chunks.  The intra-chunk WY solve is done
// on solve sub-chunks of kSimtSub = 16 tokens: inside a gate chunk of L tokens the gates are frozen
// (they read G_c = [U_b;U_w] S_{c-1}, Eq. 7 l.134), so running Alg. 2 (l.315-365) on
// 16-token pieces that hand the state to each other is the same recurrence (Eq. 5 l.108) and the
// same function of the inputs; only the fold G_c is refreshed every L tokens.  All decay ratios are
// formed pairwise in log space, exp(lg_t - lg_s) with s <= t, so no exponent is ever positive
// (gamma_{L-1} reaches e^-100 on the paper-shaped inputs and 1/gamma is never formed).
//
// This is the correctness anchor of the library and the only path for CARVE_F32 inputs (fp32
// FFMA keeps the 1e-4 tolerance; tensor cores would need TF32).
#include "simt_common.cuh"

namespace carve {
namespace {

// Shared-memory carve-up of the forward kernel, in floats.
struct FwdSmem {
    int S, Qh, Kh, Lg, Kbar, Qbar, Ktil, U, G, Tt, A, P, Gam, Beta, total;
    __host__ __device__ FwdSmem(int dk, int dv, int r)
    {
        const int SP = dk + 4, R2 = 2 * r;
        int o = 0;
        S = o;    o += dv * SP;
        Qh = o;   o += SC * dk;
        Kh = o;   o += SC * dk;
        Lg = o;   o += SC * dk;
        Kbar = o; o += SC * dk;
        Qbar = o; o += SC * dk;
        Ktil = o; o += SC * dk;
        U = o;    o += SC * dv;
        G = o;    o += R2 * SP;
        Tt = o;   o += SC * R2;
        A = o;    o += SC * AP;
        P = o;    o += SC * AP;
        Gam = o;  o += dk;
        Beta = o; o += SC;
        total = o;
    }
};

// ------------------------------------------------------------------------------------------------
// Forward.  Phases of one 16-token solve sub-chunk (the numbering is used in DESIGN.md):
//   F0 checkpoint S (if saving) and, at a gate-chunk start, fold G = [Ub;Uw] S          (Eq. 7)
//   F1 load q,k; L2-normalise                                                           (D1)
//   F2 tt = tanh(q^ G^T)                                                                (Eq. 7)
//   F3 la = g - softplus(bx + Vb tt_b)  [= log a_t];  V' = sigmoid(wx + Vw tt_w) . v    (Eq. 8-9)
//   F4 lg = cumsum_t(la) (Eq. 14);  Kbar = k^ e^{lg_{t-1}}, Qbar = q^ e^{lg_t}, Ktil = k^ e^{lg_L - lg_t}
//   F5 R = V' - Kbar S^T ;  Oi = Qbar S^T (registers)                                   (Alg. 2 step 5)
//   F6 pairwise W_ts = e^{lg_t - lg_s}: P_ts = sum_j q^_t k^_s W_ts, A_{t+1,s} = sum_j k^_{t+1} k^_s W_ts  (Eq. 15)
//   F7 forward substitution e_t = R_t - sum_{s<t} A_ts u_s, u_t = beta_t e_t             (Alg. 2 step 7)
//   F8 O = scale (Oi + P U) (step 8);  S <- S diag(gamma_L) + U^T Ktil (step 9)
// ------------------------------------------------------------------------------------------------
template <typename T, int DK, int DV>
__global__ void __launch_bounds__(NT, 1) carve_fwd_simt_kernel(const Args a)
{
    extern __shared__ __align__(16) float smem[];
    constexpr int SP = DK + 4;
    const int r = a.r, R2 = 2 * r;
    const FwdSmem L_(DK, DV, r);
    float* sS = smem + L_.S;
    float* sQh = smem + L_.Qh;
    float* sKh = smem + L_.Kh;
    float* sLg = smem + L_.Lg;
    float* sKbar = smem + L_.Kbar;
    float* sQbar = smem + L_.Qbar;
    float* sKtil = smem + L_.Ktil;
    float* sU = smem + L_.U;
    float* sG = smem + L_.G;
    float* sT = smem + L_.Tt;
    float* sA = smem + L_.A;
    float* sP = smem + L_.P;
    float* sGam = smem + L_.Gam;
    float* sBeta = smem + L_.Beta;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int chain = blockIdx.x, b = chain / a.H, h = chain % a.H;
    const int nchunks = a.T / SC, nsub = a.L / SC;
    const T* gq = static_cast<const T*>(a.q);
    const T* gk = static_cast<const T*>(a.k);
    const T* gv = static_cast<const T*>(a.v);
    const T* gf = static_cast<const T*>(a.f);
    const T* gbx = static_cast<const T*>(a.bx);
    const T* gwx = static_cast<const T*>(a.wx);
    const T* gbeta = static_cast<const T*>(a.beta);
    T* gO = static_cast<T*>(a.O);
    auto tokoff = [&](int t) -> size_t { return ((size_t)b * a.T + t) * a.H + h; };

    // initial state
    for (int i = tid; i < DV * DK / 4; i += NT) {
        const int x = i / (DK / 4), j4 = i % (DK / 4);
        float4 v4 = make_float4(0.f, 0.f, 0.f, 0.f);
        if (a.S0) v4 = ldg4(a.S0 + (size_t)chain * DV * DK + (size_t)i * 4);
        st4s(sS + x * SP + 4 * j4, v4);
    }
    __syncthreads();

    constexpr int TPT = SC * DV / NT;  // tokens per thread in the token x state products
    constexpr int JR = DK * DV / NT;   // state columns per thread in the state update

    for (int c = 0; c < nchunks; ++c) {
        const int t0 = c * SC;
        // ---- F0: checkpoint + fold
        if (a.ws_states) {
            float* dst = a.ws_states + ((size_t)chain * nchunks + c) * DV * DK;
            for (int i = tid; i < DV * DK / 4; i += NT) {
                const int x = i / (DK / 4), j4 = i % (DK / 4);
                st4s(dst + (size_t)i * 4, ld4s(sS + x * SP + 4 * j4));
            }
        }
        if (c % nsub == 0) {
            for (int it = tid; it < (DK / 4) * (R2 / 4); it += NT) {
                const int j4 = it % (DK / 4), ib = it / (DK / 4);
                float4 acc[4];
#pragma unroll
                for (int ii = 0; ii < 4; ++ii) acc[ii] = make_float4(0.f, 0.f, 0.f, 0.f);
                const float* Urow[4];
#pragma unroll
                for (int ii = 0; ii < 4; ++ii) {
                    const int i = 4 * ib + ii;
                    Urow[ii] = (i < r) ? a.Ub + (size_t)i * DV : (a.Uw ? a.Uw + (size_t)(i - r) * DV : nullptr);
                }
                for (int x = 0; x < DV; x += 4) {
                    const float4 s0 = ld4s(sS + (x + 0) * SP + 4 * j4), s1 = ld4s(sS + (x + 1) * SP + 4 * j4),
                                 s2 = ld4s(sS + (x + 2) * SP + 4 * j4), s3 = ld4s(sS + (x + 3) * SP + 4 * j4);
#pragma unroll
                    for (int ii = 0; ii < 4; ++ii) {
                        const float4 u = Urow[ii] ? ldg4(Urow[ii] + x) : make_float4(0.f, 0.f, 0.f, 0.f);   // scalar-write variant: no Uw
                        acc[ii].x += u.x * s0.x + u.y * s1.x + u.z * s2.x + u.w * s3.x;
                        acc[ii].y += u.x * s0.y + u.y * s1.y + u.z * s2.y + u.w * s3.y;
                        acc[ii].z += u.x * s0.z + u.y * s1.z + u.z * s2.z + u.w * s3.z;
                        acc[ii].w += u.x * s0.w + u.y * s1.w + u.z * s2.w + u.w * s3.w;
                    }
                }
#pragma unroll
                for (int ii = 0; ii < 4; ++ii) {
                    st4s(sG + (4 * ib + ii) * SP + 4 * j4, acc[ii]);
                    if (a.ws_G)
                        st4s(a.ws_G + (((size_t)chain * (a.T / a.L) + c / nsub) * R2 + 4 * ib + ii) * DK + 4 * j4,
                             acc[ii]);
                }
            }
        }
        // ---- F1: load q,k rows, L2-normalise
        for (int t = warp; t < SC; t += NT / 32) {
            const size_t ro = tokoff(t0 + t) * DK;
            float qv[DK / 32], kv[DK / 32];
            float sq = 0.f, sk = 0.f;
#pragma unroll
            for (int e = 0; e < DK / 32; ++e) {
                qv[e] = ldf(gq, ro + lane + 32 * e);
                kv[e] = ldf(gk, ro + lane + 32 * e);
                sq += qv[e] * qv[e];
                sk += kv[e] * kv[e];
            }
            sq = warp_sum(sq);
            sk = warp_sum(sk);
            const float rq = a.l2norm ? 1.f / sqrtf(sq + a.eps) : 1.f;
            const float rk = a.l2norm ? 1.f / sqrtf(sk + a.eps) : 1.f;
#pragma unroll
            for (int e = 0; e < DK / 32; ++e) {
                sQh[t * DK + lane + 32 * e] = qv[e] * rq;
                sKh[t * DK + lane + 32 * e] = kv[e] * rk;
            }
        }
        if (tid < SC) sBeta[tid] = ldf(gbeta, tokoff(t0 + tid));
        __syncthreads();
        // ---- F2: bottleneck tt = tanh(q^ G^T)
        for (int it = tid; it < R2 * (SC / 2); it += NT) {
            const int i = it % R2, tp = it / R2;
            float a0 = 0.f, a1 = 0.f;
            for (int j4 = 0; j4 < DK / 4; ++j4) {
                const float4 g4 = ld4s(sG + i * SP + 4 * j4);
                a0 += dot4(g4, ld4s(sQh + (2 * tp) * DK + 4 * j4));
                a1 += dot4(g4, ld4s(sQh + (2 * tp + 1) * DK + 4 * j4));
            }
            a0 = tanhf(a0);
            a1 = tanhf(a1);
            sT[(2 * tp) * R2 + i] = a0;
            sT[(2 * tp + 1) * R2 + i] = a1;
            if (a.ws_tt) {
                a.ws_tt[tokoff(t0 + 2 * tp) * R2 + i] = a0;
                a.ws_tt[tokoff(t0 + 2 * tp + 1) * R2 + i] = a1;
            }
        }
        __syncthreads();
        // ---- F3: gates.  la = log a_t = g_t - softplus(b_pre);  V' = w . v
        for (int it = tid; it < SC * DK; it += NT) {
            const int j = it % DK, t = it / DK;
            const size_t go = tokoff(t0 + t) * DK + j;
            float bp = ldf(gbx, go);
            for (int i4 = 0; i4 < r / 4; ++i4)
                bp += dot4(ldg4(a.Vb + (size_t)j * r + 4 * i4), ld4s(sT + t * R2 + 4 * i4));
            const float eA = a.A ? expf(__ldg(a.A + h * DK + j)) : 1.f;
            const float ta = a.tau ? __ldg(a.tau + h * DK + j) : 0.f;
            const float g = -eA * softplusf(ldf(gf, go) + ta);
            sLg[t * DK + j] = g - softplusf(bp);
        }
        for (int it = tid; it < SC * DV; it += NT) {
            const int x = it % DV, t = it / DV;
            const size_t go = tokoff(t0 + t) * DV + x;
            float w = 1.f;   // scalar-write variant (wx = NULL, P l.145): the write gate is the scalar already in beta
            if (gwx) {
                float wp = ldf(gwx, go);
                for (int i4 = 0; i4 < r / 4; ++i4)
                    wp += dot4(ldg4(a.Vw + (size_t)x * r + 4 * i4), ld4s(sT + t * R2 + r + 4 * i4));
                w = sigmoidf_(wp);
            }
            sU[t * DV + x] = w * ldf(gv, go);
        }
        __syncthreads();
        // ---- F4: retention prefix (Eq. 14) and the decayed operands
        if (tid < DK) {
            float run = 0.f;
#pragma unroll
            for (int t = 0; t < SC; ++t) {
                run += sLg[t * DK + tid];
                sLg[t * DK + tid] = run;
            }
            sGam[tid] = expf(run);
        }
        __syncthreads();
        for (int it = tid; it < SC * DK; it += NT) {
            const int j = it % DK, t = it / DK;
            const float lg = sLg[t * DK + j], lgm1 = t ? sLg[(t - 1) * DK + j] : 0.f, lgL = sLg[(SC - 1) * DK + j];
            const float kh = sKh[t * DK + j];
            sKbar[t * DK + j] = kh * expf(lgm1);
            sQbar[t * DK + j] = sQh[t * DK + j] * expf(lg);
            sKtil[t * DK + j] = kh * expf(lgL - lg);
        }
        __syncthreads();
        // ---- F5: R = V' - Kbar S^T,  Oi = Qbar S^T
        const int px = tid % DV, ptg = tid / DV;
        float accO[TPT];
        {
            float accR[TPT];
#pragma unroll
            for (int u = 0; u < TPT; ++u) accR[u] = accO[u] = 0.f;
            for (int j4 = 0; j4 < DK / 4; ++j4) {
                const float4 s4 = ld4s(sS + px * SP + 4 * j4);
#pragma unroll
                for (int u = 0; u < TPT; ++u) {
                    accR[u] += dot4(ld4s(sKbar + (ptg * TPT + u) * DK + 4 * j4), s4);
                    accO[u] += dot4(ld4s(sQbar + (ptg * TPT + u) * DK + 4 * j4), s4);
                }
            }
#pragma unroll
            for (int u = 0; u < TPT; ++u) sU[(ptg * TPT + u) * DV + px] -= accR[u];
        }
        // ---- F6: pairwise coupling / output matrices, one warp per (t,s), s <= t
        {
            int cnt = 0;
            for (int t = 0; t < SC; ++t)
                for (int s = 0; s <= t; ++s, ++cnt) {
                    if ((cnt & (NT / 32 - 1)) != warp) continue;
                    float pa = 0.f, pp = 0.f;
                    for (int j = lane; j < DK; j += 32) {
                        const float w = expf(sLg[t * DK + j] - sLg[s * DK + j]);
                        const float ks = sKh[s * DK + j] * w;
                        pp += sQh[t * DK + j] * ks;
                        if (t + 1 < SC) pa += sKh[(t + 1) * DK + j] * ks;
                    }
                    pp = warp_sum(pp);
                    pa = warp_sum(pa);
                    if (lane == 0) {
                        sP[t * AP + s] = pp;
                        if (t + 1 < SC) sA[(t + 1) * AP + s] = pa;
                    }
                }
        }
        __syncthreads();
        // ---- F7: forward substitution, one thread per value channel
        if (tid < DV) {
            float u[SC];
#pragma unroll
            for (int t = 0; t < SC; ++t) {
                float e = sU[t * DV + tid];
#pragma unroll
                for (int s = 0; s < t; ++s) e -= sA[t * AP + s] * u[s];
                if (a.ws_E) a.ws_E[tokoff(t0 + t) * DV + tid] = e;
                u[t] = sBeta[t] * e;
                sU[t * DV + tid] = u[t];
            }
        }
        __syncthreads();
        // ---- F8: outputs and state carry
#pragma unroll
        for (int u = 0; u < TPT; ++u) {
            const int t = ptg * TPT + u;
            float o = accO[u];
            for (int s = 0; s <= t; ++s) o += sP[t * AP + s] * sU[s * DV + px];
            stf(gO, tokoff(t0 + t) * DV + px, a.scale * o);
        }
        {
            float u[SC];
#pragma unroll
            for (int t = 0; t < SC; ++t) u[t] = sU[t * DV + px];
            for (int j4 = ptg * (JR / 4); j4 < (ptg + 1) * (JR / 4); ++j4) {
                float4 s4 = ld4s(sS + px * SP + 4 * j4);
                const float4 g4 = ld4s(sGam + 4 * j4);
                s4.x *= g4.x; s4.y *= g4.y; s4.z *= g4.z; s4.w *= g4.w;
#pragma unroll
                for (int t = 0; t < SC; ++t) {
                    const float4 k4 = ld4s(sKtil + t * DK + 4 * j4);
                    s4.x += u[t] * k4.x; s4.y += u[t] * k4.y; s4.z += u[t] * k4.z; s4.w += u[t] * k4.w;
                }
                st4s(sS + px * SP + 4 * j4, s4);
            }
        }
        __syncthreads();
    }
    // final state
    for (int i = tid; i < DV * DK / 4; i += NT) {
        const int x = i / (DK / 4), j4 = i % (DK / 4);
        st4s(a.S_final + (size_t)chain * DV * DK + (size_t)i * 4, ld4s(sS + x * SP + 4 * j4));
    }
}

template <typename T, int DK, int DV>
cudaError_t launch_fwd(const Args& a, cudaStream_t st)
{
    const size_t smem = sizeof(float) * FwdSmem(DK, DV, a.r).total;
    auto kern = carve_fwd_simt_kernel<T, DK, DV>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<a.B * a.H, NT, smem, st>>>(a);
    return cudaGetLastError();
}

template <typename T>
cudaError_t dispatch_fwd(const Args& a, cudaStream_t st)
{
#define CARVE_CASE(DK_, DV_) \
    if (a.dk == DK_ && a.dv == DV_) return launch_fwd<T, DK_, DV_>(a, st);
    CARVE_CASE(64, 64)
    CARVE_CASE(64, 128)
    CARVE_CASE(128, 64)
    CARVE_CASE(128, 128)
    CARVE_CASE(64, 256)
    CARVE_CASE(256, 64)
    CARVE_CASE(128, 256)
    CARVE_CASE(256, 128)
#undef CARVE_CASE
    return cudaErrorInvalidValue;
}

}  // namespace

size_t simt_fwd_smem_bytes(int dk, int dv, int r) { return sizeof(float) * FwdSmem(dk, dv, r).total; }

cudaError_t simt_fwd_launch(const Args& a, int dtype, cudaStream_t st)
{
    return dtype == CARVE_BF16 ? dispatch_fwd<__nv_bfloat16>(a, st) : dispatch_fwd<float>(a, st);
}

}  // namespace carve

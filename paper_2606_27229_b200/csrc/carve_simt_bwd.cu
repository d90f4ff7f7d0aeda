// carve_simt_bwd.cu -- fp32 SIMT path of the CARVE layer operator (backward).
//
// One CTA per (batch, head) chain walks the 16-token solve sub-chunks in reverse, the running
// state adjoint dS (d_v x d_k fp32) resident in shared memory.  It is the chunk-matrix adjoint of
// Alg. 2 -- the same gradient computation as the per-token reverse scan of
// Alg. 4 (l.788-817), batched over a sub-chunk -- with the fold glue of Alg. 5 (l.844-848) at every
// gate-chunk start.  DESIGN.md "Backward" derives every line; in short, with W_ts = e^{lg_t-lg_s}:
//   dU  = scale P^T dO + Ktil dS'^T            dP = scale tril(dO U^T)
//   dY_t = dU_t - sum_{t'>t} A_t't dR_t',  dR = beta dY,  dbeta_t = <dY_t, e_t>,  dA = -stril(dR U^T)
//   dS  = dS' diag(gamma_L) + scale dO^T Qbar - dR^T Kbar  (+ [Ub;Uw]^T dG at a gate-chunk start)
//   dq^, dk^, dlg from the pairwise W terms and from Kbar/Qbar/Ktil; dla = reverse cumsum(dlg)
//   dg = dla, db_pre = -dla b, dw_pre = dR v w(1-w), dv = dR w, then the gate/fold/L2-norm chain.
// Saved by the forward (workspace): the state entering every sub-chunk, e_t, tanh bottleneck tt,
// and G_c.  Everything else is recomputed.  No floating-point atomics: every accumulator has one
// owner thread, so results are run-to-run bitwise identical.
#include "simt_common.cuh"

namespace carve {
namespace {

struct BwdSmem {
    int DS, Kbar, Qbar, Ktil, Lg, Qh, Kh, Bg, DKtil, DKbar, DQbar, C, U, DO, DU, Tt, Dz, A, P, DA, DP, Gam, Cs,
        Beta, Rnq, Rnk, DbPart, AccVb, AccVw, total;
    __host__ __device__ BwdSmem(int dk, int dv, int r)
    {
        const int SP = dk + 4, R2 = 2 * r;
        int o = 0;
        DS = o;     o += dv * SP;
        Kbar = o;   o += SC * dk;   // Kbar,Qbar,Ktil,Lg are contiguous: reused as the dG dump [R2][dk]
        Qbar = o;   o += SC * dk;
        Ktil = o;   o += SC * dk;
        Lg = o;     o += SC * dk;
        Qh = o;     o += SC * dk;
        Kh = o;     o += SC * dk;
        Bg = o;     o += SC * dk;
        DKtil = o;  o += SC * dk;
        DKbar = o;  o += SC * dk;
        DQbar = o;  o += SC * dk;
        C = o;      o += SC * dk;
        U = o;      o += SC * dv;
        DO = o;     o += SC * dv;
        DU = o;     o += SC * dv;
        Tt = o;     o += SC * R2;
        Dz = o;     o += SC * R2;
        A = o;      o += SC * AP;
        P = o;      o += SC * AP;
        DA = o;     o += SC * AP;
        DP = o;     o += SC * AP;
        Gam = o;    o += dk;
        Cs = o;     o += dk;
        Beta = o;   o += SC;
        Rnq = o;    o += SC;
        Rnk = o;    o += SC;
        DbPart = o; o += (NT / 32) * SC;
        AccVb = o;  o += dk * r;
        AccVw = o;  o += dv * r;
        total = o;
    }
};

template <typename T, int DK, int DV>
__global__ void __launch_bounds__(NT, 1) carve_bwd_simt_kernel(const Args a)
{
    extern __shared__ __align__(16) float smem[];
    constexpr int SP = DK + 4;
    const int r = a.r, R2 = 2 * r;
    const BwdSmem L_(DK, DV, r);
    float* sDS = smem + L_.DS;
    float* sKbar = smem + L_.Kbar;
    float* sQbar = smem + L_.Qbar;
    float* sKtil = smem + L_.Ktil;
    float* sLg = smem + L_.Lg;
    float* sQh = smem + L_.Qh;
    float* sKh = smem + L_.Kh;
    float* sBg = smem + L_.Bg;
    float* sDKtil = smem + L_.DKtil;
    float* sDKbar = smem + L_.DKbar;
    float* sDQbar = smem + L_.DQbar;
    float* sC = smem + L_.C;
    float* sU = smem + L_.U;
    float* sDO = smem + L_.DO;
    float* sDU = smem + L_.DU;
    float* sT = smem + L_.Tt;
    float* sDz = smem + L_.Dz;
    float* sA = smem + L_.A;
    float* sP = smem + L_.P;
    float* sDA = smem + L_.DA;
    float* sDP = smem + L_.DP;
    float* sGam = smem + L_.Gam;
    float* sCs = smem + L_.Cs;
    float* sBeta = smem + L_.Beta;
    float* sRnq = smem + L_.Rnq;
    float* sRnk = smem + L_.Rnk;
    float* sDbPart = smem + L_.DbPart;
    float* sAccVb = smem + L_.AccVb;
    float* sAccVw = smem + L_.AccVw;
    float* sDG = sKbar;  // [R2][DK] dump of the dG registers at a gate-chunk start

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
    const T* gdO = static_cast<const T*>(a.dO);
    T* gdq = static_cast<T*>(a.dq);
    T* gdk = static_cast<T*>(a.dk_);
    T* gdv = static_cast<T*>(a.dv_);
    T* gdf = static_cast<T*>(a.df);
    T* gdbx = static_cast<T*>(a.dbx);
    T* gdwx = static_cast<T*>(a.dwx);
    T* gdbeta = static_cast<T*>(a.dbeta);
    auto tokoff = [&](int t) -> size_t { return ((size_t)b * a.T + t) * a.H + h; };

    constexpr int TPT = SC * DV / NT;  // tokens per thread, thread = (value channel px, token group ptg)
    constexpr int JR = DK * DV / NT;   // state columns per thread in the dS update
    constexpr int NGK = NT / DK;       // token groups, thread = (key channel kj, token group kg)
    constexpr int TPK = SC / NGK;      // tokens per thread there
    constexpr int MAXG = DK / 4;       // dG registers per thread (covers r <= 32)
    const int px = tid % DV, ptg = tid / DV;
    const int kj = tid % DK, kg = tid / DK;

    float* part = a.ws_part + (size_t)chain * a.part_stride;  // [dUb|dUw][dVb][dVw][dA][dtau]
    float* partU = part;
    float* partVb = part + 2 * r * DV;
    float* partVw = partVb + DK * r;
    float* partA = partVw + DV * r;
    float* partTau = partA + DK;

    // ---- init: dS <- dS_final, zero accumulators
    for (int i = tid; i < DV * DK / 4; i += NT) {
        const int x = i / (DK / 4), j4 = i % (DK / 4);
        float4 v4 = make_float4(0.f, 0.f, 0.f, 0.f);
        if (a.dS_final) v4 = ldg4(a.dS_final + (size_t)chain * DV * DK + (size_t)i * 4);
        st4s(sDS + x * SP + 4 * j4, v4);
    }
    for (int i = tid; i < DK * r; i += NT) sAccVb[i] = 0.f;
    for (int i = tid; i < DV * r; i += NT) sAccVw[i] = 0.f;
    for (int i = tid; i < R2 * DV; i += NT) partU[i] = 0.f;
    float accA = 0.f, accTau = 0.f;
    float dGreg[MAXG];
#pragma unroll
    for (int k = 0; k < MAXG; ++k) dGreg[k] = 0.f;
    const float eA = (a.A && tid < DK) ? expf(__ldg(a.A + h * DK + tid)) : 1.f;
    const float tauj = (a.tau && tid < DK) ? __ldg(a.tau + h * DK + tid) : 0.f;
    __syncthreads();

    for (int c = nchunks - 1; c >= 0; --c) {
        const int t0 = c * SC;
        const float* Sc = a.ws_states + ((size_t)chain * nchunks + c) * DV * DK;
        const float* Gc = a.ws_G + ((size_t)chain * (a.T / a.L) + c / nsub) * R2 * DK;

        // ---- B0: loads
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
            if (lane == 0) { sRnq[t] = rq; sRnk[t] = rk; }
        }
        if (tid < SC) sBeta[tid] = ldf(gbeta, tokoff(t0 + tid));
        for (int it = tid; it < SC * R2; it += NT) sT[it] = a.ws_tt[tokoff(t0 + it / R2) * R2 + it % R2];
        for (int it = tid; it < SC * DV; it += NT) {
            const int x = it % DV, t = it / DV;
            const size_t go = tokoff(t0 + t) * DV + x;
            sDO[it] = ldf(gdO, go);
            sU[it] = ldf(gbeta, tokoff(t0 + t)) * a.ws_E[go];
        }
        __syncthreads();
        // ---- B1: erase gate and log-retention (recomputed as in F3/F4)
        for (int it = tid; it < SC * DK; it += NT) {
            const int j = it % DK, t = it / DK;
            const size_t go = tokoff(t0 + t) * DK + j;
            float bp = ldf(gbx, go);
            for (int i4 = 0; i4 < r / 4; ++i4)
                bp += dot4(ldg4(a.Vb + (size_t)j * r + 4 * i4), ld4s(sT + t * R2 + 4 * i4));
            const float eAj = a.A ? expf(__ldg(a.A + h * DK + j)) : 1.f;
            const float ta = a.tau ? __ldg(a.tau + h * DK + j) : 0.f;
            const float g = -eAj * softplusf(ldf(gf, go) + ta);
            sBg[it] = sigmoidf_(bp);
            sLg[it] = g - softplusf(bp);
        }
        __syncthreads();
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
            const float lg = sLg[it], lgm1 = t ? sLg[it - DK] : 0.f, lgL = sLg[(SC - 1) * DK + j];
            const float kh = sKh[it];
            sKbar[it] = kh * expf(lgm1);
            sQbar[it] = sQh[it] * expf(lg);
            sKtil[it] = kh * expf(lgL - lg);
        }
        __syncthreads();
        // ---- B2: A, P (pairwise, as F6);  dU' = Ktil dS'^T (registers);  dKtil = U dS';  cs = colsum(S . dS')
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
        float dUacc[TPT];
#pragma unroll
        for (int u = 0; u < TPT; ++u) dUacc[u] = 0.f;
        for (int j4 = 0; j4 < DK / 4; ++j4) {
            const float4 d4 = ld4s(sDS + px * SP + 4 * j4);
#pragma unroll
            for (int u = 0; u < TPT; ++u) dUacc[u] += dot4(ld4s(sKtil + (ptg * TPT + u) * DK + 4 * j4), d4);
        }
        {
            float acc[TPK];
#pragma unroll
            for (int u = 0; u < TPK; ++u) acc[u] = 0.f;
            float cs = 0.f;
            for (int x = 0; x < DV; x += 4) {
                const float d0 = sDS[(x + 0) * SP + kj], d1 = sDS[(x + 1) * SP + kj], d2 = sDS[(x + 2) * SP + kj],
                            d3 = sDS[(x + 3) * SP + kj];
                if (kg == 0)
                    cs += __ldg(Sc + (size_t)(x + 0) * DK + kj) * d0 + __ldg(Sc + (size_t)(x + 1) * DK + kj) * d1 +
                          __ldg(Sc + (size_t)(x + 2) * DK + kj) * d2 + __ldg(Sc + (size_t)(x + 3) * DK + kj) * d3;
#pragma unroll
                for (int u = 0; u < TPK; ++u) {
                    const float4 u4 = ld4s(sU + (kg * TPK + u) * DV + x);
                    acc[u] += u4.x * d0 + u4.y * d1 + u4.z * d2 + u4.w * d3;
                }
            }
#pragma unroll
            for (int u = 0; u < TPK; ++u) sDKtil[(kg * TPK + u) * DK + kj] = acc[u];
            if (kg == 0) sCs[kj] = cs;
        }
        __syncthreads();
        // ---- B3: dU = dU' + scale P^T dO
#pragma unroll
        for (int u = 0; u < TPT; ++u) {
            const int t = ptg * TPT + u;
            float v = dUacc[u];
            for (int tp = t; tp < SC; ++tp) v += a.scale * sP[tp * AP + t] * sDO[tp * DV + px];
            sDU[t * DV + px] = v;
        }
        __syncthreads();
        // ---- B4: transposed solve  dY_t = dU_t - sum_{t'>t} A_t't dR_t',  dR_t = beta_t dY_t;  dbeta
        if (tid < DV) {
            float dr[SC];
#pragma unroll
            for (int t = SC - 1; t >= 0; --t) {
                float dy = sDU[t * DV + tid];
#pragma unroll
                for (int tp = t + 1; tp < SC; ++tp) dy -= sA[tp * AP + t] * dr[tp];
                float pb = dy * a.ws_E[tokoff(t0 + t) * DV + tid];
                dr[t] = sBeta[t] * dy;
                sDU[t * DV + tid] = dr[t];
                pb = warp_sum(pb);
                if (lane == 0) sDbPart[warp * SC + t] = pb;
            }
        }
        __syncthreads();
        // ---- B5: dA = -stril(dR U^T), dP = scale tril(dO U^T);  dKbar = -dR S,  dQbar = scale dO S
        {
            int cnt = 0;
            for (int t = 0; t < SC; ++t)
                for (int s = 0; s <= t; ++s, ++cnt) {
                    if ((cnt & (NT / 32 - 1)) != warp) continue;
                    float pa = 0.f, pp = 0.f;
                    for (int x = lane; x < DV; x += 32) {
                        const float us = sU[s * DV + x];
                        pa += sDU[t * DV + x] * us;
                        pp += sDO[t * DV + x] * us;
                    }
                    pp = warp_sum(pp);
                    pa = warp_sum(pa);
                    if (lane == 0) {
                        sDP[t * AP + s] = a.scale * pp;
                        sDA[t * AP + s] = (s < t) ? -pa : 0.f;
                    }
                }
        }
        {
            float aK[TPK], aQ[TPK];
#pragma unroll
            for (int u = 0; u < TPK; ++u) aK[u] = aQ[u] = 0.f;
            float n0 = __ldg(Sc + kj), n1 = __ldg(Sc + DK + kj), n2 = __ldg(Sc + 2 * DK + kj),
                  n3 = __ldg(Sc + 3 * DK + kj);
            for (int x = 0; x < DV; x += 4) {
                const float s0 = n0, s1 = n1, s2 = n2, s3 = n3;
                if (x + 4 < DV) {
                    n0 = __ldg(Sc + (size_t)(x + 4) * DK + kj);
                    n1 = __ldg(Sc + (size_t)(x + 5) * DK + kj);
                    n2 = __ldg(Sc + (size_t)(x + 6) * DK + kj);
                    n3 = __ldg(Sc + (size_t)(x + 7) * DK + kj);
                }
#pragma unroll
                for (int u = 0; u < TPK; ++u) {
                    const float4 r4 = ld4s(sDU + (kg * TPK + u) * DV + x);
                    const float4 o4 = ld4s(sDO + (kg * TPK + u) * DV + x);
                    aK[u] -= r4.x * s0 + r4.y * s1 + r4.z * s2 + r4.w * s3;
                    aQ[u] += o4.x * s0 + o4.y * s1 + o4.z * s2 + o4.w * s3;
                }
            }
#pragma unroll
            for (int u = 0; u < TPK; ++u) {
                sDKbar[(kg * TPK + u) * DK + kj] = aK[u];
                sDQbar[(kg * TPK + u) * DK + kj] = a.scale * aQ[u];
            }
        }
        __syncthreads();
        // ---- B6: dS <- dS' diag(gamma_L) + scale dO^T Qbar - dR^T Kbar   (in place)
        {
            float co[SC], cr[SC];
#pragma unroll
            for (int t = 0; t < SC; ++t) {
                co[t] = a.scale * sDO[t * DV + px];
                cr[t] = sDU[t * DV + px];
            }
            for (int j4 = ptg * (JR / 4); j4 < (ptg + 1) * (JR / 4); ++j4) {
                float4 d4 = ld4s(sDS + px * SP + 4 * j4);
                const float4 g4 = ld4s(sGam + 4 * j4);
                d4.x *= g4.x; d4.y *= g4.y; d4.z *= g4.z; d4.w *= g4.w;
#pragma unroll
                for (int t = 0; t < SC; ++t) {
                    const float4 q4 = ld4s(sQbar + t * DK + 4 * j4), k4 = ld4s(sKbar + t * DK + 4 * j4);
                    d4.x += co[t] * q4.x - cr[t] * k4.x;
                    d4.y += co[t] * q4.y - cr[t] * k4.y;
                    d4.z += co[t] * q4.z - cr[t] * k4.z;
                    d4.w += co[t] * q4.w - cr[t] * k4.w;
                }
                st4s(sDS + px * SP + 4 * j4, d4);
            }
        }
        //      write gate: dv = dR w, dw_pre = dR v w (1-w)  (Alg. 4 l.806-808 correctness note l.819)
        for (int it = tid; it < SC * DV; it += NT) {
            const int x = it % DV, t = it / DV;
            const size_t go = tokoff(t0 + t) * DV + x;
            float w = 1.f;   // scalar-write variant (wx = NULL): w == 1, no write-gate adjoint
            if (gwx) {
                float wp = ldf(gwx, go);
                for (int i4 = 0; i4 < r / 4; ++i4)
                    wp += dot4(ldg4(a.Vw + (size_t)x * r + 4 * i4), ld4s(sT + t * R2 + r + 4 * i4));
                w = sigmoidf_(wp);
            }
            const float dr = sDU[it];
            const float dwp = gwx ? dr * ldf(gv, go) * w * (1.f - w) : 0.f;
            stf(gdv, go, dr * w);
            if (gwx) stf(gdwx, go, dwp);
            sU[it] = dwp;
        }
        //      pairwise terms.  role 0 (thread j < DK): row sums, kept in registers;
        //      role 1 (thread NT-DK+j): column sums -> sC
        float colLg[SC], colKh[SC], dQrow[SC], Xr[SC];
        if (tid < DK) {
#pragma unroll
            for (int t = 0; t < SC; ++t) { colLg[t] = sLg[t * DK + tid]; colKh[t] = sKh[t * DK + tid]; }
#pragma unroll
            for (int t = 0; t < SC; ++t) {
                float dq = 0.f, xx = 0.f;
#pragma unroll
                for (int s = 0; s <= t; ++s) {
                    const float kw = colKh[s] * expf(colLg[t] - colLg[s]);
                    dq += sDP[t * AP + s] * kw;
                    if (t + 1 < SC) xx += sDA[(t + 1) * AP + s] * kw;
                }
                dQrow[t] = dq;
                Xr[t] = xx;
            }
        }
        if (tid >= NT - DK) {
            const int j = tid - (NT - DK);
            float lgc[SC], khc[SC], qhc[SC];
#pragma unroll
            for (int t = 0; t < SC; ++t) { lgc[t] = sLg[t * DK + j]; khc[t] = sKh[t * DK + j]; qhc[t] = sQh[t * DK + j]; }
#pragma unroll
            for (int s = 0; s < SC; ++s) {
                float cc = 0.f;
#pragma unroll
                for (int tp = s; tp < SC; ++tp) {
                    float term = sDP[tp * AP + s] * qhc[tp];
                    if (tp + 1 < SC) term += sDA[(tp + 1) * AP + s] * khc[tp + 1];
                    cc += term * expf(lgc[tp] - lgc[s]);
                }
                sC[s * DK + j] = cc;
            }
        }
        __syncthreads();
        // ---- B7: combine per key channel, reverse cumulative sum, decay / erase-gate gradients
        if (tid < DK) {
            const int j = tid;
            const float lgL = colLg[SC - 1];
            float extra = sGam[j] * sCs[j];
#pragma unroll
            for (int t = 0; t < SC; ++t) extra += colKh[t] * expf(lgL - colLg[t]) * sDKtil[t * DK + j];
            float run = 0.f, dKbar_next = 0.f;
#pragma unroll
            for (int t = SC - 1; t >= 0; --t) {
                const float e_lg = expf(colLg[t]), e_lgm1 = t ? expf(colLg[t > 0 ? t - 1 : 0]) : 1.f,
                            e_til = expf(lgL - colLg[t]);
                const float qh = sQh[t * DK + j];
                const float dQb = sDQbar[t * DK + j], dKb = sDKbar[t * DK + j], dKt = sDKtil[t * DK + j],
                            Cc = sC[t * DK + j];
                const float dqh = dQrow[t] + dQb * e_lg;
                const float dkh = (t ? Xr[t > 0 ? t - 1 : 0] : 0.f) + Cc + dKb * e_lgm1 + dKt * e_til;
                float dlg = qh * dQrow[t] + qh * e_lg * dQb - colKh[t] * Cc - colKh[t] * e_til * dKt;
                if (t + 1 < SC) dlg += colKh[t + 1 < SC ? t + 1 : t] * (Xr[t] + e_lg * dKbar_next);
                if (t == SC - 1) dlg += extra;
                run += dlg;  // dla_t = sum_{t' >= t} dlg_t'
                sDQbar[t * DK + j] = dqh;
                sDKbar[t * DK + j] = dkh;
                dKbar_next = dKb;
                const size_t go = tokoff(t0 + t) * DK + j;
                const float dbp = -run * sBg[t * DK + j];
                sC[t * DK + j] = dbp;
                stf(gdbx, go, dbp);
                const float fv = ldf(gf, go) + tauj;
                const float dfv = run * (-eA) * sigmoidf_(fv);
                stf(gdf, go, dfv);
                accTau += dfv;
                accA += run * (-eA * softplusf(fv));
            }
        }
        //      write-gate chain: dVw += dw_pre^T tt_w ; dz_w = (dw_pre Vw) (1 - tt_w^2)
        for (int it = tid; it < DV * (r / 4); it += NT) {
            const int i4 = it % (r / 4), x = it / (r / 4);
            float4 acc = ld4s(sAccVw + x * r + 4 * i4);
#pragma unroll
            for (int t = 0; t < SC; ++t) {
                const float dw = sU[t * DV + x];
                const float4 t4 = ld4s(sT + t * R2 + r + 4 * i4);
                acc.x += dw * t4.x; acc.y += dw * t4.y; acc.z += dw * t4.z; acc.w += dw * t4.w;
            }
            st4s(sAccVw + x * r + 4 * i4, acc);
        }
        for (int it = tid; it < SC * r; it += NT) {
            const int i = it % r, t = it / r;
            float s = 0.f;
            if (a.Vw)
                for (int x = 0; x < DV; ++x) s += sU[t * DV + x] * __ldg(a.Vw + (size_t)x * r + i);
            const float tv = sT[t * R2 + r + i];
            sDz[t * R2 + r + i] = s * (1.f - tv * tv);
        }
        __syncthreads();
        // ---- B8: erase-gate chain: dVb += db_pre^T tt_b ; dz_b = (db_pre Vb) (1 - tt_b^2)
        for (int it = tid; it < DK * (r / 4); it += NT) {
            const int i4 = it % (r / 4), j = it / (r / 4);
            float4 acc = ld4s(sAccVb + j * r + 4 * i4);
#pragma unroll
            for (int t = 0; t < SC; ++t) {
                const float db = sC[t * DK + j];
                const float4 t4 = ld4s(sT + t * R2 + 4 * i4);
                acc.x += db * t4.x; acc.y += db * t4.y; acc.z += db * t4.z; acc.w += db * t4.w;
            }
            st4s(sAccVb + j * r + 4 * i4, acc);
        }
        for (int it = tid; it < SC * r; it += NT) {
            const int i = it % r, t = it / r;
            float s = 0.f;
            for (int j = 0; j < DK; ++j) s += sC[t * DK + j] * __ldg(a.Vb + (size_t)j * r + i);
            const float tv = sT[t * R2 + i];
            sDz[t * R2 + i] = s * (1.f - tv * tv);
        }
        __syncthreads();
        // ---- B9: bottleneck: dq^ += dz G ; dG += dz^T q^
        {
            float acc[TPK];
#pragma unroll
            for (int u = 0; u < TPK; ++u) acc[u] = 0.f;
            for (int i = 0; i < R2; ++i) {
                const float g = __ldg(Gc + (size_t)i * DK + kj);
#pragma unroll
                for (int u = 0; u < TPK; ++u) acc[u] += sDz[(kg * TPK + u) * R2 + i] * g;
            }
            float qcol[SC];
#pragma unroll
            for (int t = 0; t < SC; ++t) qcol[t] = sQh[t * DK + kj];
#pragma unroll
            for (int k = 0; k < MAXG; ++k) {
                const int i = kg + NGK * k;
                if (i < R2) {
                    float s = 0.f;
#pragma unroll
                    for (int t = 0; t < SC; ++t) s += sDz[t * R2 + i] * qcol[t];
                    dGreg[k] += s;
                }
            }
#pragma unroll
            for (int u = 0; u < TPK; ++u) sDQbar[(kg * TPK + u) * DK + kj] += acc[u];
        }
        __syncthreads();
        // ---- B10: L2-norm backward, write dq, dk, dbeta;  dump dG at a gate-chunk start
        for (int t = warp; t < SC; t += NT / 32) {
            const size_t ro = tokoff(t0 + t) * DK;
            float dqv[DK / 32], dkv[DK / 32], qv[DK / 32], kv[DK / 32];
            float pq = 0.f, pk = 0.f;
#pragma unroll
            for (int e = 0; e < DK / 32; ++e) {
                const int j = lane + 32 * e;
                dqv[e] = sDQbar[t * DK + j]; qv[e] = sQh[t * DK + j];
                dkv[e] = sDKbar[t * DK + j]; kv[e] = sKh[t * DK + j];
                pq += dqv[e] * qv[e];
                pk += dkv[e] * kv[e];
            }
            pq = warp_sum(pq);
            pk = warp_sum(pk);
#pragma unroll
            for (int e = 0; e < DK / 32; ++e) {
                const int j = lane + 32 * e;
                const float oq = a.l2norm ? (dqv[e] - qv[e] * pq) * sRnq[t] : dqv[e];
                const float ok = a.l2norm ? (dkv[e] - kv[e] * pk) * sRnk[t] : dkv[e];
                stf(gdq, ro + j, oq);
                stf(gdk, ro + j, ok);
            }
        }
        if (tid < SC) {
            float s = 0.f;
            for (int w = 0; w < DV / 32; ++w) s += sDbPart[w * SC + tid];
            stf(gdbeta, tokoff(t0 + tid), s);
        }
        const bool gate_start = (c % nsub == 0);
        if (gate_start) {
#pragma unroll
            for (int k = 0; k < MAXG; ++k) {
                const int i = kg + NGK * k;
                if (i < R2) { sDG[i * DK + kj] = dGreg[k]; dGreg[k] = 0.f; }
            }
        }
        __syncthreads();
        // ---- fold glue (Alg. 5 l.844-848): d[Ub;Uw] += dG S_c^T ;  dS += [Ub;Uw]^T dG
        if (gate_start) {
            for (int x = warp; x < DV; x += NT / 32) {
                float sv[DK / 32];
#pragma unroll
                for (int e = 0; e < DK / 32; ++e) sv[e] = __ldg(Sc + (size_t)x * DK + lane + 32 * e);
                for (int i = 0; i < R2; ++i) {
                    float p = 0.f;
#pragma unroll
                    for (int e = 0; e < DK / 32; ++e) p += sDG[i * DK + lane + 32 * e] * sv[e];
                    p = warp_sum(p);
                    if (lane == 0) partU[i * DV + x] += p;
                }
            }
            for (int j4 = ptg * (JR / 4); j4 < (ptg + 1) * (JR / 4); ++j4) {
                float4 d4 = ld4s(sDS + px * SP + 4 * j4);
                for (int i = 0; i < R2; ++i) {
                    const float u = (i < r) ? __ldg(a.Ub + (size_t)i * DV + px) : (a.Uw ? __ldg(a.Uw + (size_t)(i - r) * DV + px) : 0.f);
                    const float4 g4 = ld4s(sDG + i * DK + 4 * j4);
                    d4.x += u * g4.x; d4.y += u * g4.y; d4.z += u * g4.z; d4.w += u * g4.w;
                }
                st4s(sDS + px * SP + 4 * j4, d4);
            }
            __syncthreads();  // sDG aliases Kbar..Lg, rewritten by the next sub-chunk
        }
    }
    // ---- epilogue: dS0 and the per-chain partial weight gradients
    for (int i = tid; i < DV * DK / 4; i += NT) {
        const int x = i / (DK / 4), j4 = i % (DK / 4);
        st4s(a.dS0 + (size_t)chain * DV * DK + (size_t)i * 4, ld4s(sDS + x * SP + 4 * j4));
    }
    for (int i = tid; i < DK * r; i += NT) partVb[i] = sAccVb[i];
    for (int i = tid; i < DV * r; i += NT) partVw[i] = sAccVw[i];
    if (tid < DK) { partA[tid] = accA; partTau[tid] = accTau; }
}

// Deterministic reduction of the per-chain partials (Alg. 4 line 16 l.816: "reduce over heads").
__global__ void carve_reduce_weights_kernel(const float* __restrict__ part, int chains, int stride, int H, int dk,
                                            int dv, int r, float* dUb, float* dUw, float* dVb, float* dVw,
                                            float* dA, float* dtau)
{
    const int nU = r * dv, nVb = dk * r, nVw = dv * r, nW = 2 * nU + nVb + nVw;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx < nW) {
        float s = 0.f;
        for (int c = 0; c < chains; ++c) s += part[(size_t)c * stride + idx];
        if (idx < nU) dUb[idx] = s;
        else if (idx < 2 * nU) { if (dUw) dUw[idx - nU] = s; }   // NULL in the scalar-write variant
        else if (idx < 2 * nU + nVb) dVb[idx - 2 * nU] = s;
        else if (dVw) dVw[idx - 2 * nU - nVb] = s;
    } else if (idx < nW + 2 * H * dk) {
        const int k = idx - nW, which = k / (H * dk), hj = k % (H * dk), h = hj / dk, j = hj % dk;
        float* out = which ? dtau : dA;
        if (!out) return;
        float s = 0.f;
        for (int b = 0; b < chains / H; ++b) s += part[(size_t)(b * H + h) * stride + nW + which * dk + j];
        out[hj] = s;
    }
}

template <typename T, int DK, int DV>
cudaError_t launch_bwd(const Args& a, cudaStream_t st)
{
    const size_t smem = sizeof(float) * BwdSmem(DK, DV, a.r).total;
    auto kern = carve_bwd_simt_kernel<T, DK, DV>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<a.B * a.H, NT, smem, st>>>(a);
    return cudaGetLastError();
}

template <typename T>
cudaError_t dispatch_bwd(const Args& a, cudaStream_t st)
{
#define CARVE_CASE(DK_, DV_) \
    if (a.dk == DK_ && a.dv == DV_) return launch_bwd<T, DK_, DV_>(a, st);
    CARVE_CASE(64, 64)
    CARVE_CASE(64, 128)
    CARVE_CASE(128, 64)
    CARVE_CASE(128, 128)
    CARVE_CASE(64, 256)
    CARVE_CASE(256, 64)
#undef CARVE_CASE
    return cudaErrorInvalidValue;
}

}  // namespace

size_t simt_bwd_smem_bytes(int dk, int dv, int r) { return sizeof(float) * BwdSmem(dk, dv, r).total; }

cudaError_t simt_bwd_launch(const Args& a, int dtype, float* dA, float* dtau, float* dUb, float* dUw, float* dVb,
                            float* dVw, cudaStream_t st)
{
    cudaError_t e = dtype == CARVE_BF16 ? dispatch_bwd<__nv_bfloat16>(a, st) : dispatch_bwd<float>(a, st);
    if (e != cudaSuccess) return e;
    return reduce_weights_launch(a.ws_part, a.B * a.H, a.part_stride, a.H, a.dk, a.dv, a.r, dUb, dUw, dVb, dVw, dA, dtau, st);
}

cudaError_t reduce_weights_launch(const float* part, int chains, int stride, int H, int dk, int dv, int r, float* dUb,
                                  float* dUw, float* dVb, float* dVw, float* dA, float* dtau, cudaStream_t st)
{
    const int n = 2 * r * dv + dk * r + dv * r + 2 * H * dk;
    carve_reduce_weights_kernel<<<(n + 127) / 128, 128, 0, st>>>(part, chains, stride, H, dk, dv, r, dUb, dUw, dVb, dVw,
                                                                  dA, dtau);
    return cudaGetLastError();
}

}  // namespace carve

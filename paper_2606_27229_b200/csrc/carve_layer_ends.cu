// carve_layer_ends.cu -- the layer ends around the CARVE operator: SiLU on q, k, v (Eq. 6
// l.125-126) and RMSNorm of the assembled output (Alg. 1 line 15 l.194), forward and backward.
//
// These are the two chunk-local "hoisted" launches of the paper's training schedule (Alg. 3 step 3 l.399, step 9 l.407):
// fully parallel over tokens, no state, HBM-bound.  Each is ONE launch over all of its tensors (q, k, v together; the
// normalisation and its gain in one pass; the backward's input gradient and the gain-gradient partials in one pass), sized
// for bytes in flight: a thread keeps four 16-byte pieces outstanding (SiLU), a warp owns whole token rows of up to
// 8 KB (RMSNorm).  The projections W_Q, W_K, W_V, W_O are dense GEMMs outside the path (library calls).
// They are not fused into the serial kernels: there q and k arrive by TMA straight into MMA operand tiles and every extra
// elementwise pass would sit on the chunk-to-chunk dependency chain, and RMSNorm(reshape(o)) couples the heads of a token,
// i.e. chains that live on different SMs.
#include "carve_internal.h"

namespace carve {
namespace {

__device__ __forceinline__ float ex2f(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcpf(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// sigmoid(x) = 1 / (1 + 2^(-x log2 e)), evaluated on the side where the exponential is <= 1
__device__ __forceinline__ float sigm(float x)
{
    const float e = ex2f(-fabsf(x) * 1.4426950408889634f), r = rcpf(1.f + e);
    return x >= 0.f ? r : e * r;
}
// bf16 tensors: sigmoid through one tanh.approx (|error| < 3e-4, below the bf16 rounding of what it feeds): one
// transcendental and three instructions instead of two and seven -- these passes are bound by instruction issue as much
// as by HBM (~25 instructions per element in the backward).  fp32 tensors keep the exp/reciprocal form (1e-4 tolerance).
__device__ __forceinline__ float sigm_fast(float x)
{
    float t;
    asm("tanh.approx.f32 %0, %1;" : "=f"(t) : "f"(0.5f * x));
    return fmaf(0.5f, t, 0.5f);
}
template <typename T> __device__ __forceinline__ float sig_of(float x) { return sigm(x); }
template <> __device__ __forceinline__ float sig_of<__nv_bfloat16>(float x) { return sigm_fast(x); }
template <typename T> __device__ __forceinline__ float silu_f(float x) { return x * sig_of<T>(x); }
template <typename T> __device__ __forceinline__ float silu_d(float x)
{
    const float s = sig_of<T>(x);
    return fmaf(x * s, 1.f - s, s);
}

// a 16-byte piece as floats: 4 (fp32 tensors) or 8 (bf16 tensors)
template <typename T> struct Piece;
template <> struct Piece<float> {
    static constexpr int N = 4;
    // (plain loads: the tensor may be the one the kernel rewrites in place)
    static __device__ __forceinline__ void load(const void* p, size_t piece, float (&f)[8])
    {
        const float4 v = reinterpret_cast<const float4*>(p)[piece];
        f[0] = v.x; f[1] = v.y; f[2] = v.z; f[3] = v.w;
    }
    static __device__ __forceinline__ void store(void* p, size_t piece, const float (&f)[8])
    {
        reinterpret_cast<float4*>(p)[piece] = make_float4(f[0], f[1], f[2], f[3]);
    }
};
template <> struct Piece<__nv_bfloat16> {
    static constexpr int N = 8;
    static __device__ __forceinline__ void load(const void* p, size_t piece, float (&f)[8])
    {
        const uint4 v = reinterpret_cast<const uint4*>(p)[piece];
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) { f[2 * i] = __uint_as_float(w[i] << 16); f[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u); }
    }
    static __device__ __forceinline__ void store(void* p, size_t piece, const float (&f)[8])
    {
        uint32_t w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const __nv_bfloat162 h = __floats2bfloat162_rn(f[2 * i], f[2 * i + 1]);
            w[i] = *reinterpret_cast<const uint32_t*>(&h);
        }
        reinterpret_cast<uint4*>(p)[piece] = make_uint4(w[0], w[1], w[2], w[3]);
    }
};

struct SiluArgs {
    const void* x[3];   // pre-activations qx, kx, vx
    void* y[3];         // forward: q, k, v;  backward: dq, dk, dv (gradients, rewritten in place)
    size_t pieces[3];   // 16-byte pieces per tensor (0: tensor absent)
};

// blockIdx.y = tensor; grid-stride over its pieces, UN pieces in flight per thread.
template <typename T, bool BWD>
__global__ void __launch_bounds__(256, BWD ? 3 : 4) carve_silu_kernel(const SiluArgs a)
{
    constexpr int UN = 4, N = Piece<T>::N;
    const int which = blockIdx.y;
    // (selected, not indexed: a dynamically indexed kernel-parameter array is copied to local memory)
    const void* x = which == 0 ? a.x[0] : which == 1 ? a.x[1] : a.x[2];
    void* y = which == 0 ? a.y[0] : which == 1 ? a.y[1] : a.y[2];
    const size_t n = which == 0 ? a.pieces[0] : which == 1 ? a.pieces[1] : a.pieces[2];
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i0 < n; i0 += UN * stride) {
        float fx[UN][8], fy[UN][8];
#pragma unroll
        for (int u = 0; u < UN; ++u) {
            const size_t i = i0 + u * stride;
            if (i < n) {
                Piece<T>::load(x, i, fx[u]);
                if (BWD) Piece<T>::load(y, i, fy[u]);
            }
        }
#pragma unroll
        for (int u = 0; u < UN; ++u) {
            const size_t i = i0 + u * stride;
            if (i < n) {
#pragma unroll
                for (int e = 0; e < N; ++e) fy[u][e] = BWD ? fy[u][e] * silu_d<T>(fx[u][e]) : silu_f<T>(fx[u][e]);
                Piece<T>::store(y, i, fy[u]);
            }
        }
    }
}

template <typename T, bool BWD>
cudaError_t launch_silu(const SiluArgs& a, cudaStream_t st)
{
    size_t mx = 0;
    for (int i = 0; i < 3; ++i) mx = a.pieces[i] > mx ? a.pieces[i] : mx;
    if (mx == 0) return cudaSuccess;
    const size_t want = (mx + 256 * 4 - 1) / (256 * 4);
    const unsigned gx = (unsigned)(want < 148 * 8 ? want : 148 * 8);   // 8 resident blocks per SM, then grid-stride
    carve_silu_kernel<T, BWD><<<dim3(gx, 3), 256, 0, st>>>(a);
    return cudaGetLastError();
}

// ---- RMSNorm over the H*dv channels of a token ---------------------------------------------------------------------
// One warp owns a token row (n channels = np 16-byte pieces; lane l holds pieces l, l + 32, ..: up to MAXP of them, all
// loaded before the first use) and walks rows with a grid stride; the row's sum of squares is a warp shuffle reduction.
constexpr int kNormBlocks = 148 * 2, kNormWarps = kNormBlocks * 8;   // fixed grid: fixed row -> warp map, deterministic partials

__device__ __forceinline__ float warp_sum_all(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ void load_gain(const float* gain, int col, int N, float (&g)[8])
{
    const float4 a = __ldg(reinterpret_cast<const float4*>(gain + col));
    g[0] = a.x; g[1] = a.y; g[2] = a.z; g[3] = a.w;
    if (N == 8) {
        const float4 b = __ldg(reinterpret_cast<const float4*>(gain + col + 4));
        g[4] = b.x; g[5] = b.y; g[6] = b.z; g[7] = b.w;
    }
}

template <typename T, int MAXP>
__global__ void __launch_bounds__(256) carve_out_norm_fwd_kernel(const void* __restrict__ o, const float* __restrict__ gain,
                                                                 void* __restrict__ y, int rows, int np, float inv_n, float eps)
{
    constexpr int N = Piece<T>::N;
    const int lane = threadIdx.x & 31, warp = blockIdx.x * 8 + (threadIdx.x >> 5);
    for (int row = warp; row < rows; row += kNormWarps) {
        const size_t base = (size_t)row * np;
        float f[MAXP][8];
        float ss = 0.f;
#pragma unroll
        for (int i = 0; i < MAXP; ++i)
            if (lane + 32 * i < np) Piece<T>::load(o, base + lane + 32 * i, f[i]);
#pragma unroll
        for (int i = 0; i < MAXP; ++i)
            if (lane + 32 * i < np) {
#pragma unroll
                for (int e = 0; e < N; ++e) ss = fmaf(f[i][e], f[i][e], ss);
            }
        const float r = rsqrtf(warp_sum_all(ss) * inv_n + eps);
#pragma unroll
        for (int i = 0; i < MAXP; ++i)
            if (lane + 32 * i < np) {
                float g[8];
                load_gain(gain, (lane + 32 * i) * N, N, g);
#pragma unroll
                for (int e = 0; e < N; ++e) f[i][e] = f[i][e] * r * g[e];
                Piece<T>::store(y, base + lane + 32 * i, f[i]);
            }
    }
}

// Backward: d_o = r g dy - x r^3 mean(x g dy);  the warp's share of dgain = sum over its rows of dy x r, accumulated in a
// shared-memory slice of the warp's own (no atomics); the block's slices leave as one partial[block][n] (summed in fixed order by
// carve_out_norm_dgain_kernel).  The row's pieces stay in registers in their 16-byte form between the two passes over the
// row (statistics, then outputs): with 64 fewer accumulator registers and packed rows two blocks fit an SM.
template <typename T> struct Raw;
template <> struct Raw<float> { typedef float4 type; };
template <> struct Raw<__nv_bfloat16> { typedef uint4 type; };
__device__ __forceinline__ void unpack_raw(const float4& v, float (&f)[8]) { f[0] = v.x; f[1] = v.y; f[2] = v.z; f[3] = v.w; }
__device__ __forceinline__ void unpack_raw(const uint4& v, float (&f)[8])
{
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) { f[2 * i] = __uint_as_float(w[i] << 16); f[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u); }
}

template <typename T, int MAXP>
__global__ void __launch_bounds__(256, MAXP <= 8 ? 2 : 1)
carve_out_norm_bwd_kernel(const void* __restrict__ o, const float* __restrict__ gain, const void* __restrict__ dy,
                          void* __restrict__ d_o, float* __restrict__ partial, int rows, int np, float inv_n, float eps)
{
    constexpr int N = Piece<T>::N;
    typedef typename Raw<T>::type raw_t;
    extern __shared__ __align__(16) float sdg_all[];   // [8 warps][np * N]
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, warp = blockIdx.x * 8 + wib;
    float* sdg = sdg_all + (size_t)wib * np * N;
    for (int i = lane; i < np; i += 32) {
        float4* p4 = reinterpret_cast<float4*>(sdg + (size_t)i * N);
        p4[0] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (N == 8) p4[1] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    __syncwarp();
    for (int row = warp; row < rows; row += kNormWarps) {
        const size_t base = (size_t)row * np;
        raw_t xr[MAXP], dr[MAXP];
#pragma unroll
        for (int i = 0; i < MAXP; ++i)
            if (lane + 32 * i < np) {
                xr[i] = reinterpret_cast<const raw_t*>(o)[base + lane + 32 * i];
                dr[i] = reinterpret_cast<const raw_t*>(dy)[base + lane + 32 * i];
            }
        float ss = 0.f, sc = 0.f;
#pragma unroll
        for (int i = 0; i < MAXP; ++i)
            if (lane + 32 * i < np) {
                float g[8], x[8], d[8];
                load_gain(gain, (lane + 32 * i) * N, N, g);
                unpack_raw(xr[i], x);
                unpack_raw(dr[i], d);
#pragma unroll
                for (int e = 0; e < N; ++e) {
                    ss = fmaf(x[e], x[e], ss);
                    sc = fmaf(x[e], g[e] * d[e], sc);
                }
            }
        const float r = rsqrtf(warp_sum_all(ss) * inv_n + eps);
        const float c = warp_sum_all(sc) * inv_n * r * r * r;
#pragma unroll
        for (int i = 0; i < MAXP; ++i)
            if (lane + 32 * i < np) {
                float g[8], x[8], d[8], out[8], acc[8];
                load_gain(gain, (lane + 32 * i) * N, N, g);   // (8 KB of gain: L1 hits)
                unpack_raw(xr[i], x);
                unpack_raw(dr[i], d);
                float4* p4 = reinterpret_cast<float4*>(sdg + (size_t)(lane + 32 * i) * N);
                const float4 a0 = p4[0];
                acc[0] = a0.x; acc[1] = a0.y; acc[2] = a0.z; acc[3] = a0.w;
                if (N == 8) { const float4 a1 = p4[1]; acc[4] = a1.x; acc[5] = a1.y; acc[6] = a1.z; acc[7] = a1.w; }
#pragma unroll
                for (int e = 0; e < N; ++e) {
                    acc[e] = fmaf(d[e] * x[e], r, acc[e]);
                    out[e] = fmaf(r * g[e], d[e], -x[e] * c);
                }
                p4[0] = make_float4(acc[0], acc[1], acc[2], acc[3]);
                if (N == 8) p4[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
                Piece<T>::store(d_o, base + lane + 32 * i, out);
            }
    }
    // the block's eight slices, added in warp order, leave as ONE partial per block
    __syncthreads();
    const int ncol = np * N;
    float* dst = partial + (size_t)blockIdx.x * ncol;
    for (int j = threadIdx.x; j < ncol; j += 256) {
        float t = 0.f;
#pragma unroll
        for (int w = 0; w < 8; ++w) t += sdg_all[(size_t)w * ncol + j];
        dst[j] = t;
    }
}

// dgain[j] = sum over the blocks' partials in a fixed order (run-to-run identical bits): a block owns 32 columns, its 32
// warps each add a contiguous slice of the partials (128-byte coalesced reads), the slices are combined in slice order.
__global__ void __launch_bounds__(1024) carve_out_norm_dgain_kernel(const float* __restrict__ partial, float* __restrict__ dgain,
                                                                    int n, int nwarps)
{
    __shared__ float red[32][33];
    const int c = threadIdx.x & 31, sl = threadIdx.x >> 5, j = blockIdx.x * 32 + c;
    const int per = (nwarps + 31) / 32, w0 = sl * per, w1 = min(w0 + per, nwarps);
    float s = 0.f;
    if (j < n)
        for (int w = w0; w < w1; ++w) s += partial[(size_t)w * n + j];
    red[sl][c] = s;
    __syncthreads();
    if (sl == 0 && j < n) {
        float t = 0.f;
#pragma unroll
        for (int i = 0; i < 32; ++i) t += red[i][c];
        dgain[j] = t;
    }
}

template <typename T, int MAXP>
cudaError_t launch_norm(bool bwd, const void* o, const float* gain, const void* dy, void* out, float* partial, float* dgain,
                        int rows, int np, int n, float eps, cudaStream_t st)
{
    if (!bwd) {
        carve_out_norm_fwd_kernel<T, MAXP><<<kNormBlocks, 256, 0, st>>>(o, gain, out, rows, np, 1.f / (float)n, eps);
        return cudaGetLastError();
    }
    const size_t smem = (size_t)8 * n * sizeof(float);
    auto kern = carve_out_norm_bwd_kernel<T, MAXP>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    kern<<<kNormBlocks, 256, smem, st>>>(o, gain, dy, out, partial, rows, np, 1.f / (float)n, eps);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    carve_out_norm_dgain_kernel<<<(n + 31) / 32, 1024, 0, st>>>(partial, dgain, n, kNormBlocks);
    return cudaGetLastError();
}

template <typename T>
cudaError_t dispatch_norm(bool bwd, const void* o, const float* gain, const void* dy, void* out, float* partial, float* dgain,
                          int rows, int np, int n, float eps, cudaStream_t st)
{
    const int per_lane = (np + 31) / 32;
    if (per_lane <= 1) return launch_norm<T, 1>(bwd, o, gain, dy, out, partial, dgain, rows, np, n, eps, st);
    if (per_lane <= 2) return launch_norm<T, 2>(bwd, o, gain, dy, out, partial, dgain, rows, np, n, eps, st);
    if (per_lane <= 4) return launch_norm<T, 4>(bwd, o, gain, dy, out, partial, dgain, rows, np, n, eps, st);
    if (per_lane <= 8) return launch_norm<T, 8>(bwd, o, gain, dy, out, partial, dgain, rows, np, n, eps, st);
    if (per_lane <= 16) return launch_norm<T, 16>(bwd, o, gain, dy, out, partial, dgain, rows, np, n, eps, st);
    return cudaErrorInvalidValue;
}

}  // namespace

cudaError_t silu_qkv_launch(const carve_params_t& p, const void* qx, const void* kx, const void* vx, void* q, void* k, void* v,
                            bool bwd, cudaStream_t st)
{
    const size_t tok = (size_t)p.B * p.T * p.H, e = p.dtype == CARVE_BF16 ? 2 : 4;
    SiluArgs a{};
    a.x[0] = qx; a.x[1] = kx; a.x[2] = vx;
    a.y[0] = q; a.y[1] = k; a.y[2] = v;
    a.pieces[0] = qx ? tok * p.dk * e / 16 : 0;
    a.pieces[1] = kx ? tok * p.dk * e / 16 : 0;
    a.pieces[2] = vx ? tok * p.dv * e / 16 : 0;
    if (p.dtype == CARVE_BF16) return bwd ? launch_silu<__nv_bfloat16, true>(a, st) : launch_silu<__nv_bfloat16, false>(a, st);
    return bwd ? launch_silu<float, true>(a, st) : launch_silu<float, false>(a, st);
}

}  // namespace carve

namespace carve {

// rows of H*dv channels; at most 16 pieces of 16 bytes per lane: H*dv <= 4096 (bf16) / 2048 (fp32)
bool out_norm_supported(const carve_params_t& p)
{
    const size_t n = (size_t)p.H * p.dv, e = p.dtype == CARVE_BF16 ? 2 : 4;
    return n * e % 16 == 0 && n * e / 16 <= 32 * 16;
}
size_t out_norm_ws_bytes(const carve_params_t& p) { return (size_t)kNormBlocks * p.H * p.dv * sizeof(float); }

cudaError_t out_norm_launch(const carve_params_t& p, bool bwd, const void* o, const float* gain, float eps, const void* dy,
                            void* out, float* partial, float* dgain, cudaStream_t st)
{
    const int n = p.H * p.dv, rows = p.B * p.T, np = n * (p.dtype == CARVE_BF16 ? 2 : 4) / 16;
    return p.dtype == CARVE_BF16 ? dispatch_norm<__nv_bfloat16>(bwd, o, gain, dy, out, partial, dgain, rows, np, n, eps, st)
                                 : dispatch_norm<float>(bwd, o, gain, dy, out, partial, dgain, rows, np, n, eps, st);
}

}  // namespace carve

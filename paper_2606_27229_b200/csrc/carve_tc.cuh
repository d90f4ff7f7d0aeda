// carve_tc.cuh -- shared pieces of the tensor-core (tcgen05 + TMA) CARVE kernels: the shared-memory
// and TMEM maps, the thread <-> tile-row mapping, and small math helpers.
// walks through the phases; the comments here state what each buffer holds.
//
// One CTA of 128 NP threads (NP = d/32 warpgroups: 256 threads at d = 64, 512 at d = 128) owns one (batch, head)
// chain for the whole sequence.  Every MMA has M = 128: accumulator row r lives in TMEM lane r, warp w reads
// lanes 32*(w%4).., and the NP warpgroups (w/4) split the columns of a tile into parts of 32.  Rows 0..63 of a stacked tile are the
// "K-role" rows of the chunk's 64 tokens, rows 64..127 the "Q-role" rows of the same tokens, so
// one instruction computes e.g. [Kbar; Qbar] S^T.
#pragma once
#include "carve_internal.h"
#include "tc_common.cuh"

namespace carve {

// [B,T,H,d] bf16 seen as (d, H, B*T); one TMA box = 64 channels x 1 head x `rows` tokens, 128B-swizzled (carve_tc_fwd.cu).
bool tc_make_token_map(CUtensorMap* map, const void* base, int B, int T, int H, int d, int rows);

namespace tcp {

using namespace tc;

constexpr int NT = 256;  // threads per CTA
constexpr int LC = 64;   // tokens per solve chunk (gate chunks of L = 128 run as two solve chunks)
constexpr int AB = 16;   // anchor block: decay ratios > 1 are only ever formed inside one 16-token block

// TMEM column map (512 columns x 128 lanes of fp32).
constexpr uint32_t TM_S = 0;      // [dv lanes][dk]   fp32 state S_{c-1}, updated in place at the chunk end
constexpr uint32_t TM_ACC = 128;  // [128][dv]        rows 0..63  Kbar S^T (prediction), rows 64..127 Qbar S^T + P U (output)
constexpr uint32_t TM_X1 = 256;   // [128][max d]     gate up-projections, later U = T (beta R)
constexpr uint32_t TM_X2 = 384;   // G^T | Z, then the log-retention scan, then A|P blocks, then the state increment
constexpr uint32_t TM_COLS = 512;

struct Layout {  // byte offsets into the 1024-aligned dynamic shared memory
    uint32_t Sb, Ucat, Vcat, KQraw, F, BX, WX, V, KQbar, Ktil, Us, Y0, Y1, Y2, V1, V3, TP, Mm, Tm, misc, total;
    __host__ __device__ Layout(int dk, int dv, int r2)
    {
        uint32_t o = 0;
        auto take = [&](uint32_t n) { uint32_t r = o; o += (n + 1023u) & ~1023u; return r; };
        const int dm = dk > dv ? dk : dv;
        Sb = take(tile_bytes(dv, dk));      // bf16 S_{c-1}: rows x, cols j
        Ucat = take(tile_bytes(r2, dv));    // [Ub; Uw]: rows i, cols x
        Vcat = take(tile_bytes(dm, 64));    // row n: [Vb[n][0..r) | Vw[n][0..r)]
        KQraw = take(tile_bytes(128, dk));  // TMA: rows 0..63 k, rows 64..127 q
        F = take(tile_bytes(64, dk));       // TMA: decay logits            | later Kbar,Qbar (with BX)
        BX = take(tile_bytes(64, dk));      // TMA: erase pre-activation
        WX = take(tile_bytes(64, dv));      // TMA: write pre-activation    | later Ktil
        V = take(tile_bytes(64, dv));       // TMA: values -> V' = w.v      | later U
        KQbar = F; Ktil = WX; Us = V;
        // d = 128: one CTA per SM fills the shared memory.  d = 64: compacted to 112 KB so that TWO CTAs (two chains) share an
        // SM and hide each other's latency (config 4 has 2048 chains): the row operands of anchor blocks 1 and 3 live in TP
        // (free until P9a), those of block 2 in the upper half of Y1, and beta R / the output tile need only 8 KB.
        const bool compact = dk == 64;
        Y1 = take(16384);                   // [tt_b | tt_w] (128 rows) | C (column operand of A and P, 64 rows)
        Y0 = compact ? Y1 + 8192 : take((uint32_t)dk * 128);   // row operands re-anchored at token 32
        Y2 = take(compact ? 8192 : 16384);  // beta R | output tile (| d = 128: row operands re-anchored at tokens 16, 48)
        TP = take(16384);                   // rows 0..63 T = (I + beta A)^-1, rows 64..127 P
        V1 = compact ? TP : Y2;             // row operands re-anchored at token 16 (96 rows) ...
        V3 = V1 + tile_bytes(96, dk);       // ... and at token 48 (32 rows)
        Mm = KQraw;                         // fp32 beta A [64][64] over the raw k|q tile (dead after P7)
        misc = take(6144);                  // MiscT<dk>; at d = 64 it takes 4 KB and the diagonal inverses follow it
        Tm = compact ? misc + 4096 : KQraw + 16384;   // 8x8 diagonal inverses, [64][8] fp32
        total = o + 1024;                   // slack for the manual 1024-byte alignment
    }
};

// ---- chunk record ---------------------------------------------------------------------------------
// What the training forward saves per (chain, solve chunk) for the reverse kernel (carve_tc_bwd.cu):
// ready-to-use MMA operand tiles in the shared-memory image format (fetched with 1-D bulk copies),
// plus row-private elementwise data a thread reads straight from global memory.  Offsets in bytes.
//   SB   [dv][dk]   state entering the chunk, bf16
//   KT   [64][dk]   Ktil_t = k^_t gamma_L/gamma_t
//   PT   [128][64]  rows 0..63 scale.P (masked s <= t), rows 64..127 T = (I + diag(beta) A)^-1
//   U    [64][dv]   u_t  (e_t = u_t / beta_t is formed from it)
//   K0,Q0 [64][dk]  Kbar_t = k^_t gamma_{t-1}, scale.Qbar_t = scale.q^_t gamma_t   (chunk-anchored)
//   KQo  [128][dk]  the same rows anchored at the start of their own 16-token block
//   CC   [64][dk]   C_s = k^_s gamma_a/gamma_s (a = start of s's 16-token block)
//   VWX,W [64][dv]  w.v.(1-w) and w;  Bg [64][dk] erase gate b;  FQ,IC [64][dk] gamma_t/gamma_a and its inverse (row-private, piece-major)
//   tt   [64][64]   tanh bottleneck: the K-side rows of the forward's tile, erase half in chunks 0,1, write half in chunks 2,3
//   GT   [dk][64]   the forward's Vcat tile: columns 32.. hold G^T;  etot [4][dk], rn [128], beta [64] fp32
//   (tt, GT, etot, beta leave by bulk copies: per-thread global stores in the sections only a few warps run cost far
//    more than their bytes)
struct Rec {
    uint32_t SB, KT, PT, U, K0, Q0, KQo, CC, VWX, W, Bg, FQ, IC, tt, GT, etot, rn, beta, total;
    __host__ __device__ Rec(int dk, int dv)
    {
        uint32_t o = 0;
        auto take = [&](uint32_t n) { uint32_t r = o; o += (n + 1023u) & ~1023u; return r; };
        SB = take(tile_bytes(dv, dk));
        KT = take(tile_bytes(64, dk));
        PT = take(tile_bytes(128, 64));
        U = take(tile_bytes(64, dv));
        K0 = take(tile_bytes(64, dk));
        Q0 = take(tile_bytes(64, dk));
        KQo = take(tile_bytes(128, dk));
        CC = take(tile_bytes(64, dk));
        VWX = take(tile_bytes(64, dv));
        W = take(tile_bytes(64, dv));
        Bg = take(tile_bytes(64, dk));
        FQ = take(tile_bytes(64, dk));
        IC = take(tile_bytes(64, dk));
        tt = take(64 * 128);               // rows 0..63 of the forward's [tt_b pad 16 | tt_w pad 16] tile (bulk copy)
        GT = take(tile_bytes(dk, 64));
        etot = take(4u * dk * 4u);
        rn = take(128 * 4);
        beta = take(64 * 4);
        total = o;
    }
};

// Byte offset of 16-byte piece `cc` of row `row` in a row-private record array ([64 rows][d] bf16, only ever
// read by the thread that owns the row): piece-major, so a warp (32 consecutive rows, one piece) moves 512
// contiguous bytes both when the forward stores it and when the reverse kernel loads it.
__host__ __device__ __forceinline__ uint32_t rp_off(int row, int cc) { return (uint32_t)((cc * 64 + row) * 16); }

// misc area of the forward kernel (floats unless noted), sized by the key dimension
template <int DK>
struct MiscT {
    float eA[DK], tau[DK];      // exp(A_h), tau_h
    float etot[4][DK];          // exp(sum of log a over 16-token anchor block b)
    float gamL[DK];             // gamma_{L-1} of the chunk
    float nrm[128][DK / 32];    // partial sums of squares: rows 0..63 k, 64..127 q; [column part]
    float beta[64];             // write strength of the chunk's tokens
    uint64_t bar_mma, bar_kq, bar_fb, bar_wv;
    uint64_t bar_acc;           // the state products of P8 (waited for after the A|P blocks have been consumed)
    uint32_t tmem_base;
};
static_assert(sizeof(MiscT<128>) <= 6144 && sizeof(MiscT<64>) <= 4096, "misc area too small");

// Bare MUFU transcendentals (flush-to-zero forms: no denormal range fix-up code around them; every use below either
// has a result whose flush to 0 is the correct limit or an argument >= 1).
__device__ __forceinline__ float ex2_ftz(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float lg2_ftz(float x)
{
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_ftz(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
constexpr float kLog2e = 1.4426950408889634f, kLn2 = 0.6931471805599453f;
__device__ __forceinline__ float exp_fast(float x) { return ex2_ftz(x * kLog2e); }
__device__ __forceinline__ float softplus_fast(float x) { return fmaf(kLn2, lg2_ftz(1.f + ex2_ftz(-fabsf(x) * kLog2e)), fmaxf(x, 0.f)); }
__device__ __forceinline__ float sigmoid_fast(float x) { return rcp_ftz(1.f + ex2_ftz(-x * kLog2e)); }
__device__ __forceinline__ float tanh_fast(float x)
{
    float y;
    asm("tanh.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// sigmoid through one tanh.approx (one transcendental op instead of exp + reciprocal; |error| < 3e-4, below the bf16
// rounding of the values it feeds)
__device__ __forceinline__ float sigmoid_tanh(float x) { return fmaf(0.5f, tanh_fast(0.5f * x), 0.5f); }

__device__ __forceinline__ uint4 lds128(const uint8_t* p) { return *reinterpret_cast<const uint4*>(p); }
__device__ __forceinline__ void sts128(uint8_t* p, uint4 v) { *reinterpret_cast<uint4*>(p) = v; }
__device__ __forceinline__ void unpack8(uint4 w, float (&f)[8])
{
    f[0] = bf16_lo(w.x); f[1] = bf16_hi(w.x); f[2] = bf16_lo(w.y); f[3] = bf16_hi(w.y);
    f[4] = bf16_lo(w.z); f[5] = bf16_hi(w.z); f[6] = bf16_lo(w.w); f[7] = bf16_hi(w.w);
}
// ---- packed fp32 pairs (FFMA2 / FMUL2 / FADD2: one instruction per two lanes of math).  The elementwise phases are bound
// by the length of each warp's dependent instruction stream, not by the FP32 pipe, so halving the instruction count of
// the arithmetic shortens them (measured: same ~4.5-cycle dependent latency as the scalar forms).
__device__ __forceinline__ unsigned long long f2_bits(float2 a) { return *reinterpret_cast<unsigned long long*>(&a); }
__device__ __forceinline__ float2 f2_from(unsigned long long r) { return *reinterpret_cast<float2*>(&r); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c)
{
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(f2_bits(a)), "l"(f2_bits(b)), "l"(f2_bits(c)));
    return f2_from(r);
}
__device__ __forceinline__ float2 mul2(float2 a, float2 b)
{
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_bits(a)), "l"(f2_bits(b)));
    return f2_from(r);
}
__device__ __forceinline__ float2 add2(float2 a, float2 b)
{
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_bits(a)), "l"(f2_bits(b)));
    return f2_from(r);
}
__device__ __forceinline__ float2 splat2(float x) { return make_float2(x, x); }
__device__ __forceinline__ void unpack8p(uint4 w, float2 (&f)[4])
{
    f[0] = make_float2(bf16_lo(w.x), bf16_hi(w.x)); f[1] = make_float2(bf16_lo(w.y), bf16_hi(w.y));
    f[2] = make_float2(bf16_lo(w.z), bf16_hi(w.z)); f[3] = make_float2(bf16_lo(w.w), bf16_hi(w.w));
}
__device__ __forceinline__ uint4 pack8p(const float2* f)
{
    return make_uint4(pack_bf16(f[0].x, f[0].y), pack_bf16(f[1].x, f[1].y), pack_bf16(f[2].x, f[2].y), pack_bf16(f[3].x, f[3].y));
}
__device__ __forceinline__ float2 pair_of(const uint32_t* v) { return make_float2(__uint_as_float(v[0]), __uint_as_float(v[1])); }
__device__ __forceinline__ uint4 pack8(const float* f)
{
    return make_uint4(pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
}

}  // namespace tcp
}  // namespace carve

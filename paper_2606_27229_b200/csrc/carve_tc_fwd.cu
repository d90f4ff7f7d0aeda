// carve_tc_fwd.cu -- tensor-core forward of the CARVE layer operator for bf16 token tensors
// (tcgen05.mma with TMEM accumulators, operands staged by TMA, fp32 state kept on chip).
//
// One persistent CTA per (batch, head) chain walks the sequence in solve chunks of LC = 64 tokens
// (a gate chunk of L = 128 is two solve chunks that share one folded readout G_c; L = 16, 32 run
// as short solve chunks).  Per solve chunk, in the order of PAPER.md Alg. 1-2 (l.160-196, l.315-365):
//   P0  G^T = S^T [Ub;Uw]^T                       fold, Eq. 7 (l.134)                       [tcgen05]
//   P2  Z = [k;q] G^T, tt = tanh(Z rnorm_q)       bottleneck, Eq. 7                          [tcgen05]
//   P4  [b_proj | w_proj] = [tt_b | tt_w] [Vb | Vw]^T    up-projections, Eq. 8 (l.140)      [tcgen05]
//   P5  V' = sigmoid(wx + w_proj) v;  la = g - softplus(bx + b_proj)  (= log a_t, Eq. 9 l.151, Eq. 14 l.310);
//       block-local prefix sums of la over the 16 tokens of an anchor block: segmented warp scan in fp32 registers
//   P7  decayed operands, every exponent relative to the start of a 16-token anchor block:
//       Kbar_t = k^_t gamma_{t-1}, Qbar_t = q^_t gamma_t, C_s = k^_s gamma_a/gamma_s, Ktil_t = k^_t gamma_L/gamma_t
//   P8  A|P blocks = [Kbar;Qbar] C^T (Eq. 15 l.342);  [Kbar;Qbar] S^T (Alg. 2 steps 5, 8)   [tcgen05]
//   P9  beta A, P (masked), beta R = beta (V' - Kbar S^T);  WY solve U = (I + diag(beta) A)^-1 beta R by blocked forward
//       substitution in registers (Alg. 2 step 7), T = (I + diag(beta) A)^-1 for the chunk record   [mma.sync tf32]
//   P12 O += P U (step 8);  W = U^T Ktil (step 9)                                          [tcgen05]
//   P13 O -> bf16 tile -> TMA store;  S <- S diag(gamma_L) + W  (fp32, TMEM), bf16 copy for the next chunk's MMAs
// Decay ratios: with log a ~ -1.6 per token gamma_L reaches e^-100 per chunk, so no 1/gamma is ever
// formed over more than one 16-token block; across blocks only ratios <= 1 are multiplied in.
#include <mutex>

#include "carve_tc.cuh"

namespace carve {
namespace {

using namespace tcp;
PROF_DECL(g_prof_fwd)
PROFB_DECL(g_profb_fwd)

struct TcArgs {
    int B, H, T, L, r;
    int dvf;        // full d_v of the tensors (= VS x the value channels one CTA owns)
    int l2norm;
    int sw;         // scalar-write variant (wx = Uw = Vw = NULL, P l.145): w == 1, V' = v, no write-gate load / projection / sigmoid
    float scale, eps;
    const __nv_bfloat16* beta;
    const float *A, *tau, *Ub, *Uw, *Vb, *Vw, *S0;
    __nv_bfloat16* O;
    float* S_final;
    uint8_t* rec;   // [chains][T/LC] chunk records (carve_tc.cuh Rec) for the reverse kernel, or nullptr
};

// Runtime-shaped product from two row tiles (see tc_common.cuh umma_tiles_rt); M fixed at compile time.
template <int M, int AMAJ, int BMAJ, int KMAX = 128>
__device__ __forceinline__ void mma_rt(uint32_t d_tmem, int N, uint32_t a_saddr, int a_rows, int a_o0, uint32_t b_saddr,
                                       int b_rows, int b_o0, int K, bool accumulate)
{
    umma_prod<AMAJ, BMAJ, KMAX>(d_tmem, M, N, a_saddr, a_rows, a_o0, 0, b_saddr, b_rows, b_o0, 0, K, accumulate);
}

// fp32 scratch matrices of the triangular inverse: [64][64], columns XOR-swizzled by the row.
__device__ __forceinline__ int mm_idx(int r, int c) { return r * 64 + (c ^ ((r & 7) << 2)); }

__device__ __forceinline__ void mma_tf32(float (&d)[4], const uint32_t (&a)[4], const uint32_t (&b)[2])
{
    asm volatile(
        "mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}

__device__ __forceinline__ void ldsm_x4_trans(uint32_t (&r)[4], uint32_t saddr)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
                 : "r"(saddr));
}
__device__ __forceinline__ void stsm_x4_trans(uint32_t saddr, const uint32_t (&r)[4])
{
    asm volatile("stmatrix.sync.aligned.m8n8.x4.trans.shared.b16 [%0], {%1,%2,%3,%4};" ::"r"(saddr), "r"(r[0]), "r"(r[1]),
                 "r"(r[2]), "r"(r[3])
                 : "memory");
}

// 8x8 diagonal blocks of (I + Mm)^-1 -> Tm by forward substitution (thread = (block, column)); Mm strictly lower.
__device__ __forceinline__ void diag8_inverse(const float* Mm, float* Tm, int n, int tid)
{
    if (tid < n) {
        const int c = tid & 7, o = 8 * (tid >> 3);
        float x[8];
#pragma unroll
        for (int tt = 0; tt < 8; ++tt) {
            float acc = 0.f;
#pragma unroll
            for (int s = 0; s < tt; ++s) acc += Mm[mm_idx(o + tt, o + s)] * x[s];
            x[tt] = (tt == c) ? 1.f : (tt < c ? 0.f : -acc);
            Tm[(o + tt) * 8 + c] = x[tt];   // [64][8]: the 8x8 diagonal blocks only
        }
    }
}

// WY solve, Alg. 2 step 7: X (I + Mm)^T = RHS for X = U^T (value channels x tokens) and, on four
// more warps, for X = T^T with RHS = I (the inverse itself, which the chunk record keeps for the backward).  Blocked
// forward substitution over 8-token blocks, entirely in registers on tf32 mma.sync (m16n8k8): a warp owns 16 rows of X
// (value channels, or columns of T) and walks the token blocks i = 0.. in order,
//     X_i = (RHS_i - sum_{j<i} X_j N_ij^T) T_ii^T,      N = Mm (= diag(beta) A), T_ii = 8x8 diagonal inverses (Tm).
// The accumulator fragment of X_j (row g: tokens 2 l4, 2 l4 + 1) is reused as the A operand of the later products with
// the contraction index permuted (slot l4 <- token 2 l4, slot l4 + 4 <- token 2 l4 + 1); the B operand N_ij^T is then
// the fp32 pair Mm[8i + g][8j + 2 l4 .. + 1].  No shared-memory round trip and no barrier between dependent products:
// one product is ~30 cycles of latency against ~1 K for a tcgen05 round trip, which is why this 64 x 64 solve is not
// on the tcgen05 pipe.  RHS = beta R comes from the bf16 row tile `rhs` ([64][DVC], ldmatrix.trans); U goes back as a
// bf16 row tile (stmatrix.trans) over V', T into rows 0..63 of the 128-row tile `tp`.
template <int DVC, bool WANT_T>
__device__ __forceinline__ void wy_solve(const float* Mm, const float* Tm, int n, int warp, int lane, uint32_t rhs_saddr,
                                         uint32_t us_saddr, uint32_t tp_saddr)
{
    constexpr int NUW = DVC / 16;   // warps solving for U
    const bool is_u = warp < NUW;
    const int m0 = is_u ? 16 * warp : 16 * (warp - NUW);
    // (T only feeds the chunk record: the inference kernel skips it -- its warps share the tensor pipe with the U-warps.
    //  A compile-time switch: as a run-time flag it cost the training forward 3-5 % at config 2.)
    if (!is_u && (!WANT_T || warp >= NUW + 4 || m0 >= n)) return;
    const int g = lane >> 2, l4 = lane & 3, nblk = n >> 3;
    const int mat = lane >> 3, lr = lane & 7;   // ldmatrix / stmatrix: this lane addresses row lr of matrix `mat`
    float x[8][4];
    uint32_t init[4][4];
    if (is_u) {
#pragma unroll
        for (int ip = 0; ip < 4; ++ip)
            if (2 * ip < nblk) ldsm_x4_trans(init[ip], rhs_saddr + tile_chunk_off(64, 8 * (2 * ip + (mat >> 1)) + lr, m0 / 8 + (mat & 1)));
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        if (i < nblk) {
            float y[4];
            if (is_u) {
                const uint32_t w0 = init[i >> 1][2 * (i & 1)], w1 = init[i >> 1][2 * (i & 1) + 1];
                y[0] = bf16_lo(w0); y[1] = bf16_hi(w0); y[2] = bf16_lo(w1); y[3] = bf16_hi(w1);
            } else {
                const int t0 = 8 * i + 2 * l4;
                y[0] = (m0 + g == t0) ? 1.f : 0.f; y[1] = (m0 + g == t0 + 1) ? 1.f : 0.f;
                y[2] = (m0 + g + 8 == t0) ? 1.f : 0.f; y[3] = (m0 + g + 8 == t0 + 1) ? 1.f : 0.f;
            }
            float s0[4] = {0.f, 0.f, 0.f, 0.f}, s1[4] = {0.f, 0.f, 0.f, 0.f};   // two chains: even / odd j
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                if (j < i) {
                    const float2 nb = *reinterpret_cast<const float2*>(&Mm[mm_idx(8 * i + g, 8 * j + 2 * l4)]);
                    const uint32_t af[4] = {__float_as_uint(x[j][0]), __float_as_uint(x[j][2]), __float_as_uint(x[j][1]),
                                            __float_as_uint(x[j][3])};
                    const uint32_t bf[2] = {__float_as_uint(nb.x), __float_as_uint(nb.y)};
                    if (j & 1) mma_tf32(s1, af, bf); else mma_tf32(s0, af, bf);
                }
            }
#pragma unroll
            for (int e = 0; e < 4; ++e) y[e] -= s0[e] + s1[e];
            const float2 tb = *reinterpret_cast<const float2*>(&Tm[(8 * i + g) * 8 + 2 * l4]);
            const uint32_t af[4] = {__float_as_uint(y[0]), __float_as_uint(y[2]), __float_as_uint(y[1]), __float_as_uint(y[3])};
            const uint32_t bf[2] = {__float_as_uint(tb.x), __float_as_uint(tb.y)};
#pragma unroll
            for (int e = 0; e < 4; ++e) x[i][e] = 0.f;
            mma_tf32(x[i], af, bf);
            if (i & 1) {   // blocks i-1, i complete: four 8x8 bf16 matrices (block, channel half), rows = tokens
                const uint32_t w[4] = {pack_bf16(x[i - 1][0], x[i - 1][1]), pack_bf16(x[i - 1][2], x[i - 1][3]),
                                       pack_bf16(x[i][0], x[i][1]), pack_bf16(x[i][2], x[i][3])};
                const int tok = 8 * (i - 1 + (mat >> 1)) + lr, ch = m0 / 8 + (mat & 1);
                stsm_x4_trans(is_u ? us_saddr + tile_chunk_off(64, tok, ch) : tp_saddr + tile_chunk_off(128, tok, ch), w);
            }
        }
    }
}

#define PHASE_SYNC()            \
    do {                        \
        fence_async_smem();     \
        tc_fence_before();      \
        __syncthreads();        \
        tc_fence_after();       \
    } while (0)
#define WAIT_MMA()                          \
    do {                                    \
        mbar_wait(&mi.bar_mma, mma_ph);     \
        mma_ph ^= 1u;                       \
        tc_fence_after();                   \
    } while (0)

// NP = number of column parts a tile row is split into = warpgroups per CTA (threads = 128 NP); every thread
// serves one TMEM lane (tile row) and DK/NP columns.
// VS = value split: a cluster of VS CTAs shares one chain, each owning DV of the d_v = VS*DV value channels.
// The value columns of R, U, O and S are independent of one another (Thm 11); only the fold
// G = [Ub;Uw] S sums over them, so the CTAs exchange their partial G through distributed shared memory once per
// chunk and redo the (cheap) key-axis work redundantly.
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

// SW = 1: scalar-write variant (wx = Uw = Vw = NULL, P l.145) -- w == 1, V' = v; compiled separately so that the full-gate
// kernel carries none of its branches.
// TRAIN != 0: the call writes chunk records (a.rec != NULL); TRAIN = 1 when in addition scale == 1.  FULL = 1: the solve chunk has all 64 tokens (L >= 64), so the
// live-row predicates and the anchor-block count are constants (L < 64 and the d = 128 training forward run the general
// FULL = 0 instance).
template <int DK, int DV, int NP, int VS, int SW, int TRAIN, int FULL, int RT = 0>   // RT != 0: the gate rank r as a constant
__global__ void __launch_bounds__(128 * NP, DK == 64 ? 2 : 1)
carve_fwd_tc_kernel(const TcArgs a, const __grid_constant__ CUtensorMap mq, const __grid_constant__ CUtensorMap mk,
                    const __grid_constant__ CUtensorMap mv, const __grid_constant__ CUtensorMap mf,
                    const __grid_constant__ CUtensorMap mbx, const __grid_constant__ CUtensorMap mwx,
                    const __grid_constant__ CUtensorMap mo)
{
    static_assert(DK == DV, "the shared-memory map assumes dk == dv");
    // TMEM column map: 4 regions of DK columns (d = 64: 256 columns, so that two CTAs fit the SM's 512)
    constexpr uint32_t TM_S = 0, TM_ACC = DK, TM_X1 = 2 * DK, TM_X2 = 3 * DK, TM_COLS = 4 * DK;
    constexpr int DM = DK > DV ? DK : DV;
    constexpr int NTH = 128 * NP;
    // issues (and waits for) the record's bulk copies: lane 0 of a Q-side warp of the last column part, which has
    // little or nothing to do in the phases that follow the copies (P9a/P9b/P11), unlike the MMA-issuing thread 0
    constexpr int REC_TID = NTH - 64;
    constexpr int HK = DK / NP, HV = DV / NP;  // columns per warpgroup ("half" = part index 0..NP-1)
    extern __shared__ uint8_t smem_raw[];
    // 1024-byte alignment by an offset from the __shared__ array (not by integer rounding of a generic pointer), so
    // that the compiler still knows these are shared-memory addresses: LDS/STS with 32-bit address arithmetic
    // instead of generic LD/ST with 64-bit arithmetic.
    uint8_t* sm = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const int r = RT ? RT : a.r, R2 = 2 * r;
    const Layout Lo(DK, DV, R2);
    using Misc = MiscT<DK>;
    Misc& mi = *reinterpret_cast<Misc*>(sm + Lo.misc);
    float* sBeta = mi.beta;
    const uint32_t sb = smem_u32(sm);
    float* Mm = reinterpret_cast<float*>(sm + Lo.Mm);
    float* Tm = reinterpret_cast<float*>(sm + Lo.Tm);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, q = warp & 3, half = warp >> 2;
    const int row = q * 32 + lane;   // tile row == TMEM lane served by this thread
    const bool krole = q < 2;
    const int t = row & 63;          // token of this row
    const uint32_t lane_base = (uint32_t)(q * 32) << 16;
    const int crank = VS > 1 ? (int)(blockIdx.x % VS) : 0;   // rank inside the cluster = which slice of value channels
    const int vofs = crank * DV;
    const int chain = blockIdx.x / VS, b = chain / a.H, h = chain % a.H;
    const int LCc = FULL == 1 ? LC : FULL > 1 ? FULL : (a.L < LC ? a.L : LC);   // (FULL = 16, 32: that chunk length)
    const int nchunks = a.T / LCc, gate_every = a.L / LCc;   // (a constant here was measured 4 % slower at d = 64)
    const bool warp_active = (q & 1) * 32 < LCc;  // this warp holds at least one live token row
    const bool live = t < LCc;

    PROF_INIT();
    // ---- one-time setup --------------------------------------------------------------------------
    if (tid == 0) {
        mbar_init(&mi.bar_mma, 1); mbar_init(&mi.bar_acc, 1); mbar_init(&mi.bar_kq, 1); mbar_init(&mi.bar_fb, 1); mbar_init(&mi.bar_wv, 1);
        mbar_fence_init();
        tma_prefetch_desc(&mq); tma_prefetch_desc(&mk); tma_prefetch_desc(&mv);
        tma_prefetch_desc(&mf); tma_prefetch_desc(&mbx); tma_prefetch_desc(&mwx); tma_prefetch_desc(&mo);
    }
    if (warp == 0) tmem_alloc(&mi.tmem_base, TM_COLS);
    for (int i = tid; i < R2 * DV; i += NTH) {
        const int ii = i / DV, x = i % DV;
        const float v = ii < r ? __ldg(a.Ub + (size_t)ii * a.dvf + vofs + x) : (SW ? 0.f : __ldg(a.Uw + (size_t)(ii - r) * a.dvf + vofs + x));
        *reinterpret_cast<__nv_bfloat16*>(sm + Lo.Ucat + tile_off(R2, ii, x)) = __float2bfloat16_rn(v);
    }
    for (int i = tid; i < DM * 64; i += NTH) {
        const int n = i / 64, c = i % 64;
        float v = 0.f;
        // each gate half padded to 16 columns, so that the two up-projections are separate K = 16 slices
        if (c < 16) { if (c < r && n < DK) v = __ldg(a.Vb + (size_t)n * r + c); }
        else if (c < 32) { if (c - 16 < r && n < DV && !SW) v = __ldg(a.Vw + (size_t)(vofs + n) * r + (c - 16)); }
        *reinterpret_cast<__nv_bfloat16*>(sm + Lo.Vcat + tile_off(DM, n, c)) = __float2bfloat16_rn(v);
    }
    for (int j = tid; j < 4 * DK; j += NTH) mi.etot[j / DK][j % DK] = 1.f;
    for (int j = tid; j < DK; j += NTH) {
        mi.eA[j] = a.A ? __expf(__ldg(a.A + h * DK + j)) : 1.f;
        mi.tau[j] = a.tau ? __ldg(a.tau + h * DK + j) : 0.f;
    }
    PHASE_SYNC();
    const uint32_t tmem = mi.tmem_base;
    const size_t state_tile = tile_bytes(DV, DK);
    const Rec Rc(DK, DV);
    // (the inference kernel sees a constant NULL here: all of the record code below compiles away)
    uint8_t* rec_chain = TRAIN ? a.rec + (size_t)chain * nchunks * Rc.total : nullptr;
    // scale == 1 (TRAIN = 1; TRAIN = 2 is a training call with another scale): then scale.P and scale.Qbar of the record
    // are the shared-memory tiles themselves, and the per-thread stores of the general case compile away
    const bool s1 = TRAIN == 1 ? true : a.scale == 1.f;

    // initial state: fp32 -> TMEM, bf16 -> Sb (and the workspace slot of chunk 0)
    if (row < DV) {
        const float* s0 = a.S0 ? a.S0 + ((size_t)chain * a.dvf + vofs + row) * DK : nullptr;
#pragma unroll
        for (int s = 0; s < HK; s += 32) {
            const int c0 = half * HK + s;
            uint32_t v[32];
#pragma unroll
            for (int e = 0; e < 32; e += 4) {
                float4 f4 = s0 ? __ldg(reinterpret_cast<const float4*>(s0 + c0 + e)) : make_float4(0.f, 0.f, 0.f, 0.f);
                v[e] = __float_as_uint(f4.x); v[e + 1] = __float_as_uint(f4.y);
                v[e + 2] = __float_as_uint(f4.z); v[e + 3] = __float_as_uint(f4.w);
            }
            tmem_st32(tmem + TM_S + lane_base + c0, v);
#pragma unroll
            for (int ch = 0; ch < 4; ++ch) {
                float f8[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) f8[e] = __uint_as_float(v[8 * ch + e]);
                const uint4 w = pack8(f8);
                const uint32_t off = tile_chunk_off(DV, row, c0 / 8 + ch);
                sts128(sm + Lo.Sb + off, w);
            }
        }
        tmem_wait_st();
    }

    auto sumsq = [&](int rw) {
        float ss = 0.f;
#pragma unroll
        for (int pp = 0; pp < NP; ++pp) ss += mi.nrm[rw][pp];
        return ss;
    };
    auto issue_kq = [&](int c) {
        mbar_expect_tx(&mi.bar_kq, 2u * LCc * DK * 2u);
        const int tr = b * a.T + c * LCc;
        for (int cb = 0; cb < DK / 64; ++cb) {
            tma_load_3d(sm + Lo.KQraw + cb * 128 * 128, &mk, &mi.bar_kq, cb * 64, h, tr);
            tma_load_3d(sm + Lo.KQraw + cb * 128 * 128 + 64 * 128, &mq, &mi.bar_kq, cb * 64, h, tr);
        }
    };
    auto issue_fb = [&](int c) {
        mbar_expect_tx(&mi.bar_fb, 2u * LCc * DK * 2u);
        const int tr = b * a.T + c * LCc;
        for (int cb = 0; cb < DK / 64; ++cb) {
            tma_load_3d(sm + Lo.F + cb * 64 * 128, &mf, &mi.bar_fb, cb * 64, h, tr);
            tma_load_3d(sm + Lo.BX + cb * 64 * 128, &mbx, &mi.bar_fb, cb * 64, h, tr);
        }
    };
    auto issue_wv = [&](int c) {
        mbar_expect_tx(&mi.bar_wv, (SW ? 1u : 2u) * LCc * DV * 2u);
        const int tr = b * a.T + c * LCc;
        for (int cb = 0; cb < DV / 64; ++cb) {
            if (!SW) tma_load_3d(sm + Lo.WX + cb * 64 * 128, &mwx, &mi.bar_wv, vofs + cb * 64, h, tr);
            tma_load_3d(sm + Lo.V + cb * 64 * 128, &mv, &mi.bar_wv, vofs + cb * 64, h, tr);
        }
    };
    if (VS > 1) { cluster_arrive(); cluster_wait(); }   // every CTA of the cluster runs before any distributed-shared-memory access
    if (tid == 0) { fence_async_smem(); issue_kq(0); issue_fb(0); issue_wv(0); }

    uint32_t mma_ph = 0, tma_ph = 0, acc_ph = 0;
    // Write strength of this thread's token: fetched at the top of the chunk by an asynchronous 4-byte copy (the aligned
    // word that holds the bf16 value) straight into the token's slot of mi.beta, and converted in place at the start of
    // P5, long after it has landed.  No register carries it: as a plain load one chunk ahead its register was spilled, and
    // the spill store waited for the load right there -- ~1.7 K cycles per chunk on the two warps everybody then waited for.
    const unsigned short* beta_bits = reinterpret_cast<const unsigned short*>(a.beta);
    PROF(g_prof_fwd, 38);   // one-time setup
    for (int c = 0; c < nchunks; ++c) {
        const bool fold_now = (c % gate_every) == 0;
        const size_t tok0 = (size_t)b * a.T + (size_t)c * LCc;  // first token of the chunk
        uint8_t* rc = TRAIN ? rec_chain + (size_t)c * Rc.total : nullptr;  // this chunk's record
        if (TRAIN) __builtin_assume(rc != nullptr);
        PROF(g_prof_fwd, 0);
        // ---- P0: fold G^T = S^T Ucat^T -> TM_X2[0, R2)
        PROFB_ARRIVE(0); PHASE_SYNC(); PROFB_AFTER(g_profb_fwd, 0);
        if (tid == 0 && c > 0) {   // the previous chunk's outputs (staged in Y2 by P13)
            for (int cb = 0; cb < DV / 64; ++cb) tma_store_3d(&mo, sb + Lo.Y2 + cb * 8192, vofs + cb * 64, h, b * a.T + (c - 1) * LCc);
            bulk_commit();
        }
        PROF(g_prof_fwd, 20);
        if (rc && tid == REC_TID) {   // record: state entering the chunk (Sb stays intact until P13)
            bulk_s2g(rc + Rc.SB, sb + Lo.Sb, (uint32_t)state_tile);
            bulk_commit();
        }
        if (fold_now && warp == NTH / 32 - 1) {   // (warps 0..3 have P1 behind this product)
            if (elect_one()) {
                mma_rt<128, MNMAJ, KMAJ, DV>(tmem + TM_X2, R2, sb + Lo.Sb, DV, 0, sb + Lo.Ucat, R2, 0, DV, false);
                umma_commit(&mi.bar_mma);
            }
            __syncwarp();
        }
        // meanwhile: raw k, q have landed -> partial sums of squares; beta
        PROF(g_prof_fwd, 27);
        mbar_wait(&mi.bar_kq, tma_ph);
        PROF(g_prof_fwd, 28);
        if (live) {
            float ss = 0.f;
#pragma unroll
            for (int ch = 0; ch < HK / 8; ++ch) {
                float f8[8];
                unpack8(lds128(sm + Lo.KQraw + tile_chunk_off(128, row, half * (HK / 8) + ch)), f8);
#pragma unroll
                for (int e = 0; e < 8; ++e) ss += f8[e] * f8[e];
            }
            mi.nrm[row][half] = ss;
            if (krole && half == 0) {
                const unsigned short* src = beta_bits + (tok0 + t) * a.H + h;
                asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(&sBeta[t])),
                             "l"(reinterpret_cast<uintptr_t>(src) & ~(uintptr_t)3)
                             : "memory");
                asm volatile("cp.async.commit_group;" ::: "memory");
            }
        }
        PROF(g_prof_fwd, 21);
        if (fold_now) {
            WAIT_MMA();
            PROF(g_prof_fwd, 1);
            // ---- P1: G^T (lanes j) -> bf16 into the spare columns [32, 32+R2) of the Vcat tile
            if (VS > 1) {
                // partial G^T of this CTA's value channels -> the peer's Y1 (fp32 [dk][32]); Y1 of the peer is free once it
                // has passed P8 of its previous chunk (second cluster barrier phase, armed there)
                if (c > 0) cluster_wait();
                if (half == 0 && q * 32 < DK) {
                    uint32_t raddr;
                    const uint32_t laddr = sb + Lo.Y1 + (uint32_t)row * 128u;
                    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(raddr) : "r"(laddr), "r"(crank ^ 1));
                    for (int c0 = 0; c0 < R2; c0 += 16) {
                        uint32_t v[16];
                        tmem_ld16(tmem + TM_X2 + lane_base + c0, v);
                        tmem_wait_ld();
#pragma unroll
                        for (int e = 0; e < 16; e += 4)
                            asm volatile("st.shared::cluster.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(raddr + (c0 + e) * 4), "r"(v[e]),
                                         "r"(v[e + 1]), "r"(v[e + 2]), "r"(v[e + 3])
                                         : "memory");
                    }
                }
                cluster_arrive();
                cluster_wait();
            }
            if (half == 0 && q * 32 < DK) {
                for (int c0 = 0; c0 < R2; c0 += 16) {
                    uint32_t v[16];
                    tmem_ld16(tmem + TM_X2 + lane_base + c0, v);
                    tmem_wait_ld();
                    float f[16];
#pragma unroll
                    for (int e = 0; e < 16; ++e) f[e] = __uint_as_float(v[e]);
                    if (VS > 1) {   // + the peer's partial
                        const float* pr = reinterpret_cast<const float*>(sm + Lo.Y1) + row * 32 + c0;
#pragma unroll
                        for (int e = 0; e < 16; ++e) f[e] += pr[e];
                    }
                    sts128(sm + Lo.Vcat + tile_chunk_off(DM, row, (32 + c0) / 8), pack8(f));
                    sts128(sm + Lo.Vcat + tile_chunk_off(DM, row, (32 + c0) / 8 + 1), pack8(f + 8));
                }
            }
        }
        PROF(g_prof_fwd, 2);
        // ---- P2: Z = [k;q] G^T -> TM_X2[32, 32+R2)
        PROFB_ARRIVE(1); PHASE_SYNC(); PROFB_AFTER(g_profb_fwd, 1);
        if (rc && tid == REC_TID) {   // record: the Vcat tile (its columns 32.. hold G^T) and the write strengths
            bulk_s2g(rc + Rc.GT, sb + Lo.Vcat, tile_bytes(DM, 64));
            bulk_commit();
        }
        if (warp == 0) {
            if (elect_one()) {
                mma_rt<128, KMAJ, MNMAJ, DK>(tmem + TM_X2 + 32, R2, sb + Lo.KQraw, 128, 0, sb + Lo.Vcat, DM, 32, DK, false);
                umma_commit(&mi.bar_mma);
            }
            __syncwarp();
        }
        WAIT_MMA();
        PROF(g_prof_fwd, 3);
        // ---- P3: tt = tanh(Z rnorm_q) -> [tt_b pad 16 | tt_w pad 16] (both row halves); the 2r <= 32 bottleneck columns
        //      are spread over the Q-side warps of all column parts, 8 columns (one 16-byte chunk) at a time
        if (!krole && warp_active) {
            const float rnq = a.l2norm ? rsqrtf(sumsq(row) + a.eps) : 1.f;
            const uint4 z4 = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
            for (int sc = half * (4 / NP); sc < (half + 1) * (4 / NP); ++sc) {
                if (8 * sc < R2) {
                    uint32_t v[8];
                    tmem_ld8(tmem + TM_X2 + 32 + lane_base + 8 * sc, v);
                    tmem_wait_ld();
                    if (live) {
                        float f[8];
#pragma unroll
                        for (int e = 0; e < 8; ++e) f[e] = tanh_fast(__uint_as_float(v[e]) * rnq);
                        const uint4 w = pack8(f);
                        const int dst = 8 * sc < r ? sc : 2 + (8 * sc - r) / 8;   // erase half | write half, each padded to 16
                        sts128(sm + Lo.Y1 + tile_chunk_off(128, 64 + t, dst), w);
                        sts128(sm + Lo.Y1 + tile_chunk_off(128, t, dst), w);
                    }
                } else if (live) {   // r = 8: the padding chunks 1 and 3
                    const int dst = 2 * (sc - R2 / 8) + 1;
                    sts128(sm + Lo.Y1 + tile_chunk_off(128, 64 + t, dst), z4);
                    sts128(sm + Lo.Y1 + tile_chunk_off(128, t, dst), z4);
                }
            }
        }
        PROF(g_prof_fwd, 4);
        // ---- P4: b_proj = [tt_b;tt_b] Vb^T -> TM_X1, w_proj = [tt_w;tt_w] Vw^T -> TM_X2 (both row halves get both)
        PROFB_ARRIVE(2); PHASE_SYNC(); PROFB_AFTER(g_profb_fwd, 2);
        if (rc && tid == REC_TID) {   // record: the K-side rows of the bottleneck tile (Y1 is rewritten in P7, after this thread's wait)
            bulk_s2g(rc + Rc.tt, sb + Lo.Y1, 8192);
            bulk_commit();
        }
        if (warp == 0) {
            if (elect_one()) {
                umma_prod<KMAJ, KMAJ, 16>(tmem + TM_X1, 128, DK, sb + Lo.Y1, 128, 0, 0, sb + Lo.Vcat, DM, 0, 0, 16, false);
                if (!SW) umma_prod<KMAJ, KMAJ, 16>(tmem + TM_X2, 128, DV, sb + Lo.Y1, 128, 0, 16, sb + Lo.Vcat, DM, 0, 16, 16, false);
                umma_commit(&mi.bar_mma);
            }
            __syncwarp();
        }
        PROF(g_prof_fwd, 29);
        mbar_wait(&mi.bar_fb, tma_ph);
        mbar_wait(&mi.bar_wv, tma_ph);
        PROF(g_prof_fwd, 30);
        WAIT_MMA();
        PROF(g_prof_fwd, 5);
        // ---- P5: gates and the retention prefix.  Both threads of a token (K-side lane t, Q-side lane 64+t) take half of
        //      the part's columns (two 16-byte chunks cc0, cc0+1) and do, for them: the write side V' = sigmoid(wx + w_proj) v,
        //      the erase side log a_t = g_t - softplus(bx + b_proj) (Eq. 9 l.151, Eq. 14 l.310), and the block-local
        //      prefix sums lg_t - lg_a over the 16 tokens of the anchor block -- a segmented warp scan in fp32 registers
        //      (a warp holds 32 consecutive tokens of one role), so log a never leaves the registers.
        float lg[16];
        const int cc0 = half * (HK / 8) + (krole ? 0 : HK / 16);
        if (krole && half == 0 && live) {   // the write strength has landed (see above): bf16 half of its word -> float, in place
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            const uint32_t w = *reinterpret_cast<const volatile uint32_t*>(&sBeta[t]);
            const bool hi = (((tok0 + t) * a.H + h) & 1) != 0;
            // clamped away from 0 so that e_t = u_t / beta_t exists (u_t changes by < 1e-30 |e_t|)
            sBeta[t] = fmaxf(__uint_as_float(hi ? (w & 0xFFFF0000u) : (w << 16)), 1e-30f);
        }
        if (warp_active) {
            const int blk = t >> 4;
            uint32_t pr16[16], pw16[16];
            tmem_ld16(tmem + TM_X1 + lane_base + 8 * cc0, pr16);
            if (!SW) tmem_ld16(tmem + TM_X2 + lane_base + 8 * cc0, pw16);
            tmem_wait_ld();
#pragma unroll
            for (int ci = 0; ci < 2; ++ci) {
                const int cc = cc0 + ci;
                const uint32_t off = tile_chunk_off(64, t, cc);
                if (live && !SW) {
                    float2 fw[4], fv[4];
                    unpack8p(lds128(sm + Lo.WX + off), fw);
                    unpack8p(lds128(sm + Lo.V + off), fv);
                    const float2 h2 = splat2(0.5f);
#pragma unroll
                    for (int e = 0; e < 4; ++e) {   // w = sigmoid(wx + w_proj) through one tanh.approx per element (sigmoid_tanh)
                        const float2 x = mul2(add2(fw[e], pair_of(pw16 + 8 * ci + 2 * e)), h2);
                        fw[e] = fma2(make_float2(tanh_fast(x.x), tanh_fast(x.y)), h2, h2);
                        fv[e] = mul2(fv[e], fw[e]);
                    }
                    sts128(sm + Lo.V + off, pack8p(fv));
                    if (rc) {
                        *reinterpret_cast<uint4*>(rc + Rc.W + rp_off(t, cc)) = pack8p(fw);
#pragma unroll
                        for (int e = 0; e < 4; ++e) fv[e] = mul2(fv[e], fma2(fw[e], splat2(-1.f), splat2(1.f)));
                        *reinterpret_cast<uint4*>(rc + Rc.VWX + rp_off(t, cc)) = pack8p(fv);
                    }
                }
                float fb[8], ff[8], bg[8], ea[8], ta[8];
                unpack8(lds128(sm + Lo.BX + off), fb);
                unpack8(lds128(sm + Lo.F + off), ff);
                *reinterpret_cast<float4*>(ea) = *reinterpret_cast<const float4*>(&mi.eA[8 * cc]);
                *reinterpret_cast<float4*>(ea + 4) = *reinterpret_cast<const float4*>(&mi.eA[8 * cc + 4]);
                *reinterpret_cast<float4*>(ta) = *reinterpret_cast<const float4*>(&mi.tau[8 * cc]);
                *reinterpret_cast<float4*>(ta + 4) = *reinterpret_cast<const float4*>(&mi.tau[8 * cc + 4]);
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    // sigmoid and softplus of the same argument share exp(-|pre|): 3 transcendental ops, not 4
                    const float pre = fb[e] + __uint_as_float(pr16[8 * ci + e]);
                    const float ex = ex2_ftz(-fabsf(pre) * kLog2e), s1p = 1.f + ex;
                    if (rc) {
                        const float rs = rcp_ftz(s1p);
                        bg[e] = pre >= 0.f ? rs : ex * rs;
                    }
                    const float g = -ea[e] * softplus_fast(ff[e] + ta[e]);
                    const float la = g - fmaf(kLn2, lg2_ftz(s1p), fmaxf(pre, 0.f));
                    lg[8 * ci + e] = live ? la : 0.f;
                }
                if (rc && live) *reinterpret_cast<uint4*>(rc + Rc.Bg + rp_off(t, cc)) = pack8(bg);
            }
#pragma unroll
            for (int d = 1; d < 16; d <<= 1) {
                const bool take = (lane & 15) >= d;
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const float o = __shfl_up_sync(0xFFFFFFFFu, lg[i], d, 16);
                    if (take) lg[i] += o;
                }
            }
            if (live && (lane & 15) == 15) {   // last token of its anchor block: exp of the block totals
#pragma unroll
                for (int e4 = 0; e4 < 4; ++e4)
                    *reinterpret_cast<float4*>(&mi.etot[blk][8 * cc0 + 4 * e4]) =
                        make_float4(exp_fast(lg[4 * e4]), exp_fast(lg[4 * e4 + 1]), exp_fast(lg[4 * e4 + 2]), exp_fast(lg[4 * e4 + 3]));
            }
        }
        PROF(g_prof_fwd, 6);
        if (tid == 0) bulk_wait_read();   // the output tile has left Y2 (rewritten below)
        if (rc && tid == REC_TID) bulk_wait_read();   // the previous chunk's [P;T] copy has left TP (d = 64: rewritten below; else in P9)
        fence_async_smem();   // (the block totals leave by a bulk copy)
        PROFB_ARRIVE(3); __syncthreads(); PROFB_AFTER(g_profb_fwd, 3);
        if (rc && tid == REC_TID) {   // record: exp of the block totals (blocks that do not exist at L < 64 hold 1)
            bulk_s2g(rc + Rc.etot, smem_u32(&mi.etot[0][0]), 16u * DK);
            bulk_s2g(rc + Rc.beta, smem_u32(mi.beta), 256);
            bulk_commit();
        }
        PROF(g_prof_fwd, 8);
        // ---- P7b: decayed operands.  Row operands exist in up to four anchorings: version 0 relative to the chunk
        //      start (Kbar, Qbar: also the operand of the state products), version jb relative to the start of
        //      anchor block jb (only rows at or after that block).  Column operand C_s is relative to its own block.
        if (warp_active) {
            const int blk = t >> 4;
            // smem address of chunk cc of the row of (version, role, token)
            auto ver_row = [&](int jb, bool qrole, int tok, int cc) -> uint8_t* {
                switch (jb) {
                    case 0: return sm + Lo.KQbar + tile_chunk_off(128, (qrole ? 64 : 0) + tok, cc);
                    case 1: return sm + Lo.V1 + tile_chunk_off(96, (qrole ? 48 : 0) + tok - 16, cc);
                    case 2: return sm + Lo.Y0 + tile_chunk_off(64, (qrole ? 32 : 0) + tok - 32, cc);
                    default: return sm + Lo.V3 + tile_chunk_off(32, (qrole ? 16 : 0) + tok - 48, cc);
                }
            };
            // Both threads of a token (K-side lane t, Q-side lane 64+t) hold +-(lg_t - lg_a) of the same columns: each
            // takes half of them and produces every decayed operand of the token for those columns.
            {
                const float rnq = a.l2norm ? rsqrtf(sumsq(64 + t) + a.eps) : 1.f;
                const float rnk = a.l2norm ? rsqrtf(sumsq(t) + a.eps) : 1.f;
                const int tn = t + 1;  // the key row that shares this token's retention (Kbar_{t+1} = k^_{t+1} gamma_t)
                const bool has_next = tn < LCc;
                const int bn = tn >> 4, krow = has_next ? tn : 0;
                const float rnkn = a.l2norm ? rsqrtf(sumsq(krow) + a.eps) : 1.f;
                if (rc && live && half == 0) reinterpret_cast<float*>(rc + Rc.rn)[row] = krole ? rnk : rnq;
#pragma unroll
                for (int ci = 0; ci < 2; ++ci) {
                    const int cc = cc0 + ci;
                    if (live) {
                        float2 Fp[4], qv[4], kv[4], o[4];
                        {   // column operand C_t, Ktil_t (own anchor), gamma_a/gamma_t >= 1
                            float2 kt[4], o1[4], o2[4], ic[4], et[4], sf[4];
                            unpack8p(lds128(sm + Lo.KQraw + tile_chunk_off(128, t, cc)), kt);
                            *reinterpret_cast<float4*>(et) = *reinterpret_cast<const float4*>(&mi.etot[blk][8 * cc]);
                            *reinterpret_cast<float4*>(et + 2) = *reinterpret_cast<const float4*>(&mi.etot[blk][8 * cc + 4]);
#pragma unroll
                            for (int e = 0; e < 4; ++e) sf[e] = splat2(1.f);   // gamma_L / gamma_e(blk): product of etot[b'] over b' > blk
#pragma unroll
                            for (int b2 = 3; b2 >= 1; --b2) {
                                if (b2 > blk) {
                                    float2 eb[4];
                                    *reinterpret_cast<float4*>(eb) = *reinterpret_cast<const float4*>(&mi.etot[b2][8 * cc]);
                                    *reinterpret_cast<float4*>(eb + 2) = *reinterpret_cast<const float4*>(&mi.etot[b2][8 * cc + 4]);
#pragma unroll
                                    for (int e = 0; e < 4; ++e) sf[e] = mul2(sf[e], eb[e]);
                                }
                            }
                            if (t == 0) {   // gamma_L of the chunk for these columns (state carry, P13)
                                float2 gl[4];
#pragma unroll
                                for (int e = 0; e < 4; ++e) gl[e] = mul2(sf[e], et[e]);
                                *reinterpret_cast<float4*>(&mi.gamL[8 * cc]) = *reinterpret_cast<const float4*>(gl);
                                *reinterpret_cast<float4*>(&mi.gamL[8 * cc + 4]) = *reinterpret_cast<const float4*>(gl + 2);
                            }
                            const float2 rnk2 = splat2(rnk);
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                const float2 l2 = mul2(make_float2(lg[8 * ci + 2 * e], lg[8 * ci + 2 * e + 1]), splat2(kLog2e));   // lg_t - lg_a <= 0
                                Fp[e] = make_float2(ex2_ftz(l2.x), ex2_ftz(l2.y));          // gamma_t / gamma_{a_blk}
                                const float2 cx = make_float2(ex2_ftz(-l2.x), ex2_ftz(-l2.y));   // gamma_{a_blk} / gamma_t >= 1
                                const float2 kh = mul2(kt[e], rnk2);
                                ic[e] = cx;
                                o1[e] = mul2(kh, cx);
                                o2[e] = mul2(kh, mul2(mul2(cx, et[e]), sf[e]));              // k^ gamma_L / gamma_t, every factor <= 1
                            }
                            const uint32_t off = tile_chunk_off(64, t, cc);
                            sts128(sm + Lo.Y1 + off, pack8p(o1));      // C_t
                            sts128(sm + Lo.Ktil + off, pack8p(o2));    // Ktil_t
                            if (rc) *reinterpret_cast<uint4*>(rc + Rc.IC + rp_off(t, cc)) = pack8p(ic);
                        }
                        unpack8p(lds128(sm + Lo.KQraw + tile_chunk_off(128, 64 + t, cc)), qv);
                        unpack8p(lds128(sm + Lo.KQraw + tile_chunk_off(128, krow, cc)), kv);
                        {
                            const float2 rnq2 = splat2(rnq), rnkn2 = splat2(rnkn);
#pragma unroll
                            for (int e = 0; e < 4; ++e) { qv[e] = mul2(qv[e], rnq2); kv[e] = mul2(kv[e], rnkn2); }
                        }
                        if (has_next && bn > blk) {  // first row of its block
                            sts128(ver_row(bn, false, tn, cc), pack8p(kv));
                            if (rc && (bn & 1)) *reinterpret_cast<uint4*>(rc + Rc.KQo + tile_chunk_off(128, tn, cc)) = pack8p(kv);
                        }
                        if (rc) *reinterpret_cast<uint4*>(rc + Rc.FQ + rp_off(t, cc)) = pack8p(Fp);
#pragma unroll
                        for (int jb = 3; jb >= 0; --jb) {
                            if (jb <= blk) {
#pragma unroll
                                for (int e = 0; e < 4; ++e) o[e] = mul2(qv[e], Fp[e]);
                                const uint4 wq = pack8p(o);
                                sts128(ver_row(jb, true, t, cc), wq);
                                if (rc && jb == blk && (blk & 1)) *reinterpret_cast<uint4*>(rc + Rc.KQo + tile_chunk_off(128, 64 + t, cc)) = wq;
                                if (rc && jb == 0 && !s1) {
                                    const float2 sc2 = splat2(a.scale);
#pragma unroll
                                    for (int e = 0; e < 4; ++e) o[e] = mul2(o[e], sc2);
                                    *reinterpret_cast<uint4*>(rc + Rc.Q0 + tile_chunk_off(64, t, cc)) = pack8p(o);
                                }
                                if (has_next) {
#pragma unroll
                                    for (int e = 0; e < 4; ++e) o[e] = mul2(kv[e], Fp[e]);
                                    const uint4 wk = pack8p(o);
                                    sts128(ver_row(jb, false, tn, cc), wk);
                                    if (rc && jb == blk && bn == blk && (blk & 1))
                                        *reinterpret_cast<uint4*>(rc + Rc.KQo + tile_chunk_off(128, tn, cc)) = wk;
                                }
                                if (jb > 0) {
                                    float2 eb[4];
                                    *reinterpret_cast<float4*>(eb) = *reinterpret_cast<const float4*>(&mi.etot[jb - 1][8 * cc]);
                                    *reinterpret_cast<float4*>(eb + 2) = *reinterpret_cast<const float4*>(&mi.etot[jb - 1][8 * cc + 4]);
#pragma unroll
                                    for (int e = 0; e < 4; ++e) Fp[e] = mul2(Fp[e], eb[e]);
                                }
                            }
                        }
                        if (!has_next) {  // Kbar_0 = k^_0
                            sts128(sm + Lo.KQbar + tile_chunk_off(128, 0, cc), pack8p(kv));
                        }
                    }
                }
            }
        }
        PROF(g_prof_fwd, 9);
        // ---- P8: A|P blocks (one 16-column block per anchoring) and the state products
        PROFB_ARRIVE(4); PHASE_SYNC(); PROFB_AFTER(g_profb_fwd, 4);
        PROF(g_prof_fwd, 18);
        // Issued by the last warp (Q side of the last column part): it has nothing to do in P9a / P9b, and the issuing
        // lane stays blocked for as long as these 40 instructions take to execute (the MMA queue is a few entries deep).
        if (warp == NTH / 32 - 1) {
            if (elect_one()) {
                const int nb = LCc >> 4;
                mma_rt<128, KMAJ, KMAJ, DK>(tmem + TM_X2, 16, sb + Lo.KQbar, 128, 0, sb + Lo.Y1, 64, 0, DK, false);
                if (nb > 1) mma_rt<128, KMAJ, KMAJ, DK>(tmem + TM_X2 + 16, 16, sb + Lo.V1, 96, 0, sb + Lo.Y1, 64, 16, DK, false);
                if (nb > 2) mma_rt<64, KMAJ, KMAJ, DK>(tmem + TM_X2 + 32, 16, sb + Lo.Y0, 64, 0, sb + Lo.Y1, 64, 32, DK, false);
                if (nb > 3) mma_rt<64, KMAJ, KMAJ, DK>(tmem + TM_X2 + 48, 16, sb + Lo.V3, 32, 0, sb + Lo.Y1, 64, 48, DK, false);
                umma_commit(&mi.bar_mma);   // the A|P blocks: P9a starts on them while the state products still run
                mma_rt<128, KMAJ, KMAJ, DK>(tmem + TM_ACC, DV, sb + Lo.KQbar, 128, 0, sb + Lo.Sb, DV, 0, DK, false);
                umma_commit(&mi.bar_acc);
                if (c + 1 < nchunks) {   // the next chunk's raw k, q -> L2 (their shared-memory tile is still the solve's scratch)
                    const int tr = b * a.T + (c + 1) * LCc;
                    for (int cb = 0; cb < DK / 64; ++cb) { tma_prefetch_3d(&mk, cb * 64, h, tr); tma_prefetch_3d(&mq, cb * 64, h, tr); }
                }
            }
            __syncwarp();
        }
        PROF(g_prof_fwd, 19);
        {
            const int nb = LCc >> 4;
            if (rc && tid == REC_TID) {
                // record: operand tiles straight from shared memory (bulk copies).  Only sources that stay intact until
                // the wait in P11 are used: Ktil, C, version 0 (Kbar/Qbar) and version 2 (Y0).  The rows of the odd
                // 16-token blocks (versions 1 and 3 live in Y2/TP, rewritten in P9) were stored by their threads in P7b.
                constexpr uint32_t TB = tile_bytes(64, DK);
                bulk_s2g(rc + Rc.KT, sb + Lo.Ktil, TB);
                bulk_s2g(rc + Rc.CC, sb + Lo.Y1, TB);
                for (int cb = 0; cb < DK / 64; ++cb) {
                    bulk_s2g(rc + Rc.K0 + cb * 8192, sb + Lo.KQbar + cb * 16384, 8192);                  // Kbar rows
                    if (s1) bulk_s2g(rc + Rc.Q0 + cb * 8192, sb + Lo.KQbar + cb * 16384 + 8192, 8192);   // Qbar rows
                    uint8_t* dst = rc + Rc.KQo + cb * 16384;
                    bulk_s2g(dst, sb + Lo.KQbar + cb * 16384, 2048);                 // block 0, K side (version 0)
                    bulk_s2g(dst + 8192, sb + Lo.KQbar + cb * 16384 + 8192, 2048);   // block 0, Q side
                    if (nb > 2) {
                        bulk_s2g(dst + 4096, sb + Lo.Y0 + cb * 8192, 2048);                  // block 2, K side (version 2)
                        bulk_s2g(dst + 8192 + 4096, sb + Lo.Y0 + cb * 8192 + 4096, 2048);    // block 2, Q side
                    }
                }
                bulk_commit();
            }
        }
        WAIT_MMA();
        if (VS > 1) cluster_arrive();   // C (Y1) is consumed: the peer may send the next chunk's partial G
        PROF(g_prof_fwd, 10);
        // ---- P9a: beta A -> Mm (fp32, only the strictly lower part is ever read), P -> TP rows 64.. (bf16, masked s <= t)
        {
            // one 16-column piece [16 jb, 16 jb + 16) of row `tok`
            auto put_piece = [&](bool qrole, int tok, int jb, const uint32_t (&v)[16]) {
                if (!qrole) {
                    const float bt = sBeta[tok];
#pragma unroll
                    for (int e = 0; e < 16; e += 4)   // (mm_idx swizzles whole groups of four columns: 16-byte stores)
                        *reinterpret_cast<float4*>(&Mm[mm_idx(tok, 16 * jb + e)]) =
                            make_float4(bt * __uint_as_float(v[e]), bt * __uint_as_float(v[e + 1]), bt * __uint_as_float(v[e + 2]),
                                        bt * __uint_as_float(v[e + 3]));
                } else {
                    float f[16];
#pragma unroll
                    for (int e = 0; e < 16; ++e) f[e] = (e <= tok - 16 * jb) ? __uint_as_float(v[e]) : 0.f;
                    sts128(sm + Lo.TP + tile_chunk_off(128, 64 + tok, 2 * jb), pack8(f));
                    sts128(sm + Lo.TP + tile_chunk_off(128, 64 + tok, 2 * jb + 1), pack8(f + 8));
                    if (rc && !s1) {  // the record keeps scale.P in rows 0..63 (scale = 1: bulk copy of the tile)
#pragma unroll
                        for (int e = 0; e < 16; ++e) f[e] *= a.scale;
                        *reinterpret_cast<uint4*>(rc + Rc.PT + tile_chunk_off(128, tok, 2 * jb)) = pack8(f);
                        *reinterpret_cast<uint4*>(rc + Rc.PT + tile_chunk_off(128, tok, 2 * jb + 1)) = pack8(f + 8);
                    }
                }
            };
            const int nb = LCc >> 4;
            uint32_t v[16];
            if (half == 0) {
                // version 0: lane = stacked row
                tmem_ld16(tmem + TM_X2 + lane_base, v);
                tmem_wait_ld();
                if (live) {
                    put_piece(!krole, t, 0, v);
                    if (!krole) {  // pieces above the row's own block are zero
                        const uint4 z4 = make_uint4(0u, 0u, 0u, 0u);
                        for (int jb = (t >> 4) + 1; jb < 4; ++jb) {
                            sts128(sm + Lo.TP + tile_chunk_off(128, 64 + t, 2 * jb), z4);
                            sts128(sm + Lo.TP + tile_chunk_off(128, 64 + t, 2 * jb + 1), z4);
                            if (rc && !s1) {
                                *reinterpret_cast<uint4*>(rc + Rc.PT + tile_chunk_off(128, t, 2 * jb)) = z4;
                                *reinterpret_cast<uint4*>(rc + Rc.PT + tile_chunk_off(128, t, 2 * jb + 1)) = z4;
                            }
                        }
                    }
                }
            }
            if (half == 2 % NP) {
                if (nb > 2) {
                    // version 2 (M = 64): compact row m = 16 q + lane sits in lane < 16 of warp q; m < 32: K token 32+m, else Q token m
                    tmem_ld16(tmem + TM_X2 + 32 + lane_base, v);
                    tmem_wait_ld();
                    if (lane < 16) {
                        const int tok = 32 + 16 * (q & 1) + lane;
                        if (tok < LCc) put_piece(q >= 2, tok, 2, v);
                    }
                }
            }
            if (half == 1) {
                if (nb > 1) {
                    // version 1 (M = 128 over a 96-row tile): lanes 0..47 K tokens 16.., lanes 48..95 Q tokens 16..
                    tmem_ld16(tmem + TM_X2 + 16 + lane_base, v);
                    tmem_wait_ld();
                    if (row < 96) {
                        const bool qr = row >= 48;
                        const int tok = 16 + (qr ? row - 48 : row);
                        if (tok < LCc) put_piece(qr, tok, 1, v);
                    }
                }
            }
            if (half == 3 % NP) {
                if (nb > 3) {
                    // version 3 (M = 64 over a 32-row tile): m < 16: K token 48+m (warp 0), 16 <= m < 32: Q token 32+m (warp 1)
                    tmem_ld16(tmem + TM_X2 + 48 + lane_base, v);
                    tmem_wait_ld();
                    if (lane < 16 && q < 2) put_piece(q == 1, 48 + lane, 3, v);
                }
            }
        }
        PROF(g_prof_fwd, 11);
        // ---- P9b: beta R = beta (V' - Kbar S^T) -> Y2 (rows t)
        mbar_wait(&mi.bar_acc, acc_ph);
        acc_ph ^= 1u;
        tc_fence_after();
        if (krole && warp_active) {
            const float bt = live ? sBeta[t] : 0.f;
            const float2 bt2 = splat2(bt), neg1 = splat2(-1.f);
            static_assert(HV == 32 && HK == 32, "one 32-column TMEM load per thread and phase");
            uint32_t v[32];
            tmem_ld32(tmem + TM_ACC + lane_base + half * HV, v);
            tmem_wait_ld();
            if (live) {
#pragma unroll
                for (int ch = 0; ch < 4; ++ch) {
                    float2 fv[4];
                    const uint32_t off = tile_chunk_off(64, t, half * 4 + ch);
                    unpack8p(lds128(sm + Lo.V + off), fv);
#pragma unroll
                    for (int e = 0; e < 4; ++e) fv[e] = mul2(bt2, fma2(pair_of(v + 8 * ch + 2 * e), neg1, fv[e]));
                    sts128(sm + Lo.Y2 + off, pack8p(fv));
                }
            }
        }
        PROFB_ARRIVE(5); __syncthreads(); PROFB_AFTER(g_profb_fwd, 5);
        PROF(g_prof_fwd, 12);
        // ---- P9c: WY solve U = (I + beta A)^-1 (beta R) in registers (tf32 mma.sync) -> bf16 rows over V'; T -> TP rows 0..63
        diag8_inverse(Mm, Tm, LCc, tid);
        PROFB_ARRIVE(6); __syncthreads(); PROFB_AFTER(g_profb_fwd, 6);
        PROF(g_prof_fwd, 26);
        wy_solve<DV, TRAIN != 0>(Mm, Tm, LCc, warp, lane, sb + Lo.Y2, sb + Lo.Us, sb + Lo.TP);
        // the record copies issued so far have left their buffers: the next chunk's loads (P13) may overwrite them
        if (rc && tid == REC_TID) bulk_wait_read();
        PROF(g_prof_fwd, 13);
        // ---- P12: O += P U;  W = U^T Ktil -> TM_X2
        PROFB_ARRIVE(7); PHASE_SYNC(); PROFB_AFTER(g_profb_fwd, 7);
        PROF(g_prof_fwd, 22);
        if (warp == 0) {
            if (elect_one()) {
                mma_rt<128, KMAJ, MNMAJ, LC>(tmem + TM_ACC, DV, sb + Lo.TP, 128, 0, sb + Lo.Us, 64, 0, LCc, true);
                mma_rt<128, MNMAJ, MNMAJ, LC>(tmem + TM_X2, DK, sb + Lo.Us, 64, 0, sb + Lo.Ktil, 64, 0, LCc, false);
                umma_commit(&mi.bar_mma);
                if (c + 1 < nchunks) issue_kq(c + 1);   // the inverse scratch (over the raw k|q tile at d = 128) is consumed
            }
            __syncwarp();
        }
        if (rc && tid == REC_TID) {
            // record [scale.P ; T] (the two row halves of TP swapped; TP is next written in P9 of the next chunk) and U
            // (its buffer is refilled by the next chunk's loads, issued by this thread at the end of P13)
            if (s1) bulk_s2g(rc + Rc.PT, sb + Lo.TP + 8192, 8192);
            bulk_s2g(rc + Rc.PT + 8192, sb + Lo.TP, 8192);
            bulk_s2g(rc + Rc.U, sb + Lo.Us, tile_bytes(64, DV));
            bulk_commit();
        }
        PROF(g_prof_fwd, 23);
        WAIT_MMA();
        PROF(g_prof_fwd, 16);
        // ---- P13: outputs and the state carry
        if (!krole && warp_active) {
            uint32_t v[32];
            tmem_ld32(tmem + TM_ACC + lane_base + half * HV, v);
            tmem_wait_ld();
            if (live) {
#pragma unroll
                for (int ch = 0; ch < 4; ++ch) {
                    float2 f[4];
#pragma unroll
                    for (int e = 0; e < 4; ++e) f[e] = mul2(splat2(a.scale), pair_of(v + 8 * ch + 2 * e));
                    // staged as a bf16 row tile over beta R (dead since the solve); a TMA store sends it to HBM after the
                    // next barrier: 16 KB of STG from one SM would hold the warps for ~500 cycles (27-32 B/clk per SM)
                    sts128(sm + Lo.Y2 + tile_chunk_off(64, t, half * 4 + ch), pack8p(f));
                }
            }
        }
        if (q * 32 < DV) {
            const bool last_chunk = c + 1 == nchunks;
#pragma unroll
            for (int s16 = 0; s16 < 2; ++s16) {
              uint32_t sv16[16], wv16[16];
              tmem_ld16(tmem + TM_S + lane_base + half * HK + 16 * s16, sv16);
              tmem_ld16(tmem + TM_X2 + lane_base + half * HK + 16 * s16, wv16);
              tmem_wait_ld();
#pragma unroll
              for (int c2 = 0; c2 < 2; ++c2) {
                const int cc = half * (HK / 8) + 2 * s16 + c2;
                float f[8];
                float2 gl[4];
                *reinterpret_cast<float4*>(gl) = *reinterpret_cast<const float4*>(&mi.gamL[8 * cc]);
                *reinterpret_cast<float4*>(gl + 2) = *reinterpret_cast<const float4*>(&mi.gamL[8 * cc + 4]);
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float2 y = fma2(pair_of(sv16 + 8 * c2 + 2 * e), gl[e], pair_of(wv16 + 8 * c2 + 2 * e));
                    f[2 * e] = y.x; f[2 * e + 1] = y.y;
                    sv16[8 * c2 + 2 * e] = __float_as_uint(y.x); sv16[8 * c2 + 2 * e + 1] = __float_as_uint(y.y);
                }
                const uint4 w = pack8(f);
                const uint32_t off = tile_chunk_off(DV, row, cc);
                sts128(sm + Lo.Sb + off, w);
                if (last_chunk) {
                    float* dst = a.S_final + ((size_t)chain * a.dvf + vofs + row) * DK + 8 * cc;
                    *reinterpret_cast<float4*>(dst) = make_float4(f[0], f[1], f[2], f[3]);
                    *reinterpret_cast<float4*>(dst + 4) = make_float4(f[4], f[5], f[6], f[7]);
                }
              }
              tmem_st16(tmem + TM_S + lane_base + half * HK + 16 * s16, sv16);
            }
            tmem_wait_st();
        }
        if (tid == REC_TID && c + 1 < nchunks) {   // U has left its buffer: the next chunk's gate and value tiles
            if (rc) bulk_wait_read();
            fence_async_smem();
            issue_fb(c + 1); issue_wv(c + 1);
        }
        tma_ph ^= 1u;
        PROF(g_prof_fwd, 17);
    }
    if (VS > 1) cluster_wait();   // pairs with the last arrive; also keeps this CTA's shared memory alive for the peer
    PHASE_SYNC();
    if (tid == 0) {   // the last chunk's outputs
        for (int cb = 0; cb < DV / 64; ++cb) tma_store_3d(&mo, sb + Lo.Y2 + cb * 8192, vofs + cb * 64, h, b * a.T + (nchunks - 1) * LCc);
        bulk_commit();
        bulk_wait_all();
    }
    if (rec_chain && (tid == 0 || tid == REC_TID)) bulk_wait_all();   // drain the record's bulk stores
    PROF(g_prof_fwd, 39);   // last output tile, drain
    PROF_FLUSH(g_prof_fwd)
    if (warp == 0) tmem_dealloc(tmem, TM_COLS);
}

// ---- host side ---------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    });
    return fn;
}

}  // namespace

// [B,T,H,d] bf16 seen as (d, H, B*T); one box = 64 channels x 1 head x `rows` tokens, 128B-swizzled.
bool tc_make_token_map(CUtensorMap* map, const void* base, int B, int T, int H, int d, int rows)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    cuuint64_t dims[3] = {(cuuint64_t)d, (cuuint64_t)H, (cuuint64_t)B * T};
    cuuint64_t strides[2] = {(cuuint64_t)d * 2, (cuuint64_t)H * d * 2};
    cuuint32_t box[3] = {64, 1, (cuuint32_t)rows};
    cuuint32_t es[3] = {1, 1, 1};
    return fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, es,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

#ifdef CARVE_PROFILE
extern "C" void carve_debug_profb_fwd(unsigned long long* out)
{
    cudaMemcpyFromSymbol(out, g_profb_fwd, sizeof(g_profb_fwd));
    static unsigned long long z[64 * 16];
    cudaMemcpyToSymbol(g_profb_fwd, z, sizeof(z));
}
extern "C" void carve_debug_prof_fwd(unsigned long long* out)
{
    cudaMemcpyFromSymbol(out, g_prof_fwd, sizeof(g_prof_fwd));
    unsigned long long z[80] = {};
    cudaMemcpyToSymbol(g_prof_fwd, z, sizeof(z));
}
#endif

bool tc_fwd_supported(const carve_params_t& p)
{
    if (p.dtype != CARVE_BF16 || p.r > 16) return false;
    if (p.dk == p.dv && (p.dk == 64 || p.dk == 128)) return true;
    return p.dk == 128 && p.dv == 256 && p.L <= 64;   // value channels split over a cluster of two CTAs (forward only)
}

size_t tc_state_tile_bytes(const carve_params_t& p) { return tc::tile_bytes(p.dv, p.dk); }
size_t tc_record_bytes(const carve_params_t& p) { return tcp::Rec(p.dk, p.dv).total; }

template <int D, int VS, int SW>
static cudaError_t launch_tc_fwd(const Args& a, uint8_t* rec, cudaStream_t st)
{
    const int LCc = a.L < tcp::LC ? a.L : tcp::LC;
    CUtensorMap mq, mk, mv, mf, mbx, mwx, mo;
    if (!tc_make_token_map(&mo, a.O, a.B, a.T, a.H, a.dv, LCc)) return cudaErrorInvalidValue;
    if (!tc_make_token_map(&mq, a.q, a.B, a.T, a.H, D, LCc) || !tc_make_token_map(&mk, a.k, a.B, a.T, a.H, D, LCc) ||
        !tc_make_token_map(&mv, a.v, a.B, a.T, a.H, a.dv, LCc) || !tc_make_token_map(&mf, a.f, a.B, a.T, a.H, D, LCc) ||
        !tc_make_token_map(&mbx, a.bx, a.B, a.T, a.H, D, LCc) ||
        !tc_make_token_map(&mwx, a.wx ? a.wx : a.v, a.B, a.T, a.H, a.dv, LCc))   // (scalar-write variant: the map is never used)
        return cudaErrorInvalidValue;
    TcArgs t{};
    t.B = a.B; t.H = a.H; t.T = a.T; t.L = a.L; t.r = a.r; t.l2norm = a.l2norm; t.scale = a.scale; t.eps = a.eps;
    t.dvf = a.dv; t.sw = a.wx == nullptr;
    t.beta = static_cast<const __nv_bfloat16*>(a.beta);
    t.A = a.A; t.tau = a.tau; t.Ub = a.Ub; t.Uw = a.Uw; t.Vb = a.Vb; t.Vw = a.Vw; t.S0 = a.S0;
    t.O = static_cast<__nv_bfloat16*>(a.O); t.S_final = a.S_final; t.rec = rec;
    const size_t smem = tcp::Layout(D, D, 2 * a.r).total;
    constexpr int NP = D / 32;   // 32 columns per thread: 256 threads at d = 64, 512 at d = 128
    // FULL instance for L >= 64, except the d = 128 training kernel: there the specialised code was measured 7 % slower
    // (48 instead of 16 bytes of spills at the 128-register cap), while it gains 8-19 % everywhere else
    const bool full = a.L >= tcp::LC && !(rec && D == 128 && a.scale != 1.f);
    const bool one = a.scale == 1.f;
    auto kern = full ? carve_fwd_tc_kernel<D, D, NP, VS, SW, 0, 1> : carve_fwd_tc_kernel<D, D, NP, VS, SW, 0, 0>;
    if constexpr (VS == 1) {   // (the value-split cluster is inference only: no training instances of it are compiled)
        if (rec)
            kern = one ? (full ? carve_fwd_tc_kernel<D, D, NP, VS, SW, 1, 1> : carve_fwd_tc_kernel<D, D, NP, VS, SW, 1, 0>)
                       : (full ? carve_fwd_tc_kernel<D, D, NP, VS, SW, 2, 1> : carve_fwd_tc_kernel<D, D, NP, VS, SW, 2, 0>);
    } else if (rec) {
        return cudaErrorInvalidValue;
    }
    {   // the configs' rank (r = 16 at d = 128, r = 8 at d = 64) as a constant: full chunks, scale = 1
        constexpr int RC = D == 128 ? 16 : 8;
        if (full && a.r == RC && !rec) kern = carve_fwd_tc_kernel<D, D, NP, VS, SW, 0, 1, RC>;
        if constexpr (VS == 1) {
            if (full && a.r == RC && rec && one) kern = carve_fwd_tc_kernel<D, D, NP, VS, SW, 1, 1, RC>;
        }
    }
    if constexpr (D == 128 && VS == 1 && SW == 0) {   // config 2's short chunks: the chunk length as a constant as well
        if (a.r == 16) {
            if (a.L == 16 && !rec) kern = carve_fwd_tc_kernel<D, D, NP, VS, SW, 0, 16, 16>;
            if (a.L == 32 && !rec) kern = carve_fwd_tc_kernel<D, D, NP, VS, SW, 0, 32, 16>;
            if (a.L == 16 && rec && one) kern = carve_fwd_tc_kernel<D, D, NP, VS, SW, 1, 16, 16>;
            if (a.L == 32 && rec && one) kern = carve_fwd_tc_kernel<D, D, NP, VS, SW, 1, 32, 16>;
        }
    }
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100);   // (two CTAs per SM at d = 64)
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)(a.B * a.H * VS));
    cfg.blockDim = dim3(128 * NP);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = VS; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, t, mq, mk, mv, mf, mbx, mwx, mo);
}

cudaError_t tc_fwd_launch(const Args& a, uint8_t* rec, cudaStream_t st)
{
    const bool sw = a.wx == nullptr;
    if (a.dk == 128 && a.dv == 256) return sw ? cudaErrorInvalidValue : launch_tc_fwd<128, 2, 0>(a, rec, st);   // inference only: two CTAs per chain
    if (a.dk == 128) return sw ? launch_tc_fwd<128, 1, 1>(a, rec, st) : launch_tc_fwd<128, 1, 0>(a, rec, st);
    if (a.dk == 64) return sw ? launch_tc_fwd<64, 1, 1>(a, rec, st) : launch_tc_fwd<64, 1, 0>(a, rec, st);
    return cudaErrorInvalidValue;
}

}  // namespace carve

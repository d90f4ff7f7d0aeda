// carve_tc_bwd.cu -- tensor-core backward of the CARVE layer operator for bf16 token tensors.
//
// One persistent CTA per (batch, head) chain walks the solve chunks in REVERSE with the running state
// adjoint dS (d_v x d_k fp32) resident in TMEM.  It is the chunk-matrix adjoint of Alg. 2 (PAPER.md
// l.315-365), i.e. the reverse scan of Alg. 4 (l.788-817) batched over a chunk, with the fold glue of
// Alg. 5 (l.844-848) at every chunk start.  Nothing of the forward is recomputed on this serial chain:
// the training forward (carve_tc_fwd.cu) left a "chunk record" of operand tiles (carve_tc.cuh Rec) that
// is streamed in with bulk copies.  Per chunk, with S = state entering it, dS' = adjoint of the state
// leaving it (all MMAs are tcgen05, M = 128: rows 0..63 "K side", rows 64..127 "Q side"):
//   L1  dU  = Ktil dS'^T + (scale P)^T dO                 [rows 0..63]     dKtil = U dS'
//   L2  dX  = T^T dU (transposed solve, Alg. 2 step 7)    [rows 64..127]
//       dR = beta dX,  dbeta = <dX, e>,  dv = dR w,  dw_pre = dR v w (1-w)   (Alg. 4 l.806-808)
//   L3  [dA;dP] = [-dR; dO] U^T,   SP = [-dR; dO] S,   dS = dS' diag(gamma_L) + [-dR; dO]^T [Kbar; scale Qbar]
//   L4  pairwise decay terms on mma.sync (registers allow the per-block rescaling tcgen05 cannot do):
//         PK_t = sum_{s<t} dA_ts k^_s gamma_a(t)/gamma_s,  PQ_t likewise from dP,
//         PC_s = sum_t [dA;dP]_ts [k^_t gamma_{t-1}; q^_t gamma_t] / gamma_a(s)
//       every ratio anchored at a 16-token block boundary, products of whole-block decays applied
//       by Horner steps between the block products (all factors <= 1 except one block's worth).
//   L5  dk^ = dkA + dkC, dq^ (state part), X = contributions to d log gamma
//   L6  d log a = reverse cumulative sum of X over tokens = (0/1 triangular) x X on the tensor core
//       db_pre = -dla b  (Eq. 14 l.310), dla itself goes to the epilogue kernel (df, dA, dtau)
//   L7  [dz_b | dz_w] = [db_pre; dw_pre] [Vb | Vw],  dVb, dVw += [db_pre; dw_pre]^T [tt_b | tt_w]
//   L8  dq^ += dz G,  dG = dz^T q^                        (Eq. 7 l.134 backward)
//   L9  dS += [Ub;Uw]^T dG,  d[Ub;Uw] += dG S^T            (fold glue, Alg. 5 l.846-848)
//   L10 dS -> bf16 operand copy, column sums of S . dS (the retention gradient carried into the
//       previous chunk), dS0 at the end.
// The chunk-local tail (L2-norm backward of q,k, decay activation backward, dA/dtau) runs as a
// separate fully parallel kernel over (chain, chunk): carve_bwd_tc_epilogue_kernel below.
// No floating-point atomics anywhere: results are run-to-run bitwise identical.
#include "carve_tc.cuh"

namespace carve {
namespace {

using namespace tcp;
PROF_DECL(g_prof_bwd)
PROFB_DECL(g_profb_bwd)

struct BwdArgs {
    int B, H, T, L, r;
    int l2norm;
    int sw;       // scalar-write variant (wx = Uw = Vw = NULL): w == 1, no write-gate adjoint, dwx / dUw / dVw not produced
    float scale, eps;
    const uint8_t* rec;
    const float* dS_final;
    const float *Ub, *Uw, *Vb, *Vw;
    __nv_bfloat16 *dq, *dk, *dv, *df, *dbx, *dwx, *dbeta;
    float* dS0;
    float* part;
    int part_stride;
    float* dgs;   // [chains][dk][32] dG^T of the later solve chunk of a gate chunk (L = 128)
    int* flags;   // [chains] number of chunks whose outputs are complete (read by the overlapped epilogue kernel)
};

// TMEM column map of the reverse kernel.
constexpr uint32_t BM_DS = 0;     // [dv lanes][dk]  dS (fp32), pre-scaled by gamma_L of the chunk being processed
constexpr uint32_t BM_A = 128;    // L1 dU (rows 0..63), L2 dX (rows 64..127), L3.. SP, then dq^ (rows 64..127)
constexpr uint32_t BM_KT = 256;   // L1 dKtil (rows 0..63), L6 d log a (rows 0..63)
constexpr uint32_t BM_DAP = 384;  // L3 [dA;dP] raw (64 cols); L7 ZZ (32 cols); L8 dG^T at +32 (32 cols)
constexpr uint32_t BM_WG = 448;   // [n lanes][32]  dVb | dVw, accumulated over the whole chain
constexpr uint32_t BM_WU = 480;   // [x lanes][32]  d[Ub;Uw]^T, accumulated over the whole chain

constexpr uint32_t SLOT = 16384;
struct BLayout {  // byte offsets into the 1024-aligned dynamic shared memory
    uint32_t DSB, SBq, S[7], TRI, X, VcT, Ucat, FI, misc, total;
    __host__ __device__ BLayout(int d)
    {
        uint32_t o = 0;
        auto take = [&](uint32_t n) { uint32_t r = o; o += (n + 1023u) & ~1023u; return r; };
        DSB = take(tile_bytes(d, d));   // bf16 dS' (rows x, cols j)
        SBq = take(tile_bytes(d, d));   // bf16 state entering the chunk (record SB)
        for (int i = 0; i < 7; ++i) S[i] = take(SLOT);
        TRI = take(8192);               // [64][64] 0/1: t' > t; its MN-major view is t' < t
        X = take(SLOT);                 // dw_pre (L2 .. L7: staged dwx, then the L7 operand), then dz (L7 .. L8)
        VcT = take(tile_bytes(32, d));  // rows i: [Vb^T ; Vw^T]
        Ucat = take(tile_bytes(32, d)); // rows i: [Ub ; Uw]
        // staging of row-private record tiles (FQ | IC, later b): over DSB once dS' is consumed when it fits (d = 128)
        FI = tile_bytes(d, d) >= 2 * tile_bytes(64, d) ? DSB : take(2 * tile_bytes(64, d));
        misc = take(9216);
        total = o + 1024;
    }
};

struct BMisc {
    float etot[4][128];   // exp(block sums of log a) of the chunk
    float gamLn[128];     // gamma_L of the chunk processed next (c - 1)
    float extra[128];     // column sums of S . dS: d log gamma carried in from the later chunks
    float rn[128];        // 1/|k|, 1/|q| of the chunk's tokens
    float beta[64];
    union {               // dbp lives from L2 to the start of L3, pre from L4 to L5
        float dbp[8][64];     // dbeta partial sums of the column parts of the two sides
        float pre[4][128];    // gamma_a(b)/gamma_{-1}: product of etot[b'] over b' < b
    };
    union {               // thread j turns its four column-sum partials into suf[.][j]: same addresses, no hazard
        float colp[4][128];   // column-sum partials per lane quadrant
        float suf[4][128];    // gamma_L/gamma_a(b): product of etot[b'] over b' >= b
    };
    uint64_t bar_mma, bar_g1, bar_g3, bar_sb, bar_g4a, bar_g4b, bar_g5, bar_g8, bar_fi, bar_bg, bar_pt;
    uint32_t tmem_base;
};
static_assert(sizeof(BMisc) <= 9216, "misc area too small");

// ---- PTX helpers ----------------------------------------------------------------------------------
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t (&r)[4], uint32_t saddr)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
                 : "r"(saddr));
}
__device__ __forceinline__ void ldsm_x4(uint32_t (&r)[4], uint32_t saddr)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
                 : "r"(saddr));
}
__device__ __forceinline__ void mma_bf16(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1)
{
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint4 ldg128(const uint8_t* p) { return __ldg(reinterpret_cast<const uint4*>(p)); }
__device__ __forceinline__ void stg128(void* p, uint4 v) { *reinterpret_cast<uint4*>(p) = v; }

// Product over K (multiple of 16) from two row tiles, with explicit K offsets (tc_common.cuh umma_tiles_rt), M = 128.
template <int AMAJ, int BMAJ, int KMAX>
__device__ __forceinline__ void mma_k(uint32_t d_tmem, int N, uint32_t a_saddr, int a_rows, int a_o0, int a_k0,
                                      uint32_t b_saddr, int b_rows, int b_o0, int b_k0, int K, bool accumulate)
{
    umma_prod<AMAJ, BMAJ, KMAX>(d_tmem, 128, N, a_saddr, a_rows, a_o0, a_k0, b_saddr, b_rows, b_o0, b_k0, K, accumulate);
}
// The MMA / bulk-copy issuing thread: the elected lane of warp 0, inside a warp-uniform branch (tc_common.cuh umma_prod).
#define LEADER_BEGIN if (warp == LEADER_WARP) { if (elect_one()) {
#define LEADER_END } __syncwarp(); }

// Column sums over the 32 lanes of a warp by a halving butterfly: on return lane l holds in v[0..N/32)
// the sums of columns (N/32) l + i.
template <int n, int s, int N>
__device__ __forceinline__ void colsum_stage(float (&v)[N], int lane)
{
    const bool up = (lane & s) != 0;
#pragma unroll
    for (int i = 0; i < n / 2; ++i) {
        const float send = up ? v[i] : v[i + n / 2];
        const float keep = up ? v[i + n / 2] : v[i];
        v[i] = keep + __shfl_xor_sync(0xFFFFFFFFu, send, s);
    }
}
template <int N>
__device__ __forceinline__ void warp_colsum(float (&v)[N], int lane)
{
    colsum_stage<N, 16, N>(v, lane);
    colsum_stage<N / 2, 8, N>(v, lane);
    colsum_stage<N / 4, 4, N>(v, lane);
    colsum_stage<N / 8, 2, N>(v, lane);
    colsum_stage<N / 16, 1, N>(v, lane);
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

// NP = column parts per tile row = warpgroups per CTA (threads = 128 NP): 32 columns per thread.
// SW = 1: scalar-write variant (w == 1), compiled separately.  FULL = 1: the solve chunk has all 64 tokens (L >= 64), so
// the live-row predicates and the anchor-block count are constants.
// RT != 0: the gate rank r as a constant of the instance (the configs' r = 16 at d = 128, r = 8 at d = 64, full chunks).
template <int D, int NP, int SW, int FULL, int RT = 0>
__global__ void __launch_bounds__(128 * NP, 1)
carve_bwd_tc_kernel(const BwdArgs a, const __grid_constant__ CUtensorMap mdO, const __grid_constant__ CUtensorMap mq,
                    const __grid_constant__ CUtensorMap mdq, const __grid_constant__ CUtensorMap mdk,
                    const __grid_constant__ CUtensorMap mdv, const __grid_constant__ CUtensorMap mdf,
                    const __grid_constant__ CUtensorMap mdbx, const __grid_constant__ CUtensorMap mdwx)
{
    constexpr int NTH = 128 * NP;
    constexpr int LEADER_WARP = NTH / 32 - 1;   // MMA issuer: the last warp (see L1)
    // The six per-token gradient tiles of a chunk are staged in shared memory (in place over operands that are dead by
    // then) and leave by TMA stores issued by this one thread (bulk groups are per thread); it also issues the loads that
    // overwrite a staging tile, after cp.async.bulk.wait_group.read, and publishes the chain's progress flag.
    constexpr int STORE_TID = NTH - 64;
    constexpr int HK = D / NP;                     // columns per warpgroup ("half" = part index 0..NP-1)
    constexpr uint32_t TB = tile_bytes(64, D);     // one [64][D] tile
    constexpr uint32_t SBb = tile_bytes(D, D);     // one state tile
    extern __shared__ uint8_t smem_raw[];
    // 1024-byte alignment by an offset from the __shared__ array (not by integer rounding of a generic pointer), so
    // that the compiler still knows these are shared-memory addresses: LDS/STS with 32-bit address arithmetic
    // instead of generic LD/ST with 64-bit arithmetic.
    uint8_t* sm = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const BLayout Lo(D);
    BMisc& mi = *reinterpret_cast<BMisc*>(sm + Lo.misc);
    const uint32_t sb = smem_u32(sm);
    const int r = RT ? RT : a.r, R2 = 2 * r;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, q = warp & 3, half = warp >> 2;
    const int row = q * 32 + lane;   // tile row == TMEM lane served by this thread
    const bool krole = q < 2;
    const int t = row & 63;          // token of this row
    const uint32_t lane_base = (uint32_t)(q * 32) << 16;
    const int chain = blockIdx.x, b = chain / a.H, h = chain % a.H;
    const int LCc = FULL == 1 ? LC : FULL > 1 ? FULL : (a.L < LC ? a.L : LC);   // (FULL = 16, 32: that chunk length)
    const int nchunks = a.T / LCc, nb = LCc >> 4, gate_every = FULL == 1 ? a.L / LCc : 1;   // (L < 64: one solve chunk per gate chunk)
    const bool warp_active = (q & 1) * 32 < LCc;   // this warp holds at least one live token row
    const bool live = t < LCc;
    const bool srow = row < D;                     // this thread owns a row of the state adjoint
    const int blk = t >> 4;
    const Rec Rc(D, D);
    const uint8_t* rec_chain = a.rec + (size_t)chain * nchunks * Rc.total;

    PROF_INIT();
    // ---- one-time setup --------------------------------------------------------------------------
    if (tid == 0) {
        mbar_init(&mi.bar_mma, 1); mbar_init(&mi.bar_g1, 1); mbar_init(&mi.bar_g3, 1); mbar_init(&mi.bar_sb, 1);
        mbar_init(&mi.bar_g4a, 1); mbar_init(&mi.bar_g4b, 1); mbar_init(&mi.bar_g5, 1); mbar_init(&mi.bar_g8, 1);
        mbar_init(&mi.bar_fi, 1); mbar_init(&mi.bar_bg, 1); mbar_init(&mi.bar_pt, 1);
        mbar_fence_init();
        tma_prefetch_desc(&mdO); tma_prefetch_desc(&mq); tma_prefetch_desc(&mdq); tma_prefetch_desc(&mdk);
        tma_prefetch_desc(&mdv); tma_prefetch_desc(&mdf); tma_prefetch_desc(&mdbx); tma_prefetch_desc(&mdwx);
    }
    if (warp == 0) tmem_alloc(&mi.tmem_base, TM_COLS);
    for (int i = tid; i < 32 * D; i += NTH) {
        const int ii = i / D, n = i % D;
        float vc = 0.f, uc = 0.f;
        if (ii < r) { vc = __ldg(a.Vb + (size_t)n * r + ii); uc = __ldg(a.Ub + (size_t)ii * D + n); }
        else if (ii < R2 && !SW) { vc = __ldg(a.Vw + (size_t)n * r + (ii - r)); uc = __ldg(a.Uw + (size_t)(ii - r) * D + n); }
        *reinterpret_cast<__nv_bfloat16*>(sm + Lo.VcT + tile_off(32, ii, n)) = __float2bfloat16_rn(vc);
        *reinterpret_cast<__nv_bfloat16*>(sm + Lo.Ucat + tile_off(32, ii, n)) = __float2bfloat16_rn(uc);
    }
    for (int i = tid; i < 64 * 64; i += NTH) {
        const int tt_ = i / 64, k = i % 64;
        *reinterpret_cast<uint16_t*>(sm + Lo.TRI + tile_off(64, tt_, k)) = k > tt_ ? 0x3F80u : 0u;
    }
    if (tid < D) {
        const float* et = reinterpret_cast<const float*>(rec_chain + (size_t)(nchunks - 1) * Rc.total + Rc.etot);
        mi.gamLn[tid] = et[tid] * et[D + tid] * et[2 * D + tid] * et[3 * D + tid];
    }
    PHASE_SYNC();
    const uint32_t tmem = mi.tmem_base;
    uint32_t mma_ph = 0;

    // dS (this thread's row x = `row`, columns half*HK..) -> bf16 operand copy DSB, TMEM <- dS gamma_L(next chunk),
    // and dS0 when `last`.  from_tmem: read dS from TMEM, else from dS_final (or zeros).
    auto finalize = [&](bool from_tmem, bool last) {
        if (srow) {
#pragma unroll
            for (int s = 0; s < HK; s += 32) {
                const int c0 = half * HK + s;
                uint32_t v[32];
                if (from_tmem) {
                    tmem_ld32(tmem + BM_DS + lane_base + c0, v);
                    tmem_wait_ld();
                } else {
                    const float* src = a.dS_final ? a.dS_final + ((size_t)chain * D + row) * D + c0 : nullptr;
#pragma unroll
                    for (int e = 0; e < 32; e += 4) {
                        const float4 f4 = src ? __ldg(reinterpret_cast<const float4*>(src + e)) : make_float4(0.f, 0.f, 0.f, 0.f);
                        v[e] = __float_as_uint(f4.x); v[e + 1] = __float_as_uint(f4.y);
                        v[e + 2] = __float_as_uint(f4.z); v[e + 3] = __float_as_uint(f4.w);
                    }
                }
                uint32_t sc[32];
#pragma unroll
                for (int ch = 0; ch < 4; ++ch) {
                    float f8[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        f8[e] = __uint_as_float(v[8 * ch + e]);
                        sc[8 * ch + e] = __float_as_uint(f8[e] * mi.gamLn[c0 + 8 * ch + e]);
                    }
                    sts128(sm + Lo.DSB + tile_chunk_off(D, row, c0 / 8 + ch), pack8(f8));
                    if (last) {
                        float* dst = a.dS0 + ((size_t)chain * D + row) * D + c0 + 8 * ch;
                        *reinterpret_cast<float4*>(dst) = make_float4(f8[0], f8[1], f8[2], f8[3]);
                        *reinterpret_cast<float4*>(dst + 4) = make_float4(f8[4], f8[5], f8[6], f8[7]);
                    }
                }
                tmem_st32(tmem + BM_DS + lane_base + c0, sc);
            }
            tmem_wait_st();
        }
        PHASE_SYNC();
    };

    finalize(false, false);

    // L1 / L3 operands of chunk c2 (thread 0): issued at the top for the first chunk, afterwards as soon as the
    // previous chunk's last readers of the slots are done, so that the fetch hides behind its last phases.
    auto issue_l1 = [&](int c2) {
        const uint8_t* r2 = rec_chain + (size_t)c2 * Rc.total;
        mbar_expect_tx(&mi.bar_g1, 2 * TB + (uint32_t)LCc * D * 2u + 16u * D + 512u + 256u);
        for (int b2 = 0; b2 < 4; ++b2) bulk_g2s(mi.etot[b2], r2 + Rc.etot + b2 * 4 * D, 4u * D, &mi.bar_g1);
        bulk_g2s(mi.rn, r2 + Rc.rn, 512, &mi.bar_g1);
        bulk_g2s(mi.beta, r2 + Rc.beta, 256, &mi.bar_g1);
        bulk_g2s(sm + Lo.S[0], r2 + Rc.KT, TB, &mi.bar_g1);
        bulk_g2s(sm + Lo.S[4], r2 + Rc.U, TB, &mi.bar_g1);
        for (int cb = 0; cb < D / 64; ++cb)
            tma_load_3d(sm + Lo.S[2] + cb * 16384 + 8192, &mdO, &mi.bar_g1, cb * 64, h, b * a.T + c2 * LCc);
    };
    auto issue_g3 = [&](int c2) {
        const uint8_t* r2 = rec_chain + (size_t)c2 * Rc.total;
        mbar_expect_tx(&mi.bar_g3, 2 * TB);
        bulk_g2s(sm + Lo.S[5], r2 + Rc.K0, TB, &mi.bar_g3);
        bulk_g2s(sm + Lo.S[6], r2 + Rc.Q0, TB, &mi.bar_g3);
    };
    // [LCc][D] gradient tile (64-row tile format == the 128-byte-swizzled TMA box) -> global; `cbs` = byte stride
    // between the two 64-column blocks (8192 for a 64-row tile, 16384 for the lower rows of a 128-row tile)
    auto store_tile = [&](const CUtensorMap* m, uint32_t src, uint32_t cbs, int trow_) {
        for (int cb = 0; cb < D / 64; ++cb) tma_store_3d(m, sb + src + cb * cbs, cb * 64, h, trow_);
    };
    auto publish = [&](int done) {   // the bulk stores of the first `done` chunks (in processing order) are complete
        asm volatile("fence.proxy.async.global;" ::: "memory");
        __threadfence();
        asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(a.flags + chain), "r"(done) : "memory");
    };
    auto issue_pt = [&](int c2) {
        mbar_expect_tx(&mi.bar_pt, 16384);
        bulk_g2s(sm + Lo.S[1], rec_chain + (size_t)c2 * Rc.total + Rc.PT, 16384, &mi.bar_pt);
    };
    // The chunk-local epilogue kernel is launched behind this one with programmatic stream serialization: let it start
    // now on the SMs this grid leaves idle; it follows the per-chain progress flags written below.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    bool first = true, first_glue = true;
    PROF(g_prof_bwd, 38);   // one-time setup
    for (int it = 0, c = nchunks - 1; c >= 0; --c, ++it) {
        const uint32_t ph = (uint32_t)it & 1u;
        const uint8_t* rc = rec_chain + (size_t)c * Rc.total;
        const size_t tok0 = (size_t)b * a.T + (size_t)c * LCc;
        const int trow = b * a.T + c * LCc;  // TMA row coordinate of the chunk's first token
        const bool gate_start = (c % gate_every) == 0;   // the fold G of this solve chunk read the state entering it
        // ---- loads of the chunk: L1 operands, state, chunk-anchored rows; small per-chunk vectors
        if (tid == 0) {
            if (it == 0) {   // later chunks: issued as soon as the previous chunk's last reader of SBq is done
                mbar_expect_tx(&mi.bar_sb, SBb);
                bulk_g2s(sm + Lo.SBq, rc + Rc.SB, SBb, &mi.bar_sb);
            }
            if (it == 0) { issue_l1(c); issue_g3(c); issue_pt(c); }
        }
        {
            if (tid >= 128 && tid < 128 + D) {
                const int j = tid - 128;
                float g = 1.f;
                if (c > 0) {
                    const float* en = reinterpret_cast<const float*>(rc - Rc.total + Rc.etot);
                    g = __ldg(en + j) * __ldg(en + D + j) * __ldg(en + 2 * D + j) * __ldg(en + 3 * D + j);
                }
                mi.gamLn[j] = g;   // read by finalize at the end of this chunk
            }
        }
        PROF(g_prof_bwd, 0);
        // L2 and L6 split a token's columns between its two threads: the K-side lane takes the first half of the
        // columns (x or j < D/2), the Q-side lane the second; `cq0` = this thread's first 16-byte piece (QW columns).
        constexpr int QW = D / (2 * NP);
        const int cq0 = ((krole ? 0 : D / 2) + half * QW) / 8;
        // row-private record data of L2 straight from global memory, issued now so that the latency hides behind L1
        uint4 x4[QW / 8], w4[QW / 8];
        if (live && !SW) {
#pragma unroll
            for (int i = 0; i < QW / 8; ++i) {
                const uint32_t off = rp_off(t, cq0 + i);
                x4[i] = ldg128(rc + Rc.VWX + off);
                w4[i] = ldg128(rc + Rc.W + off);
            }
        } else {
#pragma unroll
            for (int i = 0; i < QW / 8; ++i) {   // w == 1, w v (1 - w) == 0
                x4[i] = make_uint4(0u, 0u, 0u, 0u);
                w4[i] = make_uint4(0x3F803F80u, 0x3F803F80u, 0x3F803F80u, 0x3F803F80u);
            }
        }
        // ---- L1: dU = Ktil dS'^T + (scale P)^T dO -> BM_A rows 0..63;  dKtil = U dS' -> BM_KT rows 0..63
        //      (issued by the last warp, a Q-side one: only the K-side warps have work behind this product, and the issuing
        //      lane stays blocked for as long as the 20 instructions take to execute)
        if (warp == NTH / 32 - 1) { if (elect_one()) {
            mbar_wait(&mi.bar_g1, ph);
            mbar_wait(&mi.bar_pt, ph);
            tc_fence_after();
            // dU^T (lanes x, columns s): all 128 lanes carry results (as dU, lanes = tokens, half of the M = 128 rows were junk)
            mma_k<KMAJ, KMAJ, D>(tmem + BM_A, 64, sb + Lo.DSB, D, 0, 0, sb + Lo.S[0], 64, 0, 0, D, false);
            mma_k<MNMAJ, MNMAJ, LC>(tmem + BM_A, 64, sb + Lo.S[2], 128, 0, 64, sb + Lo.S[1], 128, 0, 0, LCc, true);
            mma_k<KMAJ, MNMAJ, D>(tmem + BM_KT, D, sb + Lo.S[4], 64, 0, 0, sb + Lo.DSB, D, 0, 0, D, false);
            umma_commit(&mi.bar_mma);
        LEADER_END
        WAIT_MMA();
        PROF(g_prof_bwd, 13);
        if (srow) {   // dU^T -> bf16 [D][64] tile DUT (S[0], over Ktil): 64 / NP columns per thread
            constexpr int UW = 64 / NP;
            uint32_t v[UW];
            if constexpr (UW == 32) tmem_ld32(tmem + BM_A + lane_base + UW * half, v);
            else tmem_ld16(tmem + BM_A + lane_base + UW * half, v);
            tmem_wait_ld();
#pragma unroll
            for (int ch = 0; ch < UW / 8; ++ch) {
                float f8[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) f8[e] = __uint_as_float(v[8 * ch + e]);
                sts128(sm + Lo.S[0] + tile_chunk_off(D, row, (UW / 8) * half + ch), pack8(f8));
            }
        }
        PROF(g_prof_bwd, 1);
        // ---- L2: dX = T^T dU: columns x < D/2 -> BM_A rows 0..63 (K-side lanes), x >= D/2 -> rows 64..127 (Q-side lanes)
        PROFB_ARRIVE(0); PHASE_SYNC(); PROFB_AFTER(g_profb_bwd, 0);
        PROF(g_prof_bwd, 14);
        LEADER_BEGIN
            mma_k<MNMAJ, KMAJ, LC>(tmem + BM_A + D / 2, D / 2, sb + Lo.S[1], 64, 0, 0, sb + Lo.S[0], D, D / 2, 0, LCc, false);
            mma_k<MNMAJ, KMAJ, LC>(tmem + BM_A, D / 2, sb + Lo.S[1], 64, 64, 0, sb + Lo.S[0], D, 0, 0, LCc, false);
            umma_commit(&mi.bar_mma);
        LEADER_END
        WAIT_MMA();
        PROF(g_prof_bwd, 15);
        if (tid == 0) {  // PT is dead: fetch the block-anchored column operand of L4
            mbar_expect_tx(&mi.bar_g4a, TB);
            bulk_g2s(sm + Lo.S[1], rc + Rc.CC, TB, &mi.bar_g4a);
        }
        if (warp_active) {
            const float bt = live ? mi.beta[t] : 0.f;
            const float rbt = live ? __fdividef(1.f, bt) : 0.f;   // e_t = u_t / beta_t (beta is clamped to >= 1e-30 by the forward)
            float dbs = 0.f;
            uint32_t v[QW];
            if constexpr (QW == 16) tmem_ld16(tmem + BM_A + lane_base + 8 * cq0, v);
            else tmem_ld32(tmem + BM_A + lane_base + 8 * cq0, v);
            tmem_wait_ld();
            if (live) {
#pragma unroll
                for (int i = 0; i < QW / 8; ++i) {
                    const int cc = cq0 + i;
                    float ee[8], xx[8], ww[8], ndr[8], o1[8], o2[8];
                    unpack8(lds128(sm + Lo.S[4] + tile_chunk_off(64, t, cc)), ee);   // u_t (U tile, still the L3 operand)
                    unpack8(x4[i], xx); unpack8(w4[i], ww);
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const float dx = __uint_as_float(v[8 * i + e]);
                        const float dr = bt * dx;
                        dbs += dx * (ee[e] * rbt);
                        ndr[e] = -dr;
                        o1[e] = dr * ww[e];
                        o2[e] = dr * xx[e];
                    }
                    sts128(sm + Lo.S[2] + tile_chunk_off(128, t, cc), pack8(ndr));
                    sts128(sm + Lo.S[0] + tile_chunk_off(64, t, cc), pack8(o1));   // dv, staged over dU
                    sts128(sm + Lo.X + tile_chunk_off(64, t, cc), pack8(o2));      // dw_pre = dwx (zeros when SW)
                }
                mi.dbp[(krole ? 0 : NP) + half][t] = dbs;
            }
        }
        PROF(g_prof_bwd, 2);
        // ---- L3: [dA;dP] raw, SP = [-dR;dO] S, dS += [-dR;dO]^T [Kbar; scale Qbar]
        PROFB_ARRIVE(1); PHASE_SYNC(); PROFB_AFTER(g_profb_bwd, 1);
        PROF(g_prof_bwd, 16);
        LEADER_BEGIN
            mbar_wait(&mi.bar_sb, ph);
            mbar_wait(&mi.bar_g3, ph);
            tc_fence_after();
            mma_k<KMAJ, KMAJ, D>(tmem + BM_DAP, 64, sb + Lo.S[2], 128, 0, 0, sb + Lo.S[4], 64, 0, 0, D, false);
            mma_k<KMAJ, MNMAJ, D>(tmem + BM_A, D, sb + Lo.S[2], 128, 0, 0, sb + Lo.SBq, D, 0, 0, D, false);
            mma_k<MNMAJ, MNMAJ, LC>(tmem + BM_DS, D, sb + Lo.S[2], 128, 0, 0, sb + Lo.S[5], 64, 0, 0, LCc, true);
            mma_k<MNMAJ, MNMAJ, LC>(tmem + BM_DS, D, sb + Lo.S[2], 128, 0, 64, sb + Lo.S[6], 64, 0, 0, LCc, true);
            umma_commit(&mi.bar_mma);
        LEADER_END
        if (tid == STORE_TID) {
            store_tile(&mdv, Lo.S[0], 8192, trow);
            if (!SW) store_tile(&mdwx, Lo.X, 8192, trow);
            bulk_commit();
        }
        if (!krole && half == 0 && live)
        {
            float sdb = 0.f;
#pragma unroll
            for (int pp = 0; pp < NP; ++pp) sdb += mi.dbp[pp][t] + mi.dbp[NP + pp][t];
            a.dbeta[(tok0 + t) * a.H + h] = __float2bfloat16_rn(sdb);
        }
        WAIT_MMA();
        PROF(g_prof_bwd, 17);
        if (tid == 0) {  // DRO and U are dead
            mbar_expect_tx(&mi.bar_g4b, 2 * TB);
            bulk_g2s(sm + Lo.S[2], rc + Rc.KQo, 2 * TB, &mi.bar_g4b);
        }
        {   // masked [dA;dP] -> bf16 tile DAP (S[4], over U)
            constexpr int DW = 64 / NP;   // columns of the 64-wide block handled by this thread
            uint32_t v[DW];
            if constexpr (DW == 32) tmem_ld32(tmem + BM_DAP + lane_base + DW * half, v);
            else tmem_ld16(tmem + BM_DAP + lane_base + DW * half, v);
            tmem_wait_ld();
            // keep s < t (K side) / s <= t (Q side, scaled): branch-free, one compare against a per-thread limit
            const float scl = krole ? 1.f : a.scale;
            const int lim = (live ? (krole ? t : t + 1) : 0) - DW * half;   // keep local column i iff i < lim
#pragma unroll
            for (int ch = 0; ch < DW / 8; ++ch) {
                float f8[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) f8[e] = (8 * ch + e < lim) ? scl * __uint_as_float(v[8 * ch + e]) : 0.f;
                sts128(sm + Lo.S[4] + tile_chunk_off(128, row, (DW / 8) * half + ch), pack8(f8));
            }
        }
        PROF(g_prof_bwd, 3);
        // ---- carry term of d log gamma: gamma_L . colsum(S . dS')  (dS' still sits in DSB as bf16)
        mbar_wait(&mi.bar_sb, ph);
        if (srow) {
            float p[HK];
#pragma unroll
            for (int ch = 0; ch < HK / 8; ++ch) {
                float s8[8], d8[8];
                const uint32_t off = tile_chunk_off(D, row, half * (HK / 8) + ch);
                unpack8(lds128(sm + Lo.SBq + off), s8);
                unpack8(lds128(sm + Lo.DSB + off), d8);
#pragma unroll
                for (int e = 0; e < 8; ++e) p[8 * ch + e] = s8[e] * d8[e];
            }
            warp_colsum<HK>(p, lane);
#pragma unroll
            for (int i = 0; i < HK / 32; ++i) mi.colp[q][half * HK + (HK / 32) * lane + i] = p[i];
        }
        PROF(g_prof_bwd, 4);
        // ---- L4: pairwise decay terms on mma.sync.  Warp w owns key channels [NCW w, NCW (w+1)) for all tokens, so the
        //      three pieces of d log gamma that cancel pairwise meet in one thread, in fp32:
        //        (i)  H_t  = sum_{s} [dA;dP]_ts C_s G(blk t, blk s)      (rows of both sides)
        //        (ii) H'_s = sum_{t} [dA;dP]_ts [Kbar;Qbar]own_t G(blk t, blk s)
        //      with G = product of the whole-block decays between the two blocks, applied by Horner steps.  Every pair
        //      (t,s) enters +Kbar_own_t C_s dA_ts G in row t and -C_s Kbar_own_t dA_ts G in row s with bit-identical
        //      operands, so the pairs that do not straddle a token cancel to fp32 rounding in the reverse cumulative sum.
        PROFB_ARRIVE(2); __syncthreads(); PROFB_AFTER(g_profb_bwd, 2);
        PROF(g_prof_bwd, 18);
        if (tid == 0) {   // dS' (DSB) is consumed: stage gamma_t/gamma_a and its inverse there for L5
            mbar_expect_tx(&mi.bar_fi, 2 * TB);
            bulk_g2s(sm + Lo.FI, rc + Rc.FQ, TB, &mi.bar_fi);
            bulk_g2s(sm + Lo.FI + TB, rc + Rc.IC, TB, &mi.bar_fi);
            // the erase gate b follows into the same buffer at L6: have it in L2 by then
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(rc + Rc.Bg), "r"(TB) : "memory");
        }
        if (tid < D) {
            float sx = 0.f;
#pragma unroll
            for (int qq = 0; qq < D / 32; ++qq) sx += mi.colp[qq][tid];
            const float e0 = mi.etot[0][tid], e1 = mi.etot[1][tid], e2 = mi.etot[2][tid], e3 = mi.etot[3][tid];
            mi.extra[tid] = sx * (e0 * e1 * e2 * e3);
            mi.pre[0][tid] = 1.f; mi.pre[1][tid] = e0; mi.pre[2][tid] = e0 * e1; mi.pre[3][tid] = e0 * e1 * e2;
            mi.suf[3][tid] = e3; mi.suf[2][tid] = e2 * e3; mi.suf[1][tid] = e1 * e2 * e3; mi.suf[0][tid] = e0 * e1 * e2 * e3;
        }
        {
            constexpr int NCW = D / (4 * NP), NTW = NCW / 8;   // key channels per warp, n-tiles
            const int g = lane >> 2, l4 = lane & 3, cw = NCW * warp;
            const int lrow = (lane & 7) + ((lane >> 3) & 1) * 8;
            const int lchk = NTW == 2 ? (lane >> 4) : 0;
            float et[4][NTW][2];
#pragma unroll
            for (int b2 = 0; b2 < 4; ++b2)
#pragma unroll
                for (int nt = 0; nt < NTW; ++nt) {
                    const float2 e2 = *reinterpret_cast<const float2*>(&mi.etot[b2][cw + 8 * nt + 2 * l4]);
                    et[b2][nt][0] = e2.x; et[b2][nt][1] = e2.y;
                }
            mbar_wait(&mi.bar_g4a, ph);
            PROF(g_prof_bwd, 19);
            uint32_t bC[4][NTW][2];
#pragma unroll
            for (int jb = 0; jb < 4; ++jb) {
                if (jb < nb) {
                    uint32_t tmp[4];
                    ldsm_x4_t(tmp, sb + Lo.S[1] + tile_chunk_off(64, 16 * jb + lrow, cw / 8 + lchk));
#pragma unroll
                    for (int nt = 0; nt < NTW; ++nt) { bC[jb][nt][0] = tmp[2 * nt]; bC[jb][nt][1] = tmp[2 * nt + 1]; }
                }
            }
            float accI[8][NTW][4];
#pragma unroll
            for (int mt = 0; mt < 8; ++mt)
#pragma unroll
                for (int nt = 0; nt < NTW; ++nt)
#pragma unroll
                    for (int e = 0; e < 4; ++e) accI[mt][nt][e] = 0.f;
#pragma unroll
            for (int side = 0; side < 2; ++side)
#pragma unroll
                for (int ib = 0; ib < 4; ++ib) {
                    if (ib < nb) {
                        const int mt = side * 4 + ib, r0 = side * 64 + 16 * ib;
#pragma unroll
                        for (int jb = 0; jb < 4; ++jb) {
                            if (jb <= ib) {
                                uint32_t af[4];   // A[m = t][k = s] = DAP[t][s]: matrix m: rows r0 + 8 (m&1), chunk 2 jb + (m>>1)
                                ldsm_x4(af, sb + Lo.S[4] + tile_chunk_off(128, r0 + lrow, 2 * jb + (lane >> 4)));
#pragma unroll
                                for (int nt = 0; nt < NTW; ++nt) {
                                    mma_bf16(accI[mt][nt], af, bC[jb][nt][0], bC[jb][nt][1]);
                                    if (jb < ib) {   // step over block jb: gamma_e(jb)/gamma_a(jb)
                                        accI[mt][nt][0] *= et[jb][nt][0]; accI[mt][nt][1] *= et[jb][nt][1];
                                        accI[mt][nt][2] *= et[jb][nt][0]; accI[mt][nt][3] *= et[jb][nt][1];
                                    }
                                }
                            }
                        }
                    }
                }
            mbar_wait(&mi.bar_g4b, ph);
            PROF(g_prof_bwd, 20);
            float accII[4][NTW][4];
#pragma unroll
            for (int jb = 0; jb < 4; ++jb)
#pragma unroll
                for (int nt = 0; nt < NTW; ++nt)
#pragma unroll
                    for (int e = 0; e < 4; ++e) accII[jb][nt][e] = 0.f;
#pragma unroll
            for (int ib = 3; ib >= 0; --ib) {
                if (ib < nb) {
                    uint32_t bK[2][NTW][2];
#pragma unroll
                    for (int side = 0; side < 2; ++side) {
                        uint32_t tmp[4];
                        ldsm_x4_t(tmp, sb + Lo.S[2] + tile_chunk_off(128, side * 64 + 16 * ib + lrow, cw / 8 + lchk));
#pragma unroll
                        for (int nt = 0; nt < NTW; ++nt) { bK[side][nt][0] = tmp[2 * nt]; bK[side][nt][1] = tmp[2 * nt + 1]; }
                    }
#pragma unroll
                    for (int jb = 0; jb < 4; ++jb) {
                        if (jb <= ib) {
                            if (ib < nb - 1) {
#pragma unroll
                                for (int nt = 0; nt < NTW; ++nt) {
                                    accII[jb][nt][0] *= et[ib][nt][0]; accII[jb][nt][1] *= et[ib][nt][1];
                                    accII[jb][nt][2] *= et[ib][nt][0]; accII[jb][nt][3] *= et[ib][nt][1];
                                }
                            }
#pragma unroll
                            for (int side = 0; side < 2; ++side) {
                                uint32_t af[4];
                                // A[m = s][k = t] = DAP[t][s]: transposed 8x8 loads; matrix m: rows t0 + 8 (m>>1), chunk 2 jb + (m&1)
                                ldsm_x4_t(af, sb + Lo.S[4] + tile_chunk_off(128, side * 64 + 16 * ib + (lane & 7) + (lane >> 4) * 8,
                                                                            2 * jb + ((lane >> 3) & 1)));
#pragma unroll
                                for (int nt = 0; nt < NTW; ++nt) mma_bf16(accII[jb][nt], af, bK[side][nt][0], bK[side][nt][1]);
                            }
                        }
                    }
                }
            }
            // contributions to d log gamma_t from the pairs: +Kbar_own_t H_t (to t-1), +Qbar_own_t H_t, -C_t H'_t
            float dd[8][NTW][2], aa[8][NTW][2];
#pragma unroll
            for (int b2 = 0; b2 < 4; ++b2)
#pragma unroll
                for (int hh = 0; hh < 2; ++hh) {
                    const int grp = 2 * b2 + hh, tt2 = 16 * b2 + 8 * hh + g;
#pragma unroll
                    for (int nt = 0; nt < NTW; ++nt) {
                        dd[grp][nt][0] = dd[grp][nt][1] = aa[grp][nt][0] = aa[grp][nt][1] = 0.f;
                        if (b2 < nb) {
                            const int j = cw + 8 * nt + 2 * l4;
                            const uint32_t wk = *reinterpret_cast<const uint32_t*>(sm + Lo.S[2] + tile_off(128, tt2, j));
                            const uint32_t wq = *reinterpret_cast<const uint32_t*>(sm + Lo.S[2] + tile_off(128, 64 + tt2, j));
                            const uint32_t wc = *reinterpret_cast<const uint32_t*>(sm + Lo.S[1] + tile_off(64, tt2, j));
                            const float xa0 = bf16_lo(wk) * accI[b2][nt][2 * hh], xa1 = bf16_hi(wk) * accI[b2][nt][2 * hh + 1];
                            const float xq0 = bf16_lo(wq) * accI[4 + b2][nt][2 * hh], xq1 = bf16_hi(wq) * accI[4 + b2][nt][2 * hh + 1];
                            const float xc0 = bf16_lo(wc) * accII[b2][nt][2 * hh], xc1 = bf16_hi(wc) * accII[b2][nt][2 * hh + 1];
                            dd[grp][nt][0] = (xq0 - xc0) + xa0; dd[grp][nt][1] = (xq1 - xc1) + xa1;
                            aa[grp][nt][0] = xa0; aa[grp][nt][1] = xa1;
                        }
                    }
                }
            // reverse cumulative sum over tokens (token = 8 grp + g): dlp_t = sum_{t' >= t} dd_t' - aa_t
#pragma unroll
            for (int nt = 0; nt < NTW; ++nt)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    float carry = 0.f;
#pragma unroll
                    for (int grp = 7; grp >= 0; --grp) {
                        float v = dd[grp][nt][e];
#pragma unroll
                        for (int off = 1; off < 8; off <<= 1) {
                            const float o = __shfl_down_sync(0xFFFFFFFFu, v, 4 * off);
                            if (g + off < 8) v += o;
                        }
                        const float tot = __shfl_sync(0xFFFFFFFFu, v, l4);
                        dd[grp][nt][e] = v + carry - aa[grp][nt][e];
                        carry += tot;
                    }
                }
            if (tid == STORE_TID) {
                bulk_wait_read();   // dv has left S[0] (dlp goes there below)
                if (it > 0) {       // all but the newest group (dv | dwx of this chunk): the previous chunk's stores are complete
                    bulk_wait_all_but<1>();
                    publish(it);
                }
            }
            PROFB_ARRIVE(3); __syncthreads(); PROFB_AFTER(g_profb_bwd, 3);  // every warp is done reading DAP / C / KQo
            PROF(g_prof_bwd, 21);
#pragma unroll
            for (int side = 0; side < 2; ++side)       // H raw -> S[2..3] ([128][D] tile, over KQo): for dk^, dq^
#pragma unroll
                for (int ib = 0; ib < 4; ++ib) {
                    if (ib < nb) {
                        const int mt = side * 4 + ib, r0 = side * 64 + 16 * ib;
#pragma unroll
                        for (int nt = 0; nt < NTW; ++nt) {
                            const int j = cw + 8 * nt + 2 * l4;
                            *reinterpret_cast<uint32_t*>(sm + Lo.S[2] + tile_off(128, r0 + g, j)) = pack_bf16(accI[mt][nt][0], accI[mt][nt][1]);
                            *reinterpret_cast<uint32_t*>(sm + Lo.S[2] + tile_off(128, r0 + g + 8, j)) = pack_bf16(accI[mt][nt][2], accI[mt][nt][3]);
                        }
                    }
                }
#pragma unroll
            for (int jb = 0; jb < 4; ++jb) {           // H' raw -> S[4] ([64][D] tile, over DAP);  dlp -> S[0]
                if (jb < nb) {
#pragma unroll
                    for (int nt = 0; nt < NTW; ++nt) {
                        const int j = cw + 8 * nt + 2 * l4;
                        *reinterpret_cast<uint32_t*>(sm + Lo.S[4] + tile_off(64, 16 * jb + g, j)) = pack_bf16(accII[jb][nt][0], accII[jb][nt][1]);
                        *reinterpret_cast<uint32_t*>(sm + Lo.S[4] + tile_off(64, 16 * jb + g + 8, j)) = pack_bf16(accII[jb][nt][2], accII[jb][nt][3]);
                        *reinterpret_cast<uint32_t*>(sm + Lo.S[0] + tile_off(64, 16 * jb + g, j)) = pack_bf16(dd[2 * jb][nt][0], dd[2 * jb][nt][1]);
                        *reinterpret_cast<uint32_t*>(sm + Lo.S[0] + tile_off(64, 16 * jb + g + 8, j)) = pack_bf16(dd[2 * jb + 1][nt][0], dd[2 * jb + 1][nt][1]);
                    }
                }
            }
        }
        PROF(g_prof_bwd, 5);
        // ---- L5: assemble dk^, dq^ (state part) and the state-read / state-write contributions to d log gamma
        PROFB_ARRIVE(4); __syncthreads(); PROFB_AFTER(g_profb_bwd, 4);
        mbar_wait(&mi.bar_fi, ph);
        PROF(g_prof_bwd, 22);
        if (warp_active) {
            if (krole) {
                const bool bstart = (t & 15) == 0;
                const uint4 ones4 = make_uint4(0x3F803F80u, 0x3F803F80u, 0x3F803F80u, 0x3F803F80u);
#pragma unroll
                for (int s = 0; s < HK; s += 16) {
                    uint32_t vs[16], vk[16];
                    tmem_ld16(tmem + BM_A + lane_base + half * HK + s, vs);    // SP_K = (-dR) S
                    tmem_ld16(tmem + BM_KT + lane_base + half * HK + s, vk);   // dKtil = U dS'
                    tmem_wait_ld();
                    if (live) {
#pragma unroll
                        for (int ch = 0; ch < 2; ++ch) {
                            const int i = s / 8 + ch, cc = half * (HK / 8) + i, j0 = 8 * cc;
                            float2 fp[4], ic[4], pk[4], pc[4], k0[4], c8[4], o[4], xa[4], zz[4];
                            unpack8p(bstart ? ones4 : lds128(sm + Lo.FI + rp_off(t - 1, cc)), fp);
                            unpack8p(lds128(sm + Lo.FI + TB + rp_off(t, cc)), ic);
                            unpack8p(lds128(sm + Lo.S[2] + tile_chunk_off(128, t, cc)), pk);
                            unpack8p(lds128(sm + Lo.S[4] + tile_chunk_off(64, t, cc)), pc);
                            unpack8p(lds128(sm + Lo.S[5] + tile_chunk_off(64, t, cc)), k0);
                            unpack8p(lds128(sm + Lo.S[1] + tile_chunk_off(64, t, cc)), c8);
                            float2 pre[4], suf[4];   // gamma_a(blk)/gamma_{-1} and gamma_L/gamma_a(blk)
                            *reinterpret_cast<float4*>(pre) = *reinterpret_cast<const float4*>(&mi.pre[blk][j0]);
                            *reinterpret_cast<float4*>(pre + 2) = *reinterpret_cast<const float4*>(&mi.pre[blk][j0 + 4]);
                            *reinterpret_cast<float4*>(suf) = *reinterpret_cast<const float4*>(&mi.suf[blk][j0]);
                            *reinterpret_cast<float4*>(suf + 2) = *reinterpret_cast<const float4*>(&mi.suf[blk][j0 + 4]);
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                const float2 sp = pair_of(vs + 8 * ch + 2 * e), dkt = pair_of(vk + 8 * ch + 2 * e);
                                const float2 dkA = mul2(fp[e], fma2(pre[e], sp, pk[e]));
                                const float2 dkC = mul2(ic[e], fma2(suf[e], dkt, pc[e]));
                                o[e] = add2(dkA, dkC);
                                xa[e] = mul2(k0[e], sp);                      // Kbar_t . dKbar_t (state read), to d log gamma_{t-1}
                                zz[e] = mul2(mul2(c8[e], suf[e]), dkt);       // Ktil_t . dKtil_t (state write), to d log gamma_t' for t' > t
                            }
                            sts128(sm + Lo.S[5] + tile_chunk_off(64, t, cc), pack8p(o));    // dk^, staged in place over Kbar_t
                            sts128(sm + Lo.S[2] + tile_chunk_off(128, t, cc), pack8p(xa));   // in place over H_t
                            sts128(sm + Lo.S[4] + tile_chunk_off(64, t, cc), pack8p(zz));    // in place over H'_t
                        }
                    }
                }
            } else {
#pragma unroll
                for (int s = 0; s < HK; s += 16) {
                    uint32_t vs[16];
                    tmem_ld16(tmem + BM_A + lane_base + half * HK + s, vs);    // SP_Q = dO S
                    tmem_wait_ld();
                    if (live) {
#pragma unroll
                        for (int ch = 0; ch < 2; ++ch) {
                            const int i = s / 8 + ch, cc = half * (HK / 8) + i, j0 = 8 * cc;
                            float2 fq[4], pq[4], q0[4], xq[4], pre[4];
                            unpack8p(lds128(sm + Lo.FI + rp_off(t, cc)), fq);
                            unpack8p(lds128(sm + Lo.S[2] + tile_chunk_off(128, 64 + t, cc)), pq);
                            unpack8p(lds128(sm + Lo.S[6] + tile_chunk_off(64, t, cc)), q0);
                            *reinterpret_cast<float4*>(pre) = *reinterpret_cast<const float4*>(&mi.pre[blk][j0]);
                            *reinterpret_cast<float4*>(pre + 2) = *reinterpret_cast<const float4*>(&mi.pre[blk][j0 + 4]);
                            const float2 sc2 = splat2(a.scale);
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                const float2 sp = pair_of(vs + 8 * ch + 2 * e);
                                const float2 dqv = mul2(fq[e], fma2(mul2(pre[e], sc2), sp, pq[e]));
                                vs[8 * ch + 2 * e] = __float_as_uint(dqv.x); vs[8 * ch + 2 * e + 1] = __float_as_uint(dqv.y);
                                xq[e] = mul2(q0[e], sp);            // scale Qbar_t . (dO S)_t (state read)
                            }
                            sts128(sm + Lo.S[2] + tile_chunk_off(128, 64 + t, cc), pack8p(xq));   // in place over H_t
                        }
                    }
                    tmem_st16(tmem + BM_A + lane_base + half * HK + s, vs);   // dq^ state part, completed by the L8 MMA
                }
                tmem_wait_st();
            }
        }
        PROF(g_prof_bwd, 6);
        // ---- L6: d log a_t = dlp_t + carry + sum_{t' > t} XA_t' + sum_{t' >= t} XQ_t' + sum_{t' < t} Z_t' -> BM_KT:
        //      key channels j < D/2 in rows 0..63 (K-side lanes), j >= D/2 in rows 64..127 (Q-side lanes: the 0/1 tile
        //      used as the upper half of the M = 128 operand), so both threads of a token share the epilogue
        PROFB_ARRIVE(5); PHASE_SYNC(); PROFB_AFTER(g_profb_bwd, 5);
        PROF(g_prof_bwd, 23);
        LEADER_BEGIN
            // one 0/1 tile: t' > t as stored (K-major), t' < t as its MN-major view; XQ enters with t' >= t: its diagonal
            // is added in the epilogue below.  `trh`: the tile as the upper half of the M = 128 operand.
            const uint32_t tri = sb + Lo.TRI, trh = tri - 8192;
            mma_k<KMAJ, MNMAJ, LC>(tmem + BM_KT, D / 2, tri, 64, 0, 0, sb + Lo.S[2], 128, 0, 0, LCc, false);
            mma_k<KMAJ, MNMAJ, LC>(tmem + BM_KT, D / 2, tri, 64, 0, 0, sb + Lo.S[2], 128, 0, 64, LCc, true);
            mma_k<MNMAJ, MNMAJ, LC>(tmem + BM_KT, D / 2, tri, 64, 0, 0, sb + Lo.S[4], 64, 0, 0, LCc, true);
            mma_k<KMAJ, MNMAJ, LC>(tmem + BM_KT + D / 2, D / 2, trh, 64, 0, 0, sb + Lo.S[2], 128, D / 2, 0, LCc, false);
            mma_k<KMAJ, MNMAJ, LC>(tmem + BM_KT + D / 2, D / 2, trh, 64, 0, 0, sb + Lo.S[2], 128, D / 2, 64, LCc, true);
            mma_k<MNMAJ, MNMAJ, LC>(tmem + BM_KT + D / 2, D / 2, trh, 64, 0, 0, sb + Lo.S[4], 64, D / 2, 0, LCc, true);
            umma_commit(&mi.bar_mma);
            // gamma_a/gamma_t (second half of FI) and Q0 are dead: fetch G^T of the chunk and the raw q rows for L8
            mbar_expect_tx(&mi.bar_g8, tile_bytes(D, 64));
            bulk_g2s(sm + Lo.FI + TB, rc + Rc.GT, tile_bytes(D, 64), &mi.bar_g8);
            mbar_expect_tx(&mi.bar_g5, (uint32_t)LCc * D * 2u);
            for (int cb = 0; cb < D / 64; ++cb) tma_load_3d(sm + Lo.S[6] + cb * 8192, &mq, &mi.bar_g5, cb * 64, h, trow);
        LEADER_END
        if (tid == STORE_TID) { store_tile(&mdk, Lo.S[5], 8192, trow); bulk_commit(); }
        {
            // the erase gate b of this thread's columns (row-private, L2-prefetched in L4) and, Q-side threads,
            // [tt_b|0 ; 0|tt_w] -> S[1]: global loads issued before the wait
            uint4 b4[QW / 8], t4[4];
            if (live) {
#pragma unroll
                for (int i = 0; i < QW / 8; ++i) b4[i] = ldg128(rc + Rc.Bg + rp_off(t, cq0 + i));
            }
            if (!krole && live) {
#pragma unroll
                for (int i = 0; i < 4; ++i)   // packed chunk i of [tt_b | tt_w] -> chunk of the forward's tile (each half padded to 16 columns)
                    t4[i] = ldg128(rc + Rc.tt + tile_chunk_off(128, t, i < (r >> 3) ? i : 2 + i - (r >> 3)));
            }
            WAIT_MMA();
            PROF(g_prof_bwd, 24);
            if (!krole && live) {
                // TT2: row t = [tt_b | 0], row 64+t = [0 | tt_w] over 32 columns; part 0 writes the K-side row
                const uint4 z4 = make_uint4(0u, 0u, 0u, 0u);
                const int rc8 = r >> 3;  // 16-byte chunks per gate half
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const bool is_b = i < rc8, is_w = i >= rc8 && i < 2 * rc8;
                    if (half == 0) sts128(sm + Lo.S[1] + tile_chunk_off(128, t, i), is_b ? t4[i] : z4);
                    else if (half == 1) sts128(sm + Lo.S[1] + tile_chunk_off(128, 64 + t, i), is_w ? t4[i] : z4);
                }
            }
            PROF(g_prof_bwd, 25);
            if (warp_active) {
                uint32_t v[QW];
                if constexpr (QW == 16) tmem_ld16(tmem + BM_KT + lane_base + 8 * cq0, v);
                else tmem_ld32(tmem + BM_KT + lane_base + 8 * cq0, v);
                tmem_wait_ld();
                if (live) {
#pragma unroll
                    for (int i = 0; i < QW / 8; ++i) {
                        const int cc = cq0 + i;
                        float bb[8], dp[8], xq[8], dla[8], dbp[8];
                        unpack8(b4[i], bb);
                        unpack8(lds128(sm + Lo.S[0] + tile_chunk_off(64, t, cc)), dp);
                        unpack8(lds128(sm + Lo.S[2] + tile_chunk_off(128, 64 + t, cc)), xq);   // the t' = t term of XQ
#pragma unroll
                        for (int e = 0; e < 8; ++e) {
                            dla[e] = (__uint_as_float(v[8 * i + e]) + xq[e]) + dp[e] + mi.extra[8 * cc + e];
                            dbp[e] = -dla[e] * bb[e];
                        }
                        // d log a (the epilogue kernel turns it into df), staged in place over dlp; db_pre = dbx is both the
                        // staged gradient tile and rows 0..63 of the L7 operand GW
                        sts128(sm + Lo.S[0] + tile_chunk_off(64, t, cc), pack8(dla));
                        sts128(sm + Lo.S[2] + tile_chunk_off(128, t, cc), pack8(dbp));
                    }
                }
            }
        }
        PROF(g_prof_bwd, 7);
        // ---- L7: ZZ_b = db_pre Vb -> BM_DAP rows 0..63, ZZ_w = dw_pre Vw -> BM_DAP + 16 rows 64..127 (dw_pre: the tile X
        //      as the upper half of the operand);  dVb | dVw += [db_pre; dw_pre]^T TT2 -> BM_WG
        PROFB_ARRIVE(6); PHASE_SYNC(); PROFB_AFTER(g_profb_bwd, 6);
        PROF(g_prof_bwd, 26);
        LEADER_BEGIN
            mma_k<KMAJ, KMAJ, D>(tmem + BM_DAP, 16, sb + Lo.S[2], 128, 0, 0, sb + Lo.VcT, 32, 0, 0, D, false);
            mma_k<KMAJ, KMAJ, D>(tmem + BM_DAP + 16, 16, sb + Lo.X - 8192, 64, 0, 0, sb + Lo.VcT, 32, r, 0, D, false);
            mma_k<MNMAJ, MNMAJ, LC>(tmem + BM_WG, 32, sb + Lo.S[2], 128, 0, 0, sb + Lo.S[1], 128, 0, 0, LCc, !first);
            mma_k<MNMAJ, MNMAJ, LC>(tmem + BM_WG, 32, sb + Lo.X, 64, 0, 0, sb + Lo.S[1], 128, 0, 64, LCc, true);
            umma_commit(&mi.bar_mma);
        LEADER_END
        if (tid == STORE_TID) {
            store_tile(&mdf, Lo.S[0], 8192, trow);
            store_tile(&mdbx, Lo.S[2], 16384, trow);
            bulk_commit();
        }
        if (c > 0 && live) {   // next chunk's row-private L2 inputs -> L2 cache, so that the loads at its top are short
            const uint8_t* rn_ = rc - Rc.total;
#pragma unroll
            for (int i = 0; i < QW / 8; ++i) {
                asm volatile("prefetch.global.L2 [%0];" ::"l"(rn_ + Rc.VWX + rp_off(t, cq0 + i)));
                asm volatile("prefetch.global.L2 [%0];" ::"l"(rn_ + Rc.W + rp_off(t, cq0 + i)));
            }
            if (!krole && half < 2) asm volatile("prefetch.global.L2 [%0];" ::"l"(rn_ + Rc.tt + tile_chunk_off(128, t, 0)));
        }
        WAIT_MMA();
        PROF(g_prof_bwd, 27);
        if (warp_active) {
            // dz = ZZ (1 - tt^2): K side owns the erase half (cols 0..r), Q side the write half (cols r..2r); column part
            // `half` takes the 8 columns [8 half, 8 half + 8) of its side
            const int c0 = krole ? 0 : r;
            if (half < (r >> 3)) {
                uint32_t v[8];
                tmem_ld8(tmem + BM_DAP + lane_base + (krole ? 0 : 16) + 8 * half, v);
                tmem_wait_ld();
                if (live) {
                    const float rnq = a.l2norm ? mi.rn[64 + t] : 1.f;
                    float tv[8], dz[8], dzq[8];
                    unpack8(lds128(sm + Lo.S[1] + tile_chunk_off(128, krole ? t : 64 + t, c0 / 8 + half)), tv);
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        dz[e] = __uint_as_float(v[e]) * (1.f - tv[e] * tv[e]);
                        dzq[e] = dz[e] * rnq;
                    }
                    sts128(sm + Lo.X + tile_chunk_off(64, t, c0 / 8 + half), pack8(dz));      // DZ (over dw_pre)
                    sts128(sm + Lo.S[4] + tile_chunk_off(64, t, c0 / 8 + half), pack8(dzq));   // DZQ = dz / |q|
                }
            }
            if (!krole && live) {  // zero the unused columns [2r, 32) of DZQ (the dG product has N = 32)
                const uint4 z4 = make_uint4(0u, 0u, 0u, 0u);
                for (int i = 2 * (r >> 3) + half; i < 4; i += NP) sts128(sm + Lo.S[4] + tile_chunk_off(64, t, i), z4);
            }
        }
        PROF(g_prof_bwd, 8);
        // ---- L8: dq^ += dz G -> BM_A rows 64..127;  dG^T = q^T (dz/|q|) -> BM_DAP + 32
        PROFB_ARRIVE(7); PHASE_SYNC(); PROFB_AFTER(g_profb_bwd, 7);
        PROF(g_prof_bwd, 28);
        LEADER_BEGIN
            mbar_wait(&mi.bar_g8, ph);
            mbar_wait(&mi.bar_g5, ph);
            tc_fence_after();
            // DZ: the tile X as the upper half of the operand; G^T: columns 32.. of the forward's Vcat tile
            mma_k<KMAJ, KMAJ, 32>(tmem + BM_A, D, sb + Lo.X - 8192, 128, 0, 0, sb + Lo.FI + TB, D, 0, 32, R2, true);
            mma_k<MNMAJ, MNMAJ, LC>(tmem + BM_DAP + 32, 32, sb + Lo.S[6], 64, 0, 0, sb + Lo.S[4], 64, 0, 0, LCc, false);
            umma_commit(&mi.bar_mma);
        LEADER_END
        WAIT_MMA();
        PROF(g_prof_bwd, 29);
        if (tid == STORE_TID && c > 0) {   // DZQ, GW, the L1 slots are dead; d log a and dbx have left S[0] / S[2]
            bulk_wait_read();
            issue_l1(c - 1);
        }
        if (!krole && warp_active) {
#pragma unroll
            for (int s = 0; s < HK; s += 32) {
                uint32_t v[32];
                tmem_ld32(tmem + BM_A + lane_base + half * HK + s, v);
                tmem_wait_ld();
                if (live) {
#pragma unroll
                    for (int ch = 0; ch < 4; ++ch) {
                        float f8[8];
#pragma unroll
                        for (int e = 0; e < 8; ++e) f8[e] = __uint_as_float(v[8 * ch + e]);
                        sts128(sm + Lo.S[6] + tile_chunk_off(64, t, (half * HK + s) / 8 + ch), pack8(f8));   // dq^, staged over the raw q
                    }
                }
            }
        }
        if (half == 1 && srow) {   // dG^T rows j -> bf16 tile DGT (S[1], over TT2)
            uint32_t v[32];
            tmem_ld32(tmem + BM_DAP + 32 + lane_base, v);
            tmem_wait_ld();
            if (gate_every > 1) {   // L = 128: both solve chunks of a gate chunk share G; their dG add up (same thread, same row)
                float4* st = reinterpret_cast<float4*>(a.dgs + ((size_t)chain * D + row) * 32);
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    if (!gate_start) {
                        st[e] = make_float4(__uint_as_float(v[4 * e]), __uint_as_float(v[4 * e + 1]), __uint_as_float(v[4 * e + 2]),
                                            __uint_as_float(v[4 * e + 3]));
                    } else {
                        const float4 o = st[e];
                        v[4 * e] = __float_as_uint(__uint_as_float(v[4 * e]) + o.x);
                        v[4 * e + 1] = __float_as_uint(__uint_as_float(v[4 * e + 1]) + o.y);
                        v[4 * e + 2] = __float_as_uint(__uint_as_float(v[4 * e + 2]) + o.z);
                        v[4 * e + 3] = __float_as_uint(__uint_as_float(v[4 * e + 3]) + o.w);
                    }
                }
            }
            if (gate_start) {   // (otherwise S[1] is already being refilled for the next chunk)
#pragma unroll
                for (int ch = 0; ch < 4; ++ch) {
                    float f8[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) f8[e] = __uint_as_float(v[8 * ch + e]);
                    sts128(sm + Lo.S[1] + tile_chunk_off(D, row, ch), pack8(f8));
                }
            }
        }
        PROF(g_prof_bwd, 9);
        // ---- L9: fold glue: dS += [Ub;Uw]^T dG;  d[Ub;Uw]^T += S dG^T -> BM_WU
        if (gate_start) {
            PROFB_ARRIVE(8); PHASE_SYNC(); PROFB_AFTER(g_profb_bwd, 8);
            PROF(g_prof_bwd, 30);
            LEADER_BEGIN
                mma_k<MNMAJ, KMAJ, 32>(tmem + BM_DS, D, sb + Lo.Ucat, 32, 0, 0, sb + Lo.S[1], D, 0, 0, R2, true);
                mma_k<KMAJ, MNMAJ, D>(tmem + BM_WU, 32, sb + Lo.SBq, D, 0, 0, sb + Lo.S[1], D, 0, 0, D, !first_glue);
                umma_commit(&mi.bar_mma);
            LEADER_END
            WAIT_MMA();
            PROF(g_prof_bwd, 31);
            first_glue = false;
        }
        if (tid == 0 && c > 0) {   // SBq and the dG tile are free: the state entering the next chunk, its [P;T]
            mbar_expect_tx(&mi.bar_sb, SBb);
            bulk_g2s(sm + Lo.SBq, rc - Rc.total + Rc.SB, SBb, &mi.bar_sb);
            issue_pt(c - 1);
        }
        PROF(g_prof_bwd, 10);
        // ---- L10: the adjoint of the state entering the chunk
        PROF(g_prof_bwd, 11);
        finalize(true, c == 0);
        if (tid == STORE_TID) {   // (behind the barrier inside finalize)
            store_tile(&mdq, Lo.S[6], 8192, trow);
            bulk_commit();
            if (c > 0) {   // dk^ has left S[5] long ago, dq^ leaves S[6] now: the next chunk's chunk-anchored rows go there
                bulk_wait_read();
                issue_g3(c - 1);
            }
        }
        PROF(g_prof_bwd, 12);
        first = false;
    }

    // ---- per-chain partial weight gradients: [dUb|dUw][dVb][dVw] (dA, dtau come from the epilogue kernel)
    if (half == 0 && srow) {
        float* part = a.part + (size_t)chain * a.part_stride;
        float* partVb = part + 2 * r * D;
        float* partVw = partVb + D * r;
        uint32_t wg[32], wu[32];
        tmem_ld32(tmem + BM_WG + lane_base, wg);
        tmem_ld32(tmem + BM_WU + lane_base, wu);
        tmem_wait_ld();
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            if (i < r) partVb[row * r + i] = __uint_as_float(wg[i]);
            else if (i < R2) partVw[row * r + (i - r)] = __uint_as_float(wg[i]);
            if (i < R2) part[i * D + row] = __uint_as_float(wu[i]);
        }
    }
    if (tid == STORE_TID) bulk_wait_all();
    PHASE_SYNC();
    // last publish: chunk 0 AND the partials above are in memory (the reductions run behind the epilogue grid)
    if (tid == STORE_TID) publish(nchunks);
    PROF(g_prof_bwd, 39);   // per-chain partials, last publish
    PROF_FLUSH(g_prof_bwd)
    if (warp == 0) tmem_dealloc(tmem, TM_COLS);
}

// ---- chunk-local tail, fully parallel over (chain, chunk) -----------------------------------------
// dq, dk hold the gradients w.r.t. the normalised q^, k^ and df holds d log a; in place:
//   dq = (dq^ - q^ <q^, dq^>) / sqrt(|q|^2 + eps)   (L2-norm backward, Alg. 5 step 14 l.857-860), same for k
//   df = dla . (-exp A) sigmoid(f + tau)            (Eq. 9 l.151), and the per-chunk partial sums of
//   dtau = sum df,  dA = sum dla . g  with g = -exp(A) softplus(f + tau).
template <int D>
__global__ void __launch_bounds__(256, 4)
carve_bwd_tc_epilogue_kernel(const __nv_bfloat16* __restrict__ gq, const __nv_bfloat16* __restrict__ gk,
                             const __nv_bfloat16* __restrict__ gf, const float* __restrict__ A,
                             const float* __restrict__ tau, __nv_bfloat16* dq, __nv_bfloat16* dk, __nv_bfloat16* df,
                             float* __restrict__ partAT, int T, int H, int LCc, int l2norm, float eps, const int* flags,
                             int chains)
{
    // A lane owns 8 channels (one 16-byte piece) of a row; a warp covers RPW rows per load.  All six loads of a row
    // group are issued before anything is computed or stored (the in-place stores would otherwise order every later
    // load behind them): per SM this grid runs on the few SMs the reverse kernel leaves idle, so what counts is the
    // number of bytes a warp keeps in flight, not the DRAM bandwidth of the whole machine.
    constexpr int LPR = D / 8, RPW = 32 / LPR, NIT = 64 / (8 * RPW), UN = 1;
    __shared__ float red[8][2][D];
    const int nchunks = T / LCc;
    // blocks in the order the reverse kernel finishes chunks (last chunk of every chain first): this grid may already
    // run, on idle SMs, while the reverse kernel works; a block waits for "its" chunk through the chain's progress flag
    const int c = nchunks - 1 - (int)(blockIdx.x / chains), chain = blockIdx.x % chains, b = chain / H, h = chain % H;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, sub = lane / LPR, l = lane % LPR;
    float eA[8], ta[8], accA[8], accT[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) {
        const int j = l * 8 + e;
        eA[e] = A ? __expf(__ldg(A + h * D + j)) : 1.f;
        ta[e] = tau ? __ldg(tau + h * D + j) : 0.f;
        accA[e] = accT[e] = 0.f;
    }
    if (threadIdx.x == 0) {
        int done;
        do {
            asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(done) : "l"(flags + chain) : "memory");
            if (done < nchunks - c) __nanosleep(256);
        } while (done < nchunks - c);
    }
    __syncthreads();
    auto gsum = [](float x) {   // sum over the LPR lanes of a row
#pragma unroll
        for (int o = LPR / 2; o > 0; o >>= 1) x += __shfl_xor_sync(0xFFFFFFFFu, x, o);
        return x;
    };
    const size_t row0 = ((size_t)b * T + (size_t)c * LCc) * H + h;
#pragma unroll
    for (int i0 = 0; i0 < NIT; i0 += UN) {
        uint4 in[UN][6];
        size_t ro[UN];
        bool on[UN];
#pragma unroll
        for (int u = 0; u < UN; ++u) {
            const int tt_ = ((i0 + u) * 8 + warp) * RPW + sub;
            on[u] = tt_ < LCc;
            ro[u] = (row0 + (size_t)(on[u] ? tt_ : 0) * H) * D + l * 8;
            const uint4 z = make_uint4(0u, 0u, 0u, 0u);
            in[u][0] = l2norm ? *reinterpret_cast<const uint4*>(gq + ro[u]) : z;
            in[u][1] = l2norm ? *reinterpret_cast<const uint4*>(dq + ro[u]) : z;
            in[u][2] = l2norm ? *reinterpret_cast<const uint4*>(gk + ro[u]) : z;
            in[u][3] = l2norm ? *reinterpret_cast<const uint4*>(dk + ro[u]) : z;
            in[u][4] = *reinterpret_cast<const uint4*>(gf + ro[u]);
            in[u][5] = *reinterpret_cast<const uint4*>(df + ro[u]);
        }
#pragma unroll
        for (int u = 0; u < UN; ++u) {
            if (l2norm) {
#pragma unroll
                for (int which = 0; which < 2; ++which) {
                    float x[8], dx[8];
                    unpack8(in[u][2 * which], x);
                    unpack8(in[u][2 * which + 1], dx);
                    float ss = 0.f;
#pragma unroll
                    for (int e = 0; e < 8; ++e) ss += x[e] * x[e];
                    const float rn = rsqrtf(gsum(ss) + eps);
                    float dot = 0.f;
#pragma unroll
                    for (int e = 0; e < 8; ++e) { x[e] *= rn; dot += x[e] * dx[e]; }
                    dot = gsum(dot);
#pragma unroll
                    for (int e = 0; e < 8; ++e) dx[e] = (dx[e] - x[e] * dot) * rn;
                    if (on[u]) *reinterpret_cast<uint4*>((which ? dk : dq) + ro[u]) = pack8(dx);
                }
            }
            float fv[8], dla[8];
            unpack8(in[u][4], fv);
            unpack8(in[u][5], dla);
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                // sigmoid and softplus of the same argument share exp(-|z|): 3 transcendental ops, not 4
                const float z = fv[e] + ta[e];
                const float ex = ex2_ftz(-fabsf(z) * kLog2e), s1p = 1.f + ex, rs = rcp_ftz(s1p);
                const float sg = z >= 0.f ? rs : ex * rs;
                const float sp = fmaf(kLn2, lg2_ftz(s1p), fmaxf(z, 0.f));
                const float d = dla[e] * (-eA[e]) * sg;
                if (on[u]) {
                    accT[e] += d;
                    accA[e] += dla[e] * (-eA[e] * sp);
                }
                dla[e] = d;
            }
            if (on[u]) *reinterpret_cast<uint4*>(df + ro[u]) = pack8(dla);
        }
    }
#pragma unroll
    for (int e = 0; e < 8; ++e) {   // rows of the warp -> one partial per channel
#pragma unroll
        for (int o = LPR; o < 32; o <<= 1) {
            accA[e] += __shfl_xor_sync(0xFFFFFFFFu, accA[e], o);
            accT[e] += __shfl_xor_sync(0xFFFFFFFFu, accT[e], o);
        }
        if (sub == 0) { red[warp][0][l * 8 + e] = accA[e]; red[warp][1][l * 8 + e] = accT[e]; }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 2 * D; i += 256) {
        float s = 0.f;
#pragma unroll
        for (int w = 0; w < 8; ++w) s += red[w][i / D][i % D];
        partAT[((size_t)chain * nchunks + c) * 2 * D + i] = s;
    }
    // Launched with programmatic stream serialization: the grid must not complete before the reverse kernel has (the
    // reductions that follow in the stream read its per-chain partials).  The chunk-0 blocks -- last in block order, so
    // they hold no SM while earlier chunks still have work -- wait for the primary grid here; a no-op for a plain launch.
    if (c == 0) asm volatile("griddepcontrol.wait;" ::: "memory");
}

// part[chain][nW + which*dk + j] = sum over the chain's chunks of partAT (fixed order: deterministic).
__global__ void carve_reduce_at_kernel(const float* __restrict__ partAT, float* part, int nchunks, int stride, int nW, int D)
{
    const int chain = blockIdx.x, i = threadIdx.x;
    if (i >= 2 * D) return;
    float s = 0.f;
    for (int c = 0; c < nchunks; ++c) s += partAT[((size_t)chain * nchunks + c) * 2 * D + i];
    part[(size_t)chain * stride + nW + i] = s;
}

template <int D, int SW>
cudaError_t launch_tc_bwd(const Args& a, uint8_t* ws, const TcWsLayout& w, float* dA, float* dtau, float* dUb, float* dUw,
                          float* dVb, float* dVw, cudaStream_t st)
{
    const int LCc = a.L < tcp::LC ? a.L : tcp::LC;
    CUtensorMap mdO, mq, mdq, mdk, mdv, mdf, mdbx, mdwx;
    if (!tc_make_token_map(&mdO, a.dO, a.B, a.T, a.H, D, LCc) || !tc_make_token_map(&mq, a.q, a.B, a.T, a.H, D, LCc) ||
        !tc_make_token_map(&mdq, a.dq, a.B, a.T, a.H, D, LCc) || !tc_make_token_map(&mdk, a.dk_, a.B, a.T, a.H, D, LCc) ||
        !tc_make_token_map(&mdv, a.dv_, a.B, a.T, a.H, D, LCc) || !tc_make_token_map(&mdf, a.df, a.B, a.T, a.H, D, LCc) ||
        !tc_make_token_map(&mdbx, a.dbx, a.B, a.T, a.H, D, LCc) ||
        !tc_make_token_map(&mdwx, a.dwx ? a.dwx : a.dv_, a.B, a.T, a.H, D, LCc))   // (scalar-write variant: the map is never used)
        return cudaErrorInvalidValue;
    BwdArgs t{};
    t.B = a.B; t.H = a.H; t.T = a.T; t.L = a.L; t.r = a.r; t.l2norm = a.l2norm; t.scale = a.scale; t.eps = a.eps;
    t.rec = ws + w.rec; t.dS_final = a.dS_final; t.sw = a.wx == nullptr;
    t.Ub = a.Ub; t.Uw = a.Uw; t.Vb = a.Vb; t.Vw = a.Vw;
    t.dq = static_cast<__nv_bfloat16*>(a.dq); t.dk = static_cast<__nv_bfloat16*>(a.dk_);
    t.dv = static_cast<__nv_bfloat16*>(a.dv_); t.df = static_cast<__nv_bfloat16*>(a.df);
    t.dbx = static_cast<__nv_bfloat16*>(a.dbx); t.dwx = static_cast<__nv_bfloat16*>(a.dwx);
    t.dbeta = static_cast<__nv_bfloat16*>(a.dbeta); t.dS0 = a.dS0;
    t.part = reinterpret_cast<float*>(ws + w.part); t.part_stride = w.part_stride;
    t.dgs = reinterpret_cast<float*>(ws + w.dgs);
    t.flags = reinterpret_cast<int*>(ws + w.flags);
    const size_t smem = BLayout(D).total;
    constexpr int NP = D / 32;   // 32 columns per thread: 256 threads at d = 64, 512 at d = 128
    auto kern = a.L >= tcp::LC ? carve_bwd_tc_kernel<D, NP, SW, 1> : carve_bwd_tc_kernel<D, NP, SW, 0>;
    if constexpr (D == 128 && SW == 0) {   // config 2's short chunks: the chunk length as a constant as well
        if (a.L == 16 && a.r == 16) kern = carve_bwd_tc_kernel<D, NP, SW, 16, 16>;
        if (a.L == 32 && a.r == 16) kern = carve_bwd_tc_kernel<D, NP, SW, 32, 16>;
    }
    if (a.L >= tcp::LC && a.r == (D == 128 ? 16 : 8)) kern = carve_bwd_tc_kernel<D, NP, SW, 1, (D == 128 ? 16 : 8)>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int chains = a.B * a.H, nchunks = a.T / LCc;
    if ((e = cudaMemsetAsync(t.flags, 0, (size_t)chains * sizeof(int), st)) != cudaSuccess) return e;
    kern<<<chains, 128 * NP, smem, st>>>(t, mdO, mq, mdq, mdk, mdv, mdf, mdbx, mdwx);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    float* partAT = reinterpret_cast<float*>(ws + w.partAT);
    {
        // programmatic stream serialization: the epilogue grid may be scheduled while the reverse kernel is still running
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3((unsigned)(chains * nchunks));
        cfg.blockDim = dim3(256);
        cfg.dynamicSmemBytes = 0;
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = a.epilogue_after ? 0 : 1;
        e = cudaLaunchKernelEx(&cfg, carve_bwd_tc_epilogue_kernel<D>, static_cast<const __nv_bfloat16*>(a.q),
                               static_cast<const __nv_bfloat16*>(a.k), static_cast<const __nv_bfloat16*>(a.f), a.A, a.tau, t.dq,
                               t.dk, t.df, partAT, a.T, a.H, LCc, a.l2norm, a.eps, (const int*)t.flags, chains);
        if (e != cudaSuccess) return e;
    }
    const int nW = 2 * a.r * D + 2 * D * a.r;
    carve_reduce_at_kernel<<<chains, 2 * D, 0, st>>>(partAT, t.part, nchunks, w.part_stride, nW, D);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    return reduce_weights_launch(t.part, chains, w.part_stride, a.H, D, D, a.r, dUb, dUw, dVb, dVw, dA, dtau, st);
}

}  // namespace

#ifdef CARVE_PROFILE
extern "C" void carve_debug_profb_bwd(unsigned long long* out)
{
    cudaMemcpyFromSymbol(out, g_profb_bwd, sizeof(g_profb_bwd));
    static unsigned long long z[64 * 16];
    cudaMemcpyToSymbol(g_profb_bwd, z, sizeof(z));
}
extern "C" void carve_debug_prof_bwd(unsigned long long* out)
{
    cudaMemcpyFromSymbol(out, g_prof_bwd, sizeof(g_prof_bwd));
    unsigned long long z[80] = {};
    cudaMemcpyToSymbol(g_prof_bwd, z, sizeof(z));
}
#endif

bool tc_bwd_supported(const carve_params_t& p) { return tc_fwd_supported(p) && p.dk == p.dv; }

cudaError_t tc_bwd_launch(const Args& a, uint8_t* ws, const TcWsLayout& w, float* dA, float* dtau, float* dUb, float* dUw,
                          float* dVb, float* dVw, cudaStream_t st)
{
    const bool sw = a.wx == nullptr;
    if (a.dk == 128) return sw ? launch_tc_bwd<128, 1>(a, ws, w, dA, dtau, dUb, dUw, dVb, dVw, st) : launch_tc_bwd<128, 0>(a, ws, w, dA, dtau, dUb, dUw, dVb, dVw, st);
    if (a.dk == 64) return sw ? launch_tc_bwd<64, 1>(a, ws, w, dA, dtau, dUb, dUw, dVb, dVw, st) : launch_tc_bwd<64, 0>(a, ws, w, dA, dtau, dUb, dUw, dVb, dVw, st);
    return cudaErrorInvalidValue;
}

}  // namespace carve

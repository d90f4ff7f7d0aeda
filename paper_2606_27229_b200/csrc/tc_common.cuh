// tc_common.cuh -- sm_100a building blocks of the tensor-core path: mbarrier, TMA, tcgen05 (TMEM
// allocation, UMMA issue/commit, TMEM load/store) as inline PTX, plus the ONE shared-memory tile
// format every MMA operand of the CARVE kernels uses and the UMMA descriptors that view it.
//
// Tile format ("row tile"): a logical [rows][cols] bf16 matrix, cols split into blocks of 64
// (128 bytes).  Inside a block, row r occupies 128 contiguous bytes at (r/8)*1024 + (r%8)*128 and
// its eight 16-byte chunks are XOR-swizzled with (r%8) -- the 128B swizzle TMA writes and
// tcgen05.mma reads.  Column block b starts at b*rows*128.  The same bytes are
//   * a K-major  operand with MN = row, K = col   (SWIZZLE_128B, SBO = 1024), and
//   * an MN-major operand with MN = col, K = row  (SWIZZLE_128B, LBO = rows*128, SBO = 1024),
// so a thread that owns a row writes it with 16-byte stores and the tile can feed an MMA either way.
#pragma once
#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

// Optional per-phase cycle counters (build with -DCARVE_PROFILE; block 0: thread 0 = the MMA-issuing, K-side
// thread in slots 0.., thread 64 = a Q-side thread in slots 40..).
#ifdef CARVE_PROFILE
#define PROF_DECL(name) static __device__ unsigned long long name[80];
// counters accumulate in shared memory (a global read-modify-write would stall the profiled thread for an L2 round
// trip at every point) and are added to the global array once, by PROF_FLUSH at the kernel's end
#define PROF_INIT()                                            \
    __shared__ unsigned long long prof_s_[80];                 \
    __shared__ long long prof_arr_[2][16];                     \
    if (threadIdx.x < 80) prof_s_[threadIdx.x] = 0;            \
    __syncthreads();                                           \
    long long prof_t_ = clock64();
#define PROF(name, i)                                                              \
    if (blockIdx.x == 0 && (threadIdx.x == 0 || threadIdx.x == 64)) {              \
        const long long prof_n_ = clock64();                                       \
        prof_s_[(threadIdx.x ? 40 : 0) + i] += (unsigned long long)(prof_n_ - prof_t_); \
        prof_t_ = prof_n_;                                                         \
    }
// barrier-spread profile (-DCARVE_PROFILE_BARRIERS as well: its own overhead is ~1 K cycles per site, so the per-phase
// counters are read from a build without it): per barrier site and warp, how long the warp waited for the last one
#ifdef CARVE_PROFILE_BARRIERS
#define PROFB_DECL(name) static __device__ unsigned long long name[64 * 16];
#define PROFB_ARRIVE(site) if ((threadIdx.x & 31) == 0) prof_arr_[(site) & 1][threadIdx.x >> 5] = clock64();
#define PROFB_AFTER(name, site)                                                                     \
    if (blockIdx.x == 0 && (threadIdx.x & 31) == 0) {                                               \
        long long mx_ = 0;                                                                          \
        for (int w_ = 0; w_ < (int)(blockDim.x >> 5); ++w_) mx_ = mx_ > prof_arr_[(site) & 1][w_] ? mx_ : prof_arr_[(site) & 1][w_]; \
        atomicAdd(&name[(site) * 16 + (threadIdx.x >> 5)], (unsigned long long)(mx_ - prof_arr_[(site) & 1][threadIdx.x >> 5])); \
    }
#else
#define PROFB_DECL(name) static __device__ unsigned long long name[64 * 16];
#define PROFB_ARRIVE(site)
#define PROFB_AFTER(name, site)
#endif
#define PROF_FLUSH(name)                                                           \
    __syncthreads();                                                               \
    if (blockIdx.x == 0 && threadIdx.x < 80) name[threadIdx.x] += prof_s_[threadIdx.x];
#else
#define PROF_DECL(name)
#define PROF_INIT()
#define PROF(name, i)
#define PROF_FLUSH(name)
#define PROFB_DECL(name)
#define PROFB_ARRIVE(site)
#define PROFB_AFTER(name, site)
#endif

namespace carve {
namespace tc {

// ---- addresses -----------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// Byte offset of element (row, col) inside a row tile of `rows` rows.
__host__ __device__ __forceinline__ uint32_t tile_off(int rows, int row, int col)
{
    return (uint32_t)((col >> 6) * rows * 128 + (row >> 3) * 1024 + (row & 7) * 128 +
                      ((((col & 63) >> 3) ^ (row & 7)) << 4) + (col & 7) * 2);
}
// Byte offset of the 16-byte chunk holding columns [8*chunk, 8*chunk+8) of `row`.
__host__ __device__ __forceinline__ uint32_t tile_chunk_off(int rows, int row, int chunk)
{
    return (uint32_t)((chunk >> 3) * rows * 128 + (row >> 3) * 1024 + (row & 7) * 128 + (((chunk & 7) ^ (row & 7)) << 4));
}
__host__ __device__ constexpr uint32_t tile_bytes(int rows, int cols) { return (uint32_t)(((cols + 63) / 64) * rows * 128); }

// ---- mbarrier ------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) {}
}

// ---- proxies / fences ----------------------------------------------------------------------------
// Generic-proxy smem writes -> visible to the async proxy (TMA, tcgen05.mma operand reads).
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// ---- TMA -----------------------------------------------------------------------------------------
// 3-D tiled load: coordinates (c0 = innermost).  Completion is signalled on `bar` (complete_tx).
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}
// 3-D tiled store shared -> global (bulk group of the issuing thread; the source may be rewritten after bulk_wait_read()).
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* map, uint32_t src_saddr, int c0, int c1, int c2)
{
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];" ::"l"(map), "r"(src_saddr),
                 "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
// The same box, fetched into L2 only (no shared-memory destination, no completion signal).
__device__ __forceinline__ void tma_prefetch_3d(const CUtensorMap* map, int c0, int c1, int c2)
{
    asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global.tile [%0, {%1, %2, %3}];" ::"l"(map), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map)
{
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

// 1-D bulk copies.  Global -> shared completes on an mbarrier; shared -> global is tracked by bulk groups:
// the source may be overwritten once bulk_wait_read() returns.
__device__ __forceinline__ void bulk_s2g(void* gdst, uint32_t src_saddr, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(src_saddr), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
// every bulk group of this thread except the N most recent ones is complete (writes performed)
template <int N>
__device__ __forceinline__ void bulk_wait_all_but() { asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory"); }

// ---- TMEM ----------------------------------------------------------------------------------------
// One full warp allocates `ncols` (power of two >= 32) columns; the base address lands in *dst (smem).
__device__ __forceinline__ void tmem_alloc(uint32_t* dst, uint32_t ncols)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(dst)), "r"(ncols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}

// 32 lanes x 32 columns of 32-bit: thread i of the warp receives columns [col, col+32) of lane
// (32*(warp%4) + i).  `taddr` must already carry the warp's lane base in bits [31:16].
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&r)[8])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr)
                 : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&r)[8])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                 ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
                 : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16])
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
        ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
          "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&r)[32])
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
        "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};"
        ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
          "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]),
          "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]),
          "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
        : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// ---- UMMA descriptors ----------------------------------------------------------------------------
// Shared-memory matrix descriptor (SWIZZLE_128B, version 1).  Offsets in bytes, multiples of 16.
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32) | (1ull << 46) | (2ull << 61);
}
// K-major view of a row tile (MN = row, K = col): operand rows start at `row0` (multiple of 8),
// the 16 K-values of this instruction start at column `k0` (multiple of 16).
__device__ __forceinline__ uint64_t desc_kmajor(uint32_t tile_saddr, int rows, int row0, int k0)
{
    const uint32_t a = tile_saddr + (uint32_t)((k0 >> 6) * rows * 128 + (row0 >> 3) * 1024 + ((k0 & 63) >> 3) * 16);
    return umma_desc(a, 16, 1024);
}
// MN-major view of a row tile (MN = col, K = row): MN starts at column `mn0` (multiple of 64 when
// the operand spans more than one 64-column block, else a multiple of 8), the 16 K-values start at
// row `k0` (multiple of 8).
__device__ __forceinline__ uint64_t desc_mnmajor(uint32_t tile_saddr, int rows, int mn0, int k0)
{
    const uint32_t a = tile_saddr + (uint32_t)((mn0 >> 6) * rows * 128 + (k0 >> 3) * 1024 + ((mn0 & 63) >> 3) * 16);
    return umma_desc(a, (uint32_t)rows * 128, 1024);
}
// Instruction descriptor, kind::f16, bf16 x bf16 -> fp32.  a_mn / b_mn: 1 = MN-major operand.
__host__ __device__ constexpr uint32_t umma_idesc(int M, int N, int a_mn, int b_mn)
{
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)a_mn << 15) | ((uint32_t)b_mn << 16) |
           ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
// D[tmem] (+)= A[smem] * B[smem]^T, one K=16 slice.  Issued by ONE thread.
__device__ __forceinline__ void umma(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// Arrive on `bar` when every tcgen05.mma issued so far by this thread has completed.
__device__ __forceinline__ void umma_commit(uint64_t* bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}

// Which operand view an MMA uses.
enum : int { KMAJ = 0, MNMAJ = 1 };

// Descriptor of the next K = 16 slice, given the descriptor of the slice that starts at K index `k` (relative
// to the tile): K-major operands advance 32 bytes inside a 64-column block and jump to the next block
// (rows*128 bytes further) after four slices; MN-major operands advance two 8-row groups (2048 bytes).
template <int MAJ>
__device__ __forceinline__ uint64_t desc_next(uint64_t d, int rows, int k)
{
    if (MAJ == 0) return d + ((((k + 16) & 63) == 0) ? (uint64_t)(rows * 8 - 6) : 2ull);
    return d + 128ull;
}

// Full product over K (multiple of 16) from two row tiles.  For a K-major operand `o0` is its first
// MN row and K runs over columns from `k0`; for an MN-major operand `o0` is its first MN column and
// K runs over rows from `k0`.  M = 128; N at run time.  Issued by ONE thread.
template <int AMAJ, int BMAJ>
__device__ __forceinline__ void umma_tiles_rt(uint32_t d_tmem, int M, int N, uint32_t a_saddr, int a_rows, int a_o0,
                                              int a_k0, uint32_t b_saddr, int b_rows, int b_o0, int b_k0, int K,
                                              bool accumulate)
{
    const uint32_t idesc = umma_idesc(M, N, AMAJ, BMAJ);
    uint64_t ad = AMAJ == KMAJ ? desc_kmajor(a_saddr, a_rows, a_o0, a_k0) : desc_mnmajor(a_saddr, a_rows, a_o0, a_k0);
    uint64_t bd = BMAJ == KMAJ ? desc_kmajor(b_saddr, b_rows, b_o0, b_k0) : desc_mnmajor(b_saddr, b_rows, b_o0, b_k0);
    for (int k = 0; k < K; k += 16) {
        umma(d_tmem, ad, bd, idesc, (accumulate || k > 0) ? 1u : 0u);
        ad = desc_next<AMAJ>(ad, a_rows, a_k0 + k);
        bd = desc_next<BMAJ>(bd, b_rows, b_k0 + k);
    }
}

// One lane of a converged warp (the same one every time): the thread that issues tcgen05.mma / commit / TMA.
__device__ __forceinline__ bool elect_one()
{
    uint32_t el;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(el));
    return el != 0;
}

// As umma_tiles_rt, fully unrolled over K <= KMAX (slices beyond the run-time K are predicated off): issued from a
// warp-uniform branch by the elected lane this costs ~20 cycles per instruction instead of ~90 for the rolled loop
// inside a divergent `if (tid == 0)` (measured; the compiler wraps every tcgen05.mma of a divergent region in an
// ELECT / R2UR.BROADCAST loop and keeps the descriptor arithmetic on the slow uniform datapath).
template <int AMAJ, int BMAJ, int KMAX>
__device__ __forceinline__ void umma_prod(uint32_t d_tmem, int M, int N, uint32_t a_saddr, int a_rows, int a_o0, int a_k0,
                                          uint32_t b_saddr, int b_rows, int b_o0, int b_k0, int K, bool accumulate)
{
    const uint32_t idesc = umma_idesc(M, N, AMAJ, BMAJ);
    uint64_t ad = AMAJ == KMAJ ? desc_kmajor(a_saddr, a_rows, a_o0, a_k0) : desc_mnmajor(a_saddr, a_rows, a_o0, a_k0);
    uint64_t bd = BMAJ == KMAJ ? desc_kmajor(b_saddr, b_rows, b_o0, b_k0) : desc_mnmajor(b_saddr, b_rows, b_o0, b_k0);
#pragma unroll
    for (int k = 0; k < KMAX; k += 16) {
        if (k < K) umma(d_tmem, ad, bd, idesc, (accumulate || k > 0) ? 1u : 0u);
        ad = desc_next<AMAJ>(ad, a_rows, a_k0 + k);
        bd = desc_next<BMAJ>(bd, b_rows, b_k0 + k);
    }
}

// ---- packing -------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi)
{
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xFFFF0000u); }

}  // namespace tc
}  // namespace carve

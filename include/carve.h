/*
 * carve.h -- C ABI of the B200 (sm_100a) CARVE layer operator.
 *
 * The operator is the chunk-parallel key-axis-gated delta rule of arxiv/paper_2606_27229
 * (/root/reference/PAPER.md, cited below as "P l.<line>"), forward and backward, for every
 * (batch, head) chain independently:
 *
 *   for each chunk c of L tokens, with S = state entering the chunk (S_{c-1}):
 *     q^ = q/sqrt(|q|^2+eps), k^ likewise                      (Fig. 2, P l.437; Alg. 3 step 3, P l.399)
 *     g_t = -exp(A) . softplus(f_t + tau)                      (Eq. 9,  P l.151)
 *     G   = [U_b;U_w] S ; t_t = tanh(G q^_t)                    (Eq. 7,  P l.134)  folded state readout
 *     b_t = sigmoid(bx_t + V_b t_t^(b)),  w_t = sigmoid(wx_t + V_w t_t^(w))      (Eq. 8,  P l.140)
 *     gamma_t = prod_{s<=t} exp(g_s).(1-b_s)                   (Eq. 14, P l.310)
 *     A_ts = sum_j k^_t k^_s gamma_{t-1}/gamma_s (s<t)          (Eq. 15, P l.342, Eq. 5 indices)
 *     (I + diag(beta) A) U = diag(beta) (w.v - K~ S^T),  K~_t = k^_t.gamma_{t-1}     (Alg. 2 steps 5-7, P l.333-352)
 *     o_t = scale [ S (gamma_t.q^_t) + sum_{s<=t} u_s sum_j q^_t k^_s gamma_t/gamma_s ]   (Alg. 2 step 8, P l.354)
 *     S  <- S diag(gamma_{L-1}) + sum_t u_t (k^_t.gamma_{L-1}/gamma_t)^T            (Alg. 2 step 9, P l.361)
 *
 *   which equals, token by token (Eq. 5, P l.108, with the gates frozen at the chunk boundary):
 *     u_t = beta_t (w_t.v_t - S_{t-1} k^_t);  S_t = S_{t-1} diag(exp(g_t).(1-b_t)) + u_t k^_t^T;  o_t = scale S_t q^_t.
 *
 *   carve_bwd is the adjoint of that map (Alg. 4-5, P l.788-863).  DESIGN.md lists the readings of
 *   the paper taken where it is ambiguous (write gate on v only, the scalar beta, the Eq. 5 order).
 *
 * Conventions
 *   - Every tensor pointer of carve_fwd / carve_bwd is a DEVICE pointer owned by the caller; the
 *     library allocates nothing and keeps no global state.  carve_fwd_bwd_host takes HOST pointers
 *     for the tensors and one caller-owned DEVICE arena.
 *   - Row-major, innermost dimension contiguous.  Token tensors are [B,T,H,d] (P l.125); the state is
 *     [B,H,dv,dk] (P l.11).  Base pointers must be 16-byte aligned.
 *   - `dtype` is the element type of the token tensors q,k,v,f,bx,wx,beta,O and of their gradients
 *     (CARVE_F32: float, CARVE_BF16: __nv_bfloat16 bits).  A, tau, U_b, U_w, V_b, V_w, S0, S_final and
 *     their gradients are always float.  All arithmetic on the state is fp32.
 *   - Calls are asynchronous on `cuda_stream` (a cudaStream_t passed as void*, NULL = default
 *     stream) and return after enqueueing.  Argument errors are detected on the host before any
 *     launch and leave all outputs untouched.  Gradients are OVERWRITTEN, not accumulated.
 *   - Results are run-to-run bitwise deterministic (no floating-point atomics).
 *   - Supported: T % L == 0, L in {16,32,64,128}; dk, dv in {64,128,256} with dk*dv <= 32768;
 *     r in {8,16,32}.  carve_bwd additionally needs dk*dv <= 16384 and dk <= 128.  Anything else returns
 *     CARVE_ERR_SHAPE: there is no fallback path of any kind.
 */
#ifndef CARVE_H_
#define CARVE_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    CARVE_OK = 0,
    CARVE_ERR_NULL = 1,      /* a required pointer is NULL */
    CARVE_ERR_SHAPE = 2,     /* unsupported B,H,T,L,dk,dv,r combination */
    CARVE_ERR_DTYPE = 3,     /* dtype is neither CARVE_F32 nor CARVE_BF16 */
    CARVE_ERR_ALIGN = 4,     /* a base pointer is not 16-byte aligned */
    CARVE_ERR_WORKSPACE = 5, /* workspace missing or smaller than carve_workspace_bytes() */
    CARVE_ERR_ARCH = 6,      /* current device is not compute capability 10.x */
    CARVE_ERR_CUDA = 7,      /* a CUDA runtime call failed (launch, attribute, copy) */
    CARVE_ERR_STATIC_LIMIT = 8 /* carve_fwd_bwd_static: the problem needs more than CARVE_STATIC_SCRATCH_BYTES of scratch */
} carve_status_t;

typedef enum { CARVE_F32 = 0, CARVE_BF16 = 1 } carve_dtype_t;

/* Kernel family.  AUTO picks TENSOR for the shapes it covers and SIMT otherwise.  TENSOR (tcgen05 + TMA, fp32
 * state in tensor memory) covers bf16 tokens with r <= 16 and dk == dv in {64,128} (forward and backward, every L),
 * plus dk = 128, dv = 256 with L <= 64 for inference calls (forward without workspace).  An explicit TENSOR
 * request outside that set returns CARVE_ERR_SHAPE; carve_resolved_path reports the choice. */
typedef enum { CARVE_PATH_AUTO = 0, CARVE_PATH_SIMT = 1, CARVE_PATH_TENSOR = 2 } carve_path_t;

typedef struct {
    int B, H, T;          /* batch, heads, tokens per sequence */
    int L;                /* chunk length: the gates of a chunk read the state at its start (P l.136) */
    int dk, dv, r;        /* key dim, value dim, gate bottleneck rank */
    int dtype;            /* carve_dtype_t */
    int qk_l2norm;        /* 1: L2-normalise q,k inside and differentiate through it; 0: use as given */
    float scale;          /* multiplies O (the paper is silent; 1.0f) */
    float eps;            /* inside the sqrt of the L2 norm (1e-6f) */
    int path;             /* carve_path_t */
} carve_params_t;

/* Bytes of device workspace carve_fwd needs to save what carve_bwd reads (need_bwd != 0), or 0. */
size_t carve_workspace_bytes(const carve_params_t *p, int need_bwd);

/*
 * Forward (Alg. 1-3, P l.160-196, l.315-365, l.395-409).
 *   q,k   [B,T,H,dk] dtype      v   [B,T,H,dv] dtype
 *   f,bx  [B,T,H,dk] dtype      decay logits, erase pre-activation (Eq. 6 ff., P l.128)
 *   wx    [B,T,H,dv] dtype      write pre-activation
 *   beta  [B,T,H]    dtype      write strength in [0,1], already activated
 *   A,tau [H,dk] float          Eq. 9 parameters; either may be NULL (= 0)
 *   Ub,Uw [r,dv] float          down-projections W_{U1,b}, W_{U1,w} (Eq. 7), shared by all heads
 *   Vb [dk,r], Vw [dv,r] float  up-projections W_{U2,b}, W_{U2,w} (Eq. 8)
 *   S0    [B,H,dv,dk] float     initial state, NULL = zeros
 *   O     [B,T,H,dv] dtype      out
 *   S_final [B,H,dv,dk] float   out
 *   workspace                   NULL: inference, nothing saved.  Otherwise >= carve_workspace_bytes(p,1)
 *                               bytes; it is filled for the matching carve_bwd call.
 * Scalar-write variant (P section 4.2 l.145, Thm 15 l.762-764: the per-head scalar write gate w_{h,t} = sigmoid(w^_{h,t}),
 * broadcast over d_v, is sufficient; reading A1: that scalar multiplies the whole error, so it is passed inside beta):
 * wx = Uw = Vw = NULL (all three) selects kernels' w == 1 path: V' = v, no write-gate load, projection or sigmoid, and
 * the training forward saves nothing for it.  carve_bwd / carve_step take the same three NULLs; carve_bwd then does not
 * write dwx, dUw, dVw (they may be NULL).  Only some of the three NULL is CARVE_ERR_NULL.
 */
carve_status_t carve_fwd(const carve_params_t *p, const void *q, const void *k, const void *v,
                         const void *f, const void *bx, const void *wx, const void *beta,
                         const float *A, const float *tau, const float *Ub, const float *Uw,
                         const float *Vb, const float *Vw, const float *S0, void *O, float *S_final,
                         void *workspace, size_t workspace_bytes, void *cuda_stream);

/*
 * Backward (Alg. 4-5, P l.788-863): adjoint of carve_fwd for the cotangents dO and dS_final.
 * Same inputs as the carve_fwd call that filled `workspace`, plus
 *   dO [B,T,H,dv] dtype;  dS_final [B,H,dv,dk] float, NULL = zeros.
 * Outputs (overwritten): dq,dk,df,dbx [B,T,H,dk] dtype; dv,dwx [B,T,H,dv] dtype; dbeta [B,T,H] dtype;
 *   dA,dtau [H,dk] float (either may be NULL to skip); dUb,dUw [r,dv]; dVb [dk,r]; dVw [dv,r];
 *   dS0 [B,H,dv,dk] float.
 */
carve_status_t carve_bwd(const carve_params_t *p, const void *q, const void *k, const void *v,
                         const void *f, const void *bx, const void *wx, const void *beta,
                         const float *A, const float *tau, const float *Ub, const float *Uw,
                         const float *Vb, const float *Vw, const float *S0, const void *dO,
                         const float *dS_final, void *dq, void *dk, void *dv, void *df, void *dbx,
                         void *dwx, void *dbeta, float *dA, float *dtau, float *dUb, float *dUw,
                         float *dVb, float *dVw, float *dS0, void *workspace, size_t workspace_bytes,
                         void *cuda_stream);

/*
 * Recurrent (decode) step: a few new tokens per sequence, state in and out (P Table 1 l.432 "Infer/tok O(d_v d_k)",
 * l.27; chunk mode == sequential at chunk size 1, Table 2 l.450).
 *   p->T = n new tokens per sequence, 1 <= n <= 16; they form ONE gate chunk (p->L is ignored): the content gates
 *   of all n tokens read the incoming state, G = [Ub;Uw] S (Eq. 7 l.134), and each token applies Eq. 5 (l.108).
 *   n = 1 is exact per-token content gating.  The result equals carve_fwd with T = L = n and S0 = S.
 *   q,k,f,bx [B,n,H,dk]; v,wx [B,n,H,dv]; beta [B,n,H] (dtype); weights as carve_fwd (A, tau may be NULL).
 *   S [B,H,dv,dk] float, IN/OUT: the state before the step, overwritten by the state after it (never NULL).
 *   O [B,n,H,dv] dtype, out.
 * Shapes: dk in {64,128}, dv in {64,128} (or dv = 256 with dk = 128), r in {8,16,32}; fp32 arithmetic for both
 * dtypes; one kernel launch; no workspace.  Errors as carve_fwd (CARVE_ERR_SHAPE for n > 16 or n < 1).
 */
carve_status_t carve_step(const carve_params_t *p, const void *q, const void *k, const void *v, const void *f,
                          const void *bx, const void *wx, const void *beta, const float *A, const float *tau,
                          const float *Ub, const float *Uw, const float *Vb, const float *Vw, float *S, void *O,
                          void *cuda_stream);

/*
 * carve_step on a ragged batch (the variable-length batches of a serving step: sequences that receive 0..T new tokens
 * each).  The token tensors are PACKED: q,k,f,bx [N,H,dk], v,wx,O [N,H,dv], beta [N,H] with N = cu_seqlens[B] rows in
 * total; sequence b owns rows cu_seqlens[b] .. cu_seqlens[b+1] (DEVICE int32 array of B + 1 non-decreasing entries,
 * cu_seqlens[0] = 0, read by the kernel: no host synchronisation).  p->T is the declared maximum number of new tokens of
 * any sequence (1..16); a sequence with more is processed up to p->T tokens only (the caller's contract violation, kept
 * memory-safe), a sequence with none keeps its state bit for bit and writes no output.  Each sequence's tokens form one
 * gate chunk of their own length, i.e. the result for sequence b equals carve_step on that sequence alone with
 * T = its length.  Everything else as carve_step; CARVE_ERR_NULL if cu_seqlens is NULL.
 */
carve_status_t carve_step_varlen(const carve_params_t *p, const void *q, const void *k, const void *v, const void *f,
                                 const void *bx, const void *wx, const void *beta, const float *A, const float *tau,
                                 const float *Ub, const float *Uw, const float *Vb, const float *Vw, float *S, void *O,
                                 const int *cu_seqlens, void *cuda_stream);

/*
 * Layer ends (the two chunk-local "hoisted" launches around the operator, Alg. 3 step 3 l.399 and step 9 l.407): fully
 * parallel over tokens, no state.  Only B, H, T, dk, dv and dtype of *p are read.  All pointers are DEVICE pointers,
 * 16-byte aligned, owned by the caller; token tensors are [B,T,H,d] row-major in p->dtype.
 *
 * carve_silu_qkv_fwd: q = SiLU(qx), k = SiLU(kx), v = SiLU(vx) (Eq. 6 l.125-126; qx = W_Q h etc. are the outputs of the
 *   input projections, dense GEMMs outside the path), one launch over the three tensors.  Output may alias its input.
 *   A tensor is skipped by passing NULL for both of its pointers (only one NULL: CARVE_ERR_NULL).
 * carve_silu_qkv_bwd: dq, dk, dv hold the gradients w.r.t. q, k, v (carve_bwd's outputs) and are overwritten IN PLACE by the
 *   gradients w.r.t. qx, kx, vx:  d x = d y (s + x s (1 - s)), s = sigmoid(x).
 * carve_out_norm_fwd: y = RMSNorm(reshape(o)) (Alg. 1 line 15 l.194): o, y [B,T,H,dv]; every token's H*dv channels are
 *   scaled by 1/sqrt(mean(o^2) + eps) and by gain [H*dv] (float).  W_O is a dense GEMM outside the path.  Rows of at most
 *   8 KB (H*dv <= 4096 bf16 / 2048 fp32), else CARVE_ERR_SHAPE.  y may alias o.
 * carve_out_norm_bwd: d_o [B,T,H,dv] and dgain [H*dv] (float, overwritten) from dy [B,T,H,dv]; the statistics are
 *   recomputed from o.  `workspace`: carve_out_norm_workspace_bytes(p) bytes of scratch (per-block partial sums of dgain,
 *   added in a fixed order: results are run-to-run bitwise identical), CARVE_ERR_WORKSPACE if missing or too small.
 *   d_o may alias dy.
 */
carve_status_t carve_silu_qkv_fwd(const carve_params_t *p, const void *qx, const void *kx, const void *vx, void *q, void *k,
                                  void *v, void *cuda_stream);
carve_status_t carve_silu_qkv_bwd(const carve_params_t *p, const void *qx, const void *kx, const void *vx, void *dq, void *dk,
                                  void *dv, void *cuda_stream);
carve_status_t carve_out_norm_fwd(const carve_params_t *p, const void *o, const float *gain, float eps, void *y,
                                  void *cuda_stream);
size_t carve_out_norm_workspace_bytes(const carve_params_t *p);
carve_status_t carve_out_norm_bwd(const carve_params_t *p, const void *o, const float *gain, float eps, const void *dy,
                                  void *d_o, float *dgain, void *workspace, size_t workspace_bytes, void *cuda_stream);

/* Bytes of device arena carve_fwd_bwd_host needs (device copies of every tensor + workspace). */
size_t carve_host_arena_bytes(const carve_params_t *p, int with_bwd);

/*
 * One forward (+ backward when with_bwd != 0) with HOST tensors: copies the inputs to the device
 * arena, runs carve_fwd (and carve_bwd with the host cotangents dO, dS_final), copies O, S_final
 * and the gradients back.  The batch is cut into up to 8 slices (the largest divisor of B that is <= 8), each
 * run on a short-lived stream of its own forked from and joined back into `cuda_stream`, so that copy-in,
 * kernels and copy-out of different slices overlap; work enqueued on `cuda_stream` before the call precedes
 * it, work enqueued after the call follows it.  The shared-weight gradients are the sums of the slices'
 * (fixed order: deterministic, but rounded differently from one carve_bwd over the whole batch).  Host
 * buffers should be pinned for the copies to be asynchronous.  Pointer meanings and NULL rules are those of carve_fwd / carve_bwd;
 * when with_bwd == 0 the cotangent and gradient pointers are ignored.
 */
carve_status_t carve_fwd_bwd_host(const carve_params_t *p, int with_bwd, const void *q, const void *k,
                                  const void *v, const void *f, const void *bx, const void *wx,
                                  const void *beta, const float *A, const float *tau, const float *Ub,
                                  const float *Uw, const float *Vb, const float *Vw, const float *S0,
                                  void *O, float *S_final, const void *dO, const float *dS_final,
                                  void *dq, void *dk, void *dv, void *df, void *dbx, void *dwx,
                                  void *dbeta, float *dA, float *dtau, float *dUb, float *dUw,
                                  float *dVb, float *dVw, float *dS0, void *device_arena,
                                  size_t arena_bytes, void *cuda_stream);

/*
 * The same call with caller-owned side streams and events: carve_fwd_bwd_host creates and destroys up to 8 streams and
 * 17 events per call; a context created once (carve_host_ctx_create) and passed to carve_fwd_bwd_host_ctx removes that
 * from every step.  One context serves one call at a time.  ctx = NULL behaves as carve_fwd_bwd_host.
 */
typedef struct carve_host_ctx carve_host_ctx_t;
carve_status_t carve_host_ctx_create(carve_host_ctx_t **ctx);
void carve_host_ctx_destroy(carve_host_ctx_t *ctx);
carve_status_t carve_fwd_bwd_host_ctx(carve_host_ctx_t *ctx, const carve_params_t *p, int with_bwd, const void *q,
                                      const void *k, const void *v, const void *f, const void *bx, const void *wx,
                                      const void *beta, const float *A, const float *tau, const float *Ub,
                                      const float *Uw, const float *Vb, const float *Vw, const float *S0, void *O,
                                      float *S_final, const void *dO, const float *dS_final, void *dq, void *dk,
                                      void *dv, void *df, void *dbx, void *dwx, void *dbeta, float *dA, float *dtau,
                                      float *dUb, float *dUw, float *dVb, float *dVw, float *dS0, void *device_arena,
                                      size_t arena_bytes, void *cuda_stream);

/*
 * carve_fwd_bwd_static -- training forward + backward for callers that cannot allocate device memory (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid cudaMalloc).  It is carve_fwd (training) followed by
 * carve_bwd on `cuda_stream`, with the workspace the two exchange -- the forward's chunk records (Alg. 2 l.315-365,
 * consumed by the reverse scan of Alg. 4 l.788-817), per-chain weight-gradient partials, progress flags -- held in a
 * file-scope __device__ array inside the library instead of a caller buffer.  Same kernels, same launch configuration,
 * same results as the two calls.  Arguments: exactly those of carve_fwd (inputs, O, S_final) and carve_bwd (dO,
 * dS_final, the gradients), all DEVICE pointers owned by the caller, same layouts, same NULL rules.
 *   - The array has CARVE_STATIC_SCRATCH_BYTES (16 MiB; carve_static_scratch_bytes() returns it).  Every GPU that
 *     loads the library holds it until the process exits.
 *   - A problem with carve_workspace_bytes(p, 1) > CARVE_STATIC_SCRATCH_BYTES returns CARVE_ERR_STATIC_LIMIT and
 *     launches nothing (tensor path: ~262 KB per (chain, 64-token chunk) at d = 128, i.e. <= 60 chain-chunks).
 *   - Calls no cudaMalloc, cudaFree or allocating library routine.
 *   - All calls share the array; it keeps the last call's contents.  The only region that must start at zero (the
 *     tensor path's progress flags) is cleared by the call itself on `cuda_stream`.
 *   - Calls that overlap on the GPU (two streams, or two host threads on one device) RACE on the array: keep them on
 *     one stream per device or order them with events.  Calls on different devices do not interact.
 *   - The first call on a device looks up the array's address (cudaGetSymbolAddress) and, like any first launch, loads the
 *     kernels; make that call outside stream capture.  Later calls only enqueue work on `cuda_stream`.
 * Errors: those of carve_fwd / carve_bwd, plus CARVE_ERR_STATIC_LIMIT.
 */
#define CARVE_STATIC_SCRATCH_BYTES (16u << 20)
size_t carve_static_scratch_bytes(void);
carve_status_t carve_fwd_bwd_static(const carve_params_t *p, const void *q, const void *k, const void *v, const void *f,
                                    const void *bx, const void *wx, const void *beta, const float *A, const float *tau,
                                    const float *Ub, const float *Uw, const float *Vb, const float *Vw, const float *S0,
                                    void *O, float *S_final, const void *dO, const float *dS_final, void *dq, void *dk,
                                    void *dv, void *df, void *dbx, void *dwx, void *dbeta, float *dA, float *dtau,
                                    float *dUb, float *dUw, float *dVb, float *dVw, float *dS0, void *cuda_stream);

/* Number of kernel launches carve_fwd / carve_bwd enqueue for these parameters (for accounting). */
int carve_num_launches(const carve_params_t *p, int bwd);

/* Which kernel family (CARVE_PATH_SIMT / CARVE_PATH_TENSOR) the parameters resolve to, or -1. */
int carve_resolved_path(const carve_params_t *p, int bwd);

const char *carve_status_string(carve_status_t s);
const char *carve_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CARVE_H_ */

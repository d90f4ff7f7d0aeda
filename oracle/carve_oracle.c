/*
 * carve_oracle.c -- fp64 CPU oracle for the CARVE layer operator.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_2606_27229_b200/ and neither side includes the other.
 *
 * What it computes: the chunk-parallel key-axis-gated delta-rule operator of
 * PAPER.md (arxiv/paper_2606_27229), written out step by step in the paper's order
 * and notation, in double precision, with plain loops:
 *
 *   carve_ref_fwd            chunked definition, Alg. 1 calling
 *                            Alg. 2 WYCHUNKDELTA (l.315-365), gates from Eq. 7-9
 *                            (l.134-151), retention Eq. 14 (l.310), coupling matrix
 *                            Eq. 15 (l.342).
 *   carve_ref_fwd_sequential the same function written as the per-token recurrence
 *                            Eq. 5 (l.108) with the gates still read from the
 *                            chunk-boundary state (Eq. 7, l.134-136).
 *   carve_ref_bwd            per-token reverse-scan adjoint, Alg. 4 (l.788-817), with
 *                            the chunk-boundary glue of Alg. 5 (l.844-848).
 *
 * Readings of the paper taken here (DESIGN.md section "Readings" lists them; the
 * labels A1..A13 are SURVEY.md 8(c)'s):
 *   A1  the value-axis write gate multiplies v only (Alg. 2 step 5, l.335):
 *       e_t = w_t.v_t - S_{t-1} k_t.
 *   A2  a per-token scalar write strength beta_t (north_star; GDN's, l.90) scales the
 *       whole error: u_t = beta_t e_t.  beta == 1 is Alg. 2 as printed.
 *   A3  Eq. 5 order: predict from the undecayed S_{t-1}, then decay, then write
 *       undecayed.  Hence A_ts uses gamma_{t-1}/gamma_s, outputs use gamma_t/gamma_s.
 *   A4  Alg. 2 steps 8-9 print no intra-chunk decay factors; the factors Eq. 5
 *       implies are used (the paper asserts chunk == sequential, l.450).
 *   A5  the content term is always computed from the state entering the chunk, also
 *       for chunk 0 (identical when S0 = 0).
 *   A7  the gate reads the L2-normalised, unscaled q.
 *   A8  U_b,U_w,V_b,V_w are shared by all heads and batches.
 *   A9  g = -exp(A) softplus(f + tau), A/tau optional (NULL => 0).
 *   A11 scale multiplies O; eps sits inside the sqrt of the L2 norm.
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): per-token numpy recurrence
 * written separately from Eq. 5; U=V=0 memory-blind recurrence; L=1 exact content
 * gating; closed forms of Thm 3 / Thm 15 / beta=0 / orthogonal keys; dense LU solve;
 * split-call and permutation invariance; Thm 4 and Thm 5 inequalities; central finite
 * differences and torch autograd for every gradient tensor.
 * PARITY UNPINNED: which of the readings A1/A2/A3 the authors' own code implements --
 * the paper prints no operator output that could decide it.
 *
 * Layouts (row-major, innermost contiguous):
 *   q,k,f,bx [B,T,H,dk]   v,wx,O [B,T,H,dv]   beta [B,T,H]   A,tau [H,dk]
 *   Ub,Uw [r,dv]   Vb [dk,r]   Vw [dv,r]   S0,S_final [B,H,dv,dk]
 * All pointers are HOST pointers to doubles.  Return 0 on success, nonzero on a bad
 * argument.  OpenMP runs the independent (batch, head) chains in parallel.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int B, H, T, L, dk, dv, r;
    int qk_l2norm;
    double scale;
    double eps;
} carve_ref_params_t;

static double sigmoid_(double x) { return 1.0 / (1.0 + exp(-x)); }
static double softplus_(double x) { return x > 0.0 ? x + log1p(exp(-x)) : log1p(exp(x)); }

int carve_ref_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- per-chunk scratch ------------------------------------------------------- */
typedef struct {
    int L, dk, dv, r;
    double *qh, *kh;      /* [L,dk]  normalised q, k                (D1) */
    double *qn, *kn;      /* [L]     sqrt(|q|^2+eps), same for k         */
    double *g;            /* [L,dk]  decay log                      (D2) */
    double *G;            /* [2r,dk] folded readout                 (D3) */
    double *tt;           /* [L,2r]  tanh bottleneck                (D4) */
    double *b, *w;        /* [L,dk], [L,dv] gates                   (D4) */
    double *lg;           /* [L,dk]  log gamma_t                    (D5) */
    double *Am;           /* [L,L]   coupling matrix                (D6) */
    double *R, *U;        /* [L,dv]                                 (D7) */
} chunk_ws_t;

static int ws_alloc(chunk_ws_t *w_, int L, int dk, int dv, int r)
{
    w_->L = L; w_->dk = dk; w_->dv = dv; w_->r = r;
    size_t n = (size_t)L * dk * 5 + (size_t)L * 2 + (size_t)2 * r * dk + (size_t)L * 2 * r +
               (size_t)L * dv * 3 + (size_t)L * L;
    double *p = (double *)calloc(n, sizeof(double));
    if (!p) return 1;
    w_->qh = p; p += (size_t)L * dk;
    w_->kh = p; p += (size_t)L * dk;
    w_->g = p;  p += (size_t)L * dk;
    w_->b = p;  p += (size_t)L * dk;
    w_->lg = p; p += (size_t)L * dk;
    w_->qn = p; p += L;
    w_->kn = p; p += L;
    w_->G = p;  p += (size_t)2 * r * dk;
    w_->tt = p; p += (size_t)L * 2 * r;
    w_->w = p;  p += (size_t)L * dv;
    w_->R = p;  p += (size_t)L * dv;
    w_->U = p;  p += (size_t)L * dv;
    w_->Am = p;
    return 0;
}
static void ws_free(chunk_ws_t *w_) { free(w_->qh); }

/* Token (b, t, h) of a [B,T,H,d] tensor. */
static const double *tok(const double *x, const carve_ref_params_t *p, int b, int t, int h, int d)
{
    return x + (((size_t)b * p->T + t) * p->H + h) * d;
}
static double *tokw(double *x, const carve_ref_params_t *p, int b, int t, int h, int d)
{
    return x + (((size_t)b * p->T + t) * p->H + h) * d;
}

/*
 * D1-D5 for the chunk of (b,h) starting at token t0, given the state S entering it.
 * Fills qh,kh,qn,kn,g,G,tt,b,w,lg.
 */
static void chunk_gates(const carve_ref_params_t *p, int b, int h, int t0, const double *S,
                        const double *q, const double *k, const double *f, const double *bx,
                        const double *wx, const double *Adec, const double *tau,
                        const double *Ub, const double *Uw, const double *Vb, const double *Vw,
                        chunk_ws_t *c)
{
    const int L = p->L, dk = p->dk, dv = p->dv, r = p->r;
    /* D1: L2 normalisation of q and k per token (Fig. 2 l.437; Alg. 3 step 3 l.399). */
    for (int t = 0; t < L; ++t) {
        const double *qt = tok(q, p, b, t0 + t, h, dk), *kt = tok(k, p, b, t0 + t, h, dk);
        double sq = 0.0, sk = 0.0;
        for (int j = 0; j < dk; ++j) { sq += qt[j] * qt[j]; sk += kt[j] * kt[j]; }
        c->qn[t] = p->qk_l2norm ? sqrt(sq + p->eps) : 1.0;
        c->kn[t] = p->qk_l2norm ? sqrt(sk + p->eps) : 1.0;
        for (int j = 0; j < dk; ++j) {
            c->qh[t * dk + j] = qt[j] / c->qn[t];
            c->kh[t * dk + j] = kt[j] / c->kn[t];
        }
    }
    /* D2: g_t = -exp(A) . softplus(f_t + tau)  (Eq. 9 l.151). */
    for (int t = 0; t < L; ++t) {
        const double *ft = tok(f, p, b, t0 + t, h, dk);
        for (int j = 0; j < dk; ++j) {
            double a = Adec ? Adec[h * dk + j] : 0.0, ta = tau ? tau[h * dk + j] : 0.0;
            c->g[t * dk + j] = -exp(a) * softplus_(ft[j] + ta);
        }
    }
    /* D3: G = [U_b; U_w] S  in R^{2r x dk}  (Eq. 7 l.134), once per chunk. */
    for (int i = 0; i < 2 * r; ++i) {
        const double *Urow = (i < r) ? Ub + (size_t)i * dv : Uw + (size_t)(i - r) * dv;
        for (int j = 0; j < dk; ++j) {
            double s = 0.0;
            for (int v = 0; v < dv; ++v) s += Urow[v] * S[(size_t)v * dk + j];
            c->G[i * dk + j] = s;
        }
    }
    /* D4: t_t = tanh(G q_t); b_t = sigma(b_x + V_b t^(b)); w_t = sigma(w_x + V_w t^(w))
     * (Eq. 7-8 l.134-140). */
    for (int t = 0; t < L; ++t) {
        for (int i = 0; i < 2 * r; ++i) {
            double s = 0.0;
            for (int j = 0; j < dk; ++j) s += c->G[i * dk + j] * c->qh[t * dk + j];
            c->tt[t * 2 * r + i] = tanh(s);
        }
        const double *bxt = tok(bx, p, b, t0 + t, h, dk), *wxt = tok(wx, p, b, t0 + t, h, dv);
        for (int j = 0; j < dk; ++j) {
            double s = bxt[j];
            for (int i = 0; i < r; ++i) s += Vb[(size_t)j * r + i] * c->tt[t * 2 * r + i];
            c->b[t * dk + j] = sigmoid_(s);
        }
        for (int v = 0; v < dv; ++v) {
            double s = wxt[v];
            for (int i = 0; i < r; ++i) s += Vw[(size_t)v * r + i] * c->tt[t * 2 * r + r + i];
            c->w[t * dv + v] = sigmoid_(s);
        }
    }
    /* D5: a_t = exp(g_t).(1-b_t); log gamma_t = sum_{s<=t} log a_s  (Eq. 14 l.310). */
    for (int j = 0; j < dk; ++j) {
        double acc = 0.0;
        for (int t = 0; t < L; ++t) {
            acc += c->g[t * dk + j] + log1p(-c->b[t * dk + j]);
            c->lg[t * dk + j] = acc;
        }
    }
}

/* log gamma_{t} with gamma_{-1} = 1. */
static double lgam(const chunk_ws_t *c, int t, int j) { return t < 0 ? 0.0 : c->lg[t * c->dk + j]; }

/*
 * carve_ref_fwd -- chunked definition (Alg. 1 + Alg. 2).
 */
int carve_ref_fwd(const carve_ref_params_t *p, const double *q, const double *k, const double *v,
                  const double *f, const double *bx, const double *wx, const double *beta,
                  const double *Adec, const double *tau, const double *Ub, const double *Uw,
                  const double *Vb, const double *Vw, const double *S0, double *O, double *S_final)
{
    if (!p || !q || !k || !v || !f || !bx || !wx || !beta || !Ub || !Uw || !Vb || !Vw || !O || !S_final)
        return 1;
    if (p->L <= 0 || p->T % p->L != 0 || p->B <= 0 || p->H <= 0 || p->dk <= 0 || p->dv <= 0 || p->r <= 0)
        return 2;
    const int L = p->L, dk = p->dk, dv = p->dv, n = p->T / p->L;
    int err = 0;
#pragma omp parallel for schedule(dynamic) reduction(| : err)
    for (int bh = 0; bh < p->B * p->H; ++bh) {
        const int b = bh / p->H, h = bh % p->H;
        chunk_ws_t c;
        double *S = (double *)malloc(sizeof(double) * dv * dk);
        double *Sn = (double *)malloc(sizeof(double) * dv * dk);
        if (!S || !Sn || ws_alloc(&c, L, dk, dv, p->r)) { err |= 1; free(S); free(Sn); continue; }
        for (int i = 0; i < dv * dk; ++i) S[i] = S0 ? S0[(size_t)bh * dv * dk + i] : 0.0;
        for (int ci = 0; ci < n; ++ci) {
            const int t0 = ci * L;
            chunk_gates(p, b, h, t0, S, q, k, f, bx, wx, Adec, tau, Ub, Uw, Vb, Vw, &c);
            /* Alg. 2 step 5: r_t = w_t.v_t - S_prev (gamma_{t-1} . k_t)   (l.335). */
            for (int t = 0; t < L; ++t) {
                const double *vt = tok(v, p, b, t0 + t, h, dv);
                for (int x = 0; x < dv; ++x) {
                    double s = 0.0;
                    for (int j = 0; j < dk; ++j)
                        s += S[(size_t)x * dk + j] * exp(lgam(&c, t - 1, j)) * c.kh[t * dk + j];
                    c.R[t * dv + x] = c.w[t * dv + x] * vt[x] - s;
                }
            }
            /* Alg. 2 step 6 / Eq. 15 with the Eq. 5 indices (A3):
             * A_ts = sum_j k_t[j] k_s[j] gamma_{t-1}[j]/gamma_s[j], s < t. */
            for (int t = 0; t < L; ++t)
                for (int s = 0; s < L; ++s) {
                    double a = 0.0;
                    if (s < t)
                        for (int j = 0; j < dk; ++j)
                            a += c.kh[t * dk + j] * c.kh[s * dk + j] *
                                 exp(lgam(&c, t - 1, j) - lgam(&c, s, j));
                    c.Am[t * L + s] = a;
                }
            /* Alg. 2 step 7: forward substitution on (I + diag(beta) A) U = diag(beta) R. */
            for (int t = 0; t < L; ++t) {
                const double bt = *tok(beta, p, b, t0 + t, h, 1);
                for (int x = 0; x < dv; ++x) {
                    double s = c.R[t * dv + x];
                    for (int s_ = 0; s_ < t; ++s_) s -= c.Am[t * L + s_] * c.U[s_ * dv + x];
                    c.U[t * dv + x] = bt * s;
                }
            }
            /* Alg. 2 step 8 (with A4): o_t = scale [ S_prev (gamma_t . q_t)
             *   + sum_{s<=t} u_s sum_j q_t[j] k_s[j] gamma_t[j]/gamma_s[j] ]. */
            for (int t = 0; t < L; ++t) {
                double *ot = tokw(O, p, b, t0 + t, h, dv);
                for (int x = 0; x < dv; ++x) {
                    double s = 0.0;
                    for (int j = 0; j < dk; ++j)
                        s += S[(size_t)x * dk + j] * exp(lgam(&c, t, j)) * c.qh[t * dk + j];
                    ot[x] = s;
                }
                for (int s_ = 0; s_ <= t; ++s_) {
                    double pts = 0.0;
                    for (int j = 0; j < dk; ++j)
                        pts += c.qh[t * dk + j] * c.kh[s_ * dk + j] * exp(lgam(&c, t, j) - lgam(&c, s_, j));
                    for (int x = 0; x < dv; ++x) ot[x] += pts * c.U[s_ * dv + x];
                }
                for (int x = 0; x < dv; ++x) ot[x] *= p->scale;
            }
            /* Alg. 2 step 9 (with A4): S_next = S_prev diag(gamma_{L-1})
             *   + sum_t u_t (k_t . gamma_{L-1}/gamma_t)^T. */
            for (int x = 0; x < dv; ++x)
                for (int j = 0; j < dk; ++j) {
                    double s = S[(size_t)x * dk + j] * exp(lgam(&c, L - 1, j));
                    for (int t = 0; t < L; ++t)
                        s += c.U[t * dv + x] * c.kh[t * dk + j] * exp(lgam(&c, L - 1, j) - lgam(&c, t, j));
                    Sn[(size_t)x * dk + j] = s;
                }
            memcpy(S, Sn, sizeof(double) * dv * dk);
        }
        memcpy(S_final + (size_t)bh * dv * dk, S, sizeof(double) * dv * dk);
        ws_free(&c); free(S); free(Sn);
    }
    return err;
}

/*
 * One token of Eq. 5 (l.108) under readings A1-A3:
 *   e = w.v - S k;  u = beta e;  S <- S diag(a) + u k^T;  o = scale S q.
 * If e_out/u_out are non-NULL the error and the write are returned.
 */
static void token_step(int dk, int dv, double *S, const double *a, const double *kh, const double *qh,
                       const double *w, const double *v, double beta, double scale, double *o,
                       double *e_out, double *u_out)
{
    for (int x = 0; x < dv; ++x) {
        double pred = 0.0;
        for (int j = 0; j < dk; ++j) pred += S[(size_t)x * dk + j] * kh[j];
        double e = w[x] * v[x] - pred, u = beta * e;
        if (e_out) e_out[x] = e;
        if (u_out) u_out[x] = u;
        double out = 0.0;
        for (int j = 0; j < dk; ++j) {
            double s = S[(size_t)x * dk + j] * a[j] + u * kh[j];
            S[(size_t)x * dk + j] = s;
            out += s * qh[j];
        }
        if (o) o[x] = scale * out;
    }
}

/*
 * carve_ref_fwd_sequential -- the same function as carve_ref_fwd, evaluated token by
 * token with Eq. 5; the gates of every token in a chunk are still read from the state
 * at the chunk boundary (Eq. 7 l.134-136, "one chunk stale").
 */
int carve_ref_fwd_sequential(const carve_ref_params_t *p, const double *q, const double *k,
                             const double *v, const double *f, const double *bx, const double *wx,
                             const double *beta, const double *Adec, const double *tau,
                             const double *Ub, const double *Uw, const double *Vb, const double *Vw,
                             const double *S0, double *O, double *S_final)
{
    if (!p || !q || !k || !v || !f || !bx || !wx || !beta || !Ub || !Uw || !Vb || !Vw || !O || !S_final)
        return 1;
    if (p->L <= 0 || p->T % p->L != 0) return 2;
    const int L = p->L, dk = p->dk, dv = p->dv, n = p->T / p->L;
    int err = 0;
#pragma omp parallel for schedule(dynamic) reduction(| : err)
    for (int bh = 0; bh < p->B * p->H; ++bh) {
        const int b = bh / p->H, h = bh % p->H;
        chunk_ws_t c;
        double *S = (double *)malloc(sizeof(double) * dv * dk);
        double *a = (double *)malloc(sizeof(double) * dk);
        if (!S || !a || ws_alloc(&c, L, dk, dv, p->r)) { err |= 1; free(S); free(a); continue; }
        for (int i = 0; i < dv * dk; ++i) S[i] = S0 ? S0[(size_t)bh * dv * dk + i] : 0.0;
        for (int ci = 0; ci < n; ++ci) {
            const int t0 = ci * L;
            chunk_gates(p, b, h, t0, S, q, k, f, bx, wx, Adec, tau, Ub, Uw, Vb, Vw, &c);
            for (int t = 0; t < L; ++t) {
                for (int j = 0; j < dk; ++j) a[j] = exp(c.g[t * dk + j]) * (1.0 - c.b[t * dk + j]);
                token_step(dk, dv, S, a, c.kh + t * dk, c.qh + t * dk, c.w + t * dv,
                           tok(v, p, b, t0 + t, h, dv), *tok(beta, p, b, t0 + t, h, 1), p->scale,
                           tokw(O, p, b, t0 + t, h, dv), NULL, NULL);
            }
        }
        memcpy(S_final + (size_t)bh * dv * dk, S, sizeof(double) * dv * dk);
        ws_free(&c); free(S); free(a);
    }
    return err;
}

/*
 * carve_ref_bwd -- per-token reverse-scan adjoint (Alg. 4 l.788-817) with the
 * chunk-boundary glue of Alg. 5 (l.844-848: dS_{c-1} += [U_b;U_w]^T dG_c and
 * d[U_b;U_w] += dG_c S_{c-1}^T).  Chunk-boundary states are recomputed by a forward
 * sweep (Alg. 4 line 3), then S_{t-1} inside each chunk (Alg. 4 line 6).
 *
 * Inputs as carve_ref_fwd, plus dO [B,T,H,dv] and dS_final [B,H,dv,dk] (NULL => 0).
 * Outputs (overwritten): dq,dk_,df,dbx [B,T,H,dk]; dv_,dwx [B,T,H,dv]; dbeta [B,T,H];
 * dA,dtau [H,dk] (may be NULL to skip); dUb,dUw [r,dv]; dVb [dk,r]; dVw [dv,r];
 * dS0 [B,H,dv,dk].
 */
int carve_ref_bwd(const carve_ref_params_t *p, const double *q, const double *k, const double *v,
                  const double *f, const double *bx, const double *wx, const double *beta,
                  const double *Adec, const double *tau, const double *Ub, const double *Uw,
                  const double *Vb, const double *Vw, const double *S0, const double *dO,
                  const double *dS_final, double *dq, double *dk_, double *dv_, double *df,
                  double *dbx, double *dwx, double *dbeta, double *dA, double *dtau, double *dUb,
                  double *dUw, double *dVb, double *dVw, double *dS0)
{
    if (!p || !q || !k || !v || !f || !bx || !wx || !beta || !Ub || !Uw || !Vb || !Vw || !dO || !dq ||
        !dk_ || !dv_ || !df || !dbx || !dwx || !dbeta || !dUb || !dUw || !dVb || !dVw || !dS0)
        return 1;
    if (p->L <= 0 || p->T % p->L != 0) return 2;
    const int L = p->L, dk = p->dk, dv = p->dv, r = p->r, n = p->T / p->L, H = p->H;
    const size_t sz = (size_t)dv * dk;
    const int nch = p->B * H;
    /* per-chain partial weight gradients, summed in chain order afterwards */
    const size_t wsz = (size_t)2 * r * dv + (size_t)dk * r + (size_t)dv * r + (size_t)2 * dk;
    double *part = (double *)calloc((size_t)nch * wsz, sizeof(double));
    if (!part) return 3;
    int err = 0;
#pragma omp parallel for schedule(dynamic) reduction(| : err)
    for (int bh = 0; bh < nch; ++bh) {
        const int b = bh / H, h = bh % H;
        chunk_ws_t c;
        double *Sb = (double *)malloc(sizeof(double) * sz * (n + 1)); /* chunk-boundary states */
        double *St = (double *)malloc(sizeof(double) * sz * (L + 1)); /* S_{t-1}, t in chunk   */
        double *dS = (double *)malloc(sizeof(double) * sz);
        double *tmp = (double *)malloc(sizeof(double) * (size_t)(6 * dk + 6 * dv + 4 * r) +
                                       sizeof(double) * (size_t)(2 * r * dk + L * dv * 2));
        if (!Sb || !St || !dS || !tmp || ws_alloc(&c, L, dk, dv, r)) {
            err |= 1; free(Sb); free(St); free(dS); free(tmp); continue;
        }
        double *a = tmp, *da = a + dk, *dqh = da + dk, *dkh = dqh + dk, *dbpre = dkh + dk, *dgv = dbpre + dk;
        double *du = dgv + dk, *de = du + dv, *dwpre = de + dv, *dwt = dwpre + dv, *o_unused = dwt + dv,
               *sp = o_unused + dv;
        double *dz = sp + dv, *dtt = dz + 2 * r;
        double *dG = dtt + 2 * r;
        double *Ech = dG + (size_t)2 * r * dk, *Uch = Ech + (size_t)L * dv;
        double *pUb = part + (size_t)bh * wsz, *pUw = pUb + (size_t)r * dv, *pVb = pUw + (size_t)r * dv,
               *pVw = pVb + (size_t)dk * r, *pA = pVw + (size_t)dv * r, *pTau = pA + dk;

        /* Alg. 4 line 3: forward recompute of the chunk-boundary states. */
        for (size_t i = 0; i < sz; ++i) Sb[i] = S0 ? S0[(size_t)bh * sz + i] : 0.0;
        for (int ci = 0; ci < n; ++ci) {
            double *S = Sb + (size_t)(ci + 1) * sz;
            memcpy(S, Sb + (size_t)ci * sz, sizeof(double) * sz);
            chunk_gates(p, b, h, ci * L, Sb + (size_t)ci * sz, q, k, f, bx, wx, Adec, tau, Ub, Uw, Vb, Vw, &c);
            for (int t = 0; t < L; ++t) {
                for (int j = 0; j < dk; ++j) a[j] = exp(c.g[t * dk + j]) * (1.0 - c.b[t * dk + j]);
                token_step(dk, dv, S, a, c.kh + t * dk, c.qh + t * dk, c.w + t * dv,
                           tok(v, p, b, ci * L + t, h, dv), *tok(beta, p, b, ci * L + t, h, 1), p->scale,
                           NULL, NULL, NULL);
            }
        }
        /* Alg. 4 line 4 / Alg. 5 line 4: dS <- dS_final. */
        for (size_t i = 0; i < sz; ++i) dS[i] = dS_final ? dS_final[(size_t)bh * sz + i] : 0.0;

        for (int ci = n - 1; ci >= 0; --ci) {
            const int t0 = ci * L;
            const double *Sc = Sb + (size_t)ci * sz;
            chunk_gates(p, b, h, t0, Sc, q, k, f, bx, wx, Adec, tau, Ub, Uw, Vb, Vw, &c);
            /* recompute S_{t-1} for every t of the chunk, with e_t and u_t */
            memcpy(St, Sc, sizeof(double) * sz);
            for (int t = 0; t < L; ++t) {
                double *Snext = St + (size_t)(t + 1) * sz;
                memcpy(Snext, St + (size_t)t * sz, sizeof(double) * sz);
                for (int j = 0; j < dk; ++j) a[j] = exp(c.g[t * dk + j]) * (1.0 - c.b[t * dk + j]);
                token_step(dk, dv, Snext, a, c.kh + t * dk, c.qh + t * dk, c.w + t * dv,
                           tok(v, p, b, t0 + t, h, dv), *tok(beta, p, b, t0 + t, h, 1), p->scale, NULL,
                           Ech + (size_t)t * dv, Uch + (size_t)t * dv);
            }
            memset(dG, 0, sizeof(double) * 2 * r * dk);
            for (int t = L - 1; t >= 0; --t) {
                const double *Sprev = St + (size_t)t * sz, *Scur = St + (size_t)(t + 1) * sz;
                const double *qh = c.qh + t * dk, *kh = c.kh + t * dk;
                const double *dot = tok(dO, p, b, t0 + t, h, dv), *vt = tok(v, p, b, t0 + t, h, dv);
                const double bt = *tok(beta, p, b, t0 + t, h, 1);
                const double *et = Ech + (size_t)t * dv, *ut = Uch + (size_t)t * dv;
                /* Alg. 4 line 7: dS += do q^T ; dq = S_t^T do */
                for (int j = 0; j < dk; ++j) dqh[j] = 0.0;
                for (int x = 0; x < dv; ++x)
                    for (int j = 0; j < dk; ++j) {
                        dS[(size_t)x * dk + j] += p->scale * dot[x] * qh[j];
                        dqh[j] += p->scale * Scur[(size_t)x * dk + j] * dot[x];
                    }
                /* write path: du = dS k ; dk = dS^T u ; key-axis path: da = colsum(dS . S_{t-1}) */
                for (int j = 0; j < dk; ++j) { dkh[j] = 0.0; da[j] = 0.0; }
                for (int x = 0; x < dv; ++x) {
                    double s = 0.0;
                    for (int j = 0; j < dk; ++j) {
                        s += dS[(size_t)x * dk + j] * kh[j];
                        dkh[j] += dS[(size_t)x * dk + j] * ut[x];
                        da[j] += dS[(size_t)x * dk + j] * Sprev[(size_t)x * dk + j];
                    }
                    du[x] = s;
                }
                /* Alg. 4 line 8: dS_prev = dS diag(exp g) diag(1-b) */
                for (int j = 0; j < dk; ++j) a[j] = exp(c.g[t * dk + j]) * (1.0 - c.b[t * dk + j]);
                for (int x = 0; x < dv; ++x)
                    for (int j = 0; j < dk; ++j) dS[(size_t)x * dk + j] *= a[j];
                /* u = beta e ; e = w.v - S_{t-1} k   (Alg. 4 lines 9-12 under A1/A2; note the
                 * correctness remark l.819: dw = de . v, whereas dv = de . w) */
                double dbt = 0.0;
                for (int x = 0; x < dv; ++x) {
                    de[x] = bt * du[x];
                    dbt += du[x] * et[x];
                    dwt[x] = de[x] * vt[x];
                    tokw(dv_, p, b, t0 + t, h, dv)[x] = de[x] * c.w[t * dv + x];
                }
                *tokw(dbeta, p, b, t0 + t, h, 1) = dbt;
                for (int x = 0; x < dv; ++x)
                    for (int j = 0; j < dk; ++j) {
                        dS[(size_t)x * dk + j] -= de[x] * kh[j];
                        dkh[j] -= Sprev[(size_t)x * dk + j] * de[x];
                    }
                /* Alg. 4 lines 9-10: a = exp(g)(1-b): dg = da a ; db = -da exp(g) */
                const double *ft = tok(f, p, b, t0 + t, h, dk);
                double *dft = tokw(df, p, b, t0 + t, h, dk), *dbxt = tokw(dbx, p, b, t0 + t, h, dk);
                double *dwxt = tokw(dwx, p, b, t0 + t, h, dv);
                for (int j = 0; j < dk; ++j) {
                    double bj = c.b[t * dk + j];
                    dgv[j] = da[j] * a[j];
                    double db = -da[j] * exp(c.g[t * dk + j]);
                    dbpre[j] = db * bj * (1.0 - bj);
                    dbxt[j] = dbpre[j];
                    /* Eq. 9: g = -exp(A) softplus(f+tau) */
                    double A_ = Adec ? Adec[h * dk + j] : 0.0, ta = tau ? tau[h * dk + j] : 0.0;
                    dft[j] = dgv[j] * (-exp(A_)) * sigmoid_(ft[j] + ta);
                    pTau[j] += dft[j];
                    pA[j] += dgv[j] * c.g[t * dk + j];
                }
                for (int x = 0; x < dv; ++x) {
                    double wv = c.w[t * dv + x];
                    dwpre[x] = dwt[x] * wv * (1.0 - wv);
                    dwxt[x] = dwpre[x];
                }
                /* Eq. 8 up-projections and Eq. 7 bottleneck */
                const double *tt = c.tt + (size_t)t * 2 * r;
                for (int i = 0; i < r; ++i) {
                    double sb = 0.0, sw = 0.0;
                    for (int j = 0; j < dk; ++j) {
                        sb += Vb[(size_t)j * r + i] * dbpre[j];
                        pVb[(size_t)j * r + i] += dbpre[j] * tt[i];
                    }
                    for (int x = 0; x < dv; ++x) {
                        sw += Vw[(size_t)x * r + i] * dwpre[x];
                        pVw[(size_t)x * r + i] += dwpre[x] * tt[r + i];
                    }
                    dtt[i] = sb; dtt[r + i] = sw;
                }
                for (int i = 0; i < 2 * r; ++i) {
                    dz[i] = dtt[i] * (1.0 - tt[i] * tt[i]);
                    for (int j = 0; j < dk; ++j) {
                        dG[i * dk + j] += dz[i] * qh[j];
                        dqh[j] += c.G[i * dk + j] * dz[i];
                    }
                }
                /* D1 backward: x_hat = x / n, n = sqrt(|x|^2 + eps) */
                double *dqt = tokw(dq, p, b, t0 + t, h, dk), *dkt = tokw(dk_, p, b, t0 + t, h, dk);
                if (p->qk_l2norm) {
                    double pq = 0.0, pk = 0.0;
                    for (int j = 0; j < dk; ++j) { pq += qh[j] * dqh[j]; pk += kh[j] * dkh[j]; }
                    for (int j = 0; j < dk; ++j) {
                        dqt[j] = (dqh[j] - qh[j] * pq) / c.qn[t];
                        dkt[j] = (dkh[j] - kh[j] * pk) / c.kn[t];
                    }
                } else {
                    for (int j = 0; j < dk; ++j) { dqt[j] = dqh[j]; dkt[j] = dkh[j]; }
                }
            }
            /* Alg. 5 lines 8-9: fold glue at the chunk start, G = [U_b;U_w] S_{c-1}. */
            for (int i = 0; i < 2 * r; ++i) {
                const double *Urow = (i < r) ? Ub + (size_t)i * dv : Uw + (size_t)(i - r) * dv;
                double *pU = (i < r) ? pUb + (size_t)i * dv : pUw + (size_t)(i - r) * dv;
                for (int x = 0; x < dv; ++x) {
                    double s = 0.0;
                    for (int j = 0; j < dk; ++j) {
                        s += dG[i * dk + j] * Sc[(size_t)x * dk + j];
                        dS[(size_t)x * dk + j] += Urow[x] * dG[i * dk + j];
                    }
                    pU[x] += s;
                }
            }
        }
        memcpy(dS0 + (size_t)bh * sz, dS, sizeof(double) * sz);
        ws_free(&c); free(Sb); free(St); free(dS); free(tmp);
    }
    /* Alg. 4 line 16: reduce the weight gradients over batch and heads. */
    memset(dUb, 0, sizeof(double) * r * dv); memset(dUw, 0, sizeof(double) * r * dv);
    memset(dVb, 0, sizeof(double) * dk * r); memset(dVw, 0, sizeof(double) * dv * r);
    if (dA) memset(dA, 0, sizeof(double) * H * dk);
    if (dtau) memset(dtau, 0, sizeof(double) * H * dk);
    for (int bh = 0; bh < nch; ++bh) {
        const int h = bh % H;
        const double *pUb = part + (size_t)bh * wsz, *pUw = pUb + (size_t)r * dv, *pVb = pUw + (size_t)r * dv,
                     *pVw = pVb + (size_t)dk * r, *pA = pVw + (size_t)dv * r, *pTau = pA + dk;
        for (int i = 0; i < r * dv; ++i) { dUb[i] += pUb[i]; dUw[i] += pUw[i]; }
        for (int i = 0; i < dk * r; ++i) dVb[i] += pVb[i];
        for (int i = 0; i < dv * r; ++i) dVw[i] += pVw[i];
        for (int j = 0; j < dk; ++j) {
            if (dA) dA[h * dk + j] += pA[j];
            if (dtau) dtau[h * dk + j] += pTau[j];
        }
    }
    free(part);
    return err;
}

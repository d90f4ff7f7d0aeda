"""Pins for the fp64 oracle (no GPU).  Each test fixes a part of oracle/carve_oracle.c against
something other than itself; the docstrings name the passage of PAPER.md being pinned.
"""
import numpy as np
import pytest

from paper_2606_27229_b200 import synth
from tests import ref_np


def rel(a, b):
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


def small_cfg(**kw):
    base = dict(name="t", B=2, H=2, T=32, L=8, dk=6, dv=5, r=3, dtype="f32", wstd=0.5, s0_std=0.3, seed=3)
    base.update(kw)
    return synth.Config(**base)


def shape_of(oracle, cfg, **kw):
    d = dict(B=cfg.B, H=cfg.H, T=cfg.T, L=cfg.L, dk=cfg.dk, dv=cfg.dv, r=cfg.r,
             qk_l2norm=cfg.qk_l2norm, scale=cfg.scale, eps=cfg.eps)
    d.update(kw)
    return oracle.Shape(**d)


def perturbed(cfg, **kw):
    """Inputs with un-normalised q,k so that the L2-norm step actually does something."""
    x = synth.make_inputs(cfg, **kw)
    rng = np.random.default_rng(11)
    x["q"] = x["q"] * rng.uniform(0.5, 2.0, size=x["q"].shape[:-1] + (1,)).astype(np.float32)
    x["k"] = x["k"] * rng.uniform(0.5, 2.0, size=x["k"].shape[:-1] + (1,)).astype(np.float32)
    return x


# ---------------------------------------------------------------- P1 / P3
@pytest.mark.parametrize("L", [1, 2, 8, 16, 64])
def test_chunked_equals_per_token_recurrence(oracle, L):
    """P1 (Table 2 l.450; north_star check 2): Alg. 2's WY chunk solve == Eq. 5 evaluated
    token by token (numpy, written separately) with the same chunk-stale gates."""
    cfg = small_cfg(T=64, L=L, dk=7, dv=5, r=3)
    x = perturbed(cfg, with_decay_params=True)
    s = shape_of(oracle, cfg, scale=0.7)
    O, Sf = oracle.fwd(s, x)
    O2, Sf2 = ref_np.recurrence_content(s, x, L)
    assert rel(O, O2) < 1e-12 and rel(Sf, Sf2) < 1e-12
    O3, Sf3 = oracle.fwd_sequential(s, x)
    assert rel(O3, O2) < 1e-12 and rel(Sf3, Sf2) < 1e-12


def test_L1_is_exact_content_gating(oracle):
    """P3: at L=1 the chunked definition has no staleness: gates read S_{t-1} (l.136)."""
    cfg = small_cfg(T=24, L=1)
    x = perturbed(cfg)
    s = shape_of(oracle, cfg)
    O, Sf = oracle.fwd(s, x)
    O2, Sf2 = ref_np.recurrence_content(s, x, 1)
    assert rel(O, O2) < 1e-12 and rel(Sf, Sf2) < 1e-12
    # and staleness is real: L=8 differs visibly from L=1 with these O(1) content weights
    O8, _ = oracle.fwd(shape_of(oracle, cfg, L=8), x)
    assert rel(O8, O) > 1e-4


def test_dense_lu_solve(oracle):
    """P5: forward substitution (Alg. 2 step 7 l.348-352) == dense LU on (I+diag(beta)A),
    with A and the outputs built by broadcasting in numpy."""
    cfg = small_cfg(T=48, L=16, dk=8, dv=6, r=2)
    x = perturbed(cfg, with_decay_params=True)
    s = shape_of(oracle, cfg)
    O, Sf = oracle.fwd(s, x)
    O2, Sf2 = ref_np.chunk_dense_solve(s, x)
    assert rel(O, O2) < 1e-11 and rel(Sf, Sf2) < 1e-11


# ---------------------------------------------------------------- P2
def test_zero_content_is_memory_blind_baseline(oracle):
    """P2 (l.143, Table 2 l.451): with zero content projections CARVE is the memory-blind
    key-axis recurrence; compared with a recurrence that contains no gate-fold code."""
    cfg = small_cfg(T=40, L=8)
    x0 = perturbed(cfg, zero_content=True)
    s = shape_of(oracle, cfg)
    O0, S0f = oracle.fwd(s, x0)
    Ob, Sb = ref_np.recurrence_memory_blind(s, x0)
    assert rel(O0, Ob) < 1e-12 and rel(S0f, Sb) < 1e-12
    # bit-identical inside the oracle whenever either projection is zero (l.143 "bit-identical")
    x = perturbed(cfg)
    for zero in (("Vb", "Vw"), ("Ub", "Uw")):
        xz = dict(x)
        for n in zero:
            xz[n] = np.zeros_like(x[n])
        Oz, Sz = oracle.fwd(s, xz)
        assert np.array_equal(Oz, O0) and np.array_equal(Sz, S0f)
    # and the chunk length is irrelevant without content gates
    O1, S1 = oracle.fwd(shape_of(oracle, cfg, L=1), x0)
    assert rel(O1, O0) < 1e-12


def test_zero_content_grads(oracle):
    """P2: U=V=0 => content-parameter gradients exactly 0; V=0, U!=0 => dV != 0, dU == 0."""
    cfg = small_cfg(T=16, L=4)
    s = shape_of(oracle, cfg)
    ct = synth.make_cotangents(cfg)
    x0 = perturbed(cfg, zero_content=True)
    g0 = oracle.bwd(s, x0, ct["dO"], ct["dS_final"])
    for n in ("dUb", "dUw", "dVb", "dVw"):
        assert np.all(g0[n] == 0.0)
    x = perturbed(cfg)
    xv = dict(x, Vb=np.zeros_like(x["Vb"]), Vw=np.zeros_like(x["Vw"]))
    gv = oracle.bwd(s, xv, ct["dO"], ct["dS_final"])
    assert np.all(gv["dUb"] == 0.0) and np.all(gv["dUw"] == 0.0)
    assert np.abs(gv["dVb"]).max() > 0 and np.abs(gv["dVw"]).max() > 0


# ---------------------------------------------------------------- P3 fold associativity
def test_fold_associativity(oracle):
    """P3 (l.136): (U S) q == U (S q).  The oracle folds (D3); ref_np.recurrence_content
    reads out S q per token and then projects -- agreement of the two at L=T (one chunk,
    nonzero S0) isolates the fold."""
    cfg = small_cfg(T=8, L=8, s0_std=1.0)
    x = perturbed(cfg)
    s = shape_of(oracle, cfg)
    O, _ = oracle.fwd(s, x)
    O2, _ = ref_np.recurrence_content(s, x, 8)
    assert rel(O, O2) < 1e-13


# ---------------------------------------------------------------- P4 closed forms
def _blank(B, H, T, dk, dv, r):
    z = lambda *sh: np.zeros(sh)
    return dict(q=z(B, T, H, dk), k=z(B, T, H, dk), v=z(B, T, H, dv), f=z(B, T, H, dk) - 40.0,
                bx=z(B, T, H, dk) - 40.0, wx=z(B, T, H, dv) + 40.0, beta=np.ones((B, T, H)),
                A=None, tau=None, Ub=z(r, dv), Uw=z(r, dv), Vb=z(dk, r), Vw=z(dv, r), S0=None)


def test_capacity_orthonormal_keys(oracle):
    """P4(i) Thm 3 (l.224): orthonormal keys, no decay/erase, beta=w=1, S0=0 =>
    S_T = sum_i v_i k_i^T exactly after n* = min(dv,dk) writes, and S_T k_i = v_i."""
    dk, dv, T = 6, 6, 6
    rng = np.random.default_rng(0)
    Q, _ = np.linalg.qr(rng.standard_normal((dk, dk)))
    x = _blank(1, 1, T, dk, dv, 2)
    x["k"][0, :, 0] = Q[:, :T].T
    x["q"][0, :, 0] = Q[:, :T].T
    x["v"][0, :, 0] = rng.standard_normal((T, dv))
    s = oracle.Shape(B=1, H=1, T=T, L=3, dk=dk, dv=dv, r=2, qk_l2norm=0, eps=0.0)
    O, Sf = oracle.fwd(s, x)
    want = x["v"][0, :, 0].T @ x["k"][0, :, 0]
    assert np.abs(Sf[0, 0] - want).max() < 1e-12
    assert np.abs(Sf[0, 0] @ Q[:, :T] - x["v"][0, :, 0].T).max() < 1e-12
    # o_t = S_t q_t with q_t = k_t retrieves v_t right after its write
    assert np.abs(O[0, :, 0] - x["v"][0, :, 0]).max() < 1e-12


def test_single_slot_retrieval(oracle):
    """P4(ii) Thm 15 (l.764) under readings A1/A2: one write (k,v) into S0=0, query q=k
    => o = beta (w.v) |k|^2."""
    dk, dv = 5, 4
    rng = np.random.default_rng(1)
    x = _blank(1, 1, 1, dk, dv, 2)
    k = rng.standard_normal(dk)
    v = rng.standard_normal(dv)
    wx = rng.standard_normal(dv)
    x["k"][0, 0, 0] = k
    x["q"][0, 0, 0] = k
    x["v"][0, 0, 0] = v
    x["wx"][0, 0, 0] = wx
    x["beta"][0, 0, 0] = 0.37
    s = oracle.Shape(B=1, H=1, T=1, L=1, dk=dk, dv=dv, r=2, qk_l2norm=0, eps=0.0)
    O, Sf = oracle.fwd(s, x)
    w = 1.0 / (1.0 + np.exp(-wx))
    assert np.abs(O[0, 0, 0] - 0.37 * w * v * (k @ k)).max() < 1e-13
    assert np.abs(Sf[0, 0] - 0.37 * np.outer(w * v, k)).max() < 1e-13


def test_beta_zero_is_pure_decay(oracle):
    """P4(iii): beta=0 => S_t = S0 diag(gamma_t), o_t = scale S0 (gamma_t . q_t)  (Eq. 14)."""
    cfg = small_cfg(T=16, L=4, wstd=0.0)
    x = perturbed(cfg, zero_content=True)
    x["beta"] = np.zeros_like(x["beta"])
    s = shape_of(oracle, cfg, qk_l2norm=0, scale=1.3)
    O, Sf = oracle.fwd(s, x)
    g = -np.logaddexp(0.0, x["f"].astype(np.float64))
    la = g + np.log1p(-1.0 / (1.0 + np.exp(-x["bx"].astype(np.float64))))
    lg = np.cumsum(la, axis=1)                              # [B,T,H,dk]
    S0 = x["S0"].astype(np.float64)
    want = 1.3 * np.einsum("bhvj,bthj->bthv", S0, np.exp(lg) * x["q"])
    assert rel(O, want) < 1e-12
    assert rel(Sf, S0 * np.exp(lg[:, -1])[:, :, None, :]) < 1e-12


def test_orthogonal_keys_linear_attention(oracle):
    """P4(iv) (l.90): mutually orthogonal keys and a=1 => predictions vanish and
    S_T = S0' + sum_t beta_t (w_t.v_t) k_t^T with S0 orthogonal to the keys."""
    dk, dv, T = 8, 3, 5
    rng = np.random.default_rng(2)
    Q, _ = np.linalg.qr(rng.standard_normal((dk, dk)))
    x = _blank(1, 1, T, dk, dv, 2)
    x["k"][0, :, 0] = 1.7 * Q[:, :T].T
    x["q"][0, :, 0] = rng.standard_normal((T, dk))
    x["v"][0, :, 0] = rng.standard_normal((T, dv))
    x["wx"][0, :, 0] = rng.standard_normal((T, dv))
    x["beta"][0, :, 0] = rng.uniform(0.1, 1.0, T)
    S0 = rng.standard_normal((dv, dk)) @ (np.eye(dk) - Q[:, :T] @ Q[:, :T].T)
    x["S0"] = S0[None, None]
    s = oracle.Shape(B=1, H=1, T=T, L=T, dk=dk, dv=dv, r=2, qk_l2norm=0, eps=0.0)
    _, Sf = oracle.fwd(s, x)
    w = 1.0 / (1.0 + np.exp(-x["wx"][0, :, 0]))
    want = S0 + ((x["beta"][0, :, 0, None] * w * x["v"][0, :, 0]).T @ x["k"][0, :, 0])
    assert np.abs(Sf[0, 0] - want).max() < 1e-12


def test_golden_contraction_ratio(oracle):
    """Golden value the paper prints (l.239, l.721): b = 0.05 and exp(g) = 0.95 give the
    joint contraction rho = (0.95)^2 = 0.9025.  With beta = 0 one step multiplies the
    state by exactly rho: pins a = exp(g) (1 - b) (Eq. 5, Eq. 14)."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "rho_carve.txt")
    vals = [ln.split("#")[0].split() for ln in open(path) if ln.strip() and not ln.startswith("#")]
    b_min, eg, rho = (float(v) for v in vals[0])
    dk, dv = 3, 2
    x = _blank(1, 1, 2, dk, dv, 1)
    # softplus(f) = -log(eg)  =>  f = log(exp(-log eg) - 1) ;  sigma(bx) = b_min
    x["f"][:] = np.log(np.expm1(-np.log(eg)))
    x["bx"][:] = np.log(b_min / (1 - b_min))
    x["beta"][:] = 0.0
    S0 = np.arange(1, dv * dk + 1, dtype=np.float64).reshape(1, 1, dv, dk)
    x["S0"] = S0
    s = oracle.Shape(B=1, H=1, T=2, L=1, dk=dk, dv=dv, r=1, qk_l2norm=0, eps=0.0)
    _, Sf = oracle.fwd(s, x)
    assert abs(rho - 0.9025) < 1e-15
    assert np.abs(Sf - rho * rho * S0).max() < 1e-13


# ---------------------------------------------------------------- P6 call structure
def test_split_call_and_permutation(oracle):
    """P6 (Table 2 l.452): one call over T == two calls over T/2 with S_final -> S0;
    permuting (b,h) permutes the outputs."""
    cfg = small_cfg(T=32, L=8)
    x = perturbed(cfg)
    s = shape_of(oracle, cfg)
    O, Sf = oracle.fwd(s, x)
    half = shape_of(oracle, cfg, T=16)
    xa = {n: (a[:, :16] if n in synth.TOKEN_TENSORS else a) for n, a in x.items()}
    xb = {n: (a[:, 16:] if n in synth.TOKEN_TENSORS else a) for n, a in x.items()}
    Oa, Sa = oracle.fwd(half, xa)
    xb["S0"] = Sa
    Ob, Sb = oracle.fwd(half, xb)
    assert np.array_equal(np.concatenate([Oa, Ob], axis=1), O) and np.array_equal(Sb, Sf)
    xp = {n: (a[::-1, :, ::-1] if n in synth.TOKEN_TENSORS else a) for n, a in x.items()}
    xp["S0"] = x["S0"][::-1, ::-1]
    Op, Sp = oracle.fwd(s, xp)
    assert np.array_equal(Op[::-1, :, ::-1], O) and np.array_equal(Sp[::-1, ::-1], Sf)


# ---------------------------------------------------------------- P7 inequalities
def test_lyapunov_bound(oracle):
    """P7 Thm 4 (l.234): |S_t|_F <= rho^t |S0|_F + M/(1-rho) with rho = max_t,j a_t[j] and
    M = max_t |u_t k_t^T|_F, both measured by stepping the oracle one token at a time
    (content projections zero, so a_t is known from the inputs alone)."""
    cfg = small_cfg(B=1, H=1, T=48, L=1, dk=6, dv=5, s0_std=2.0)
    x = perturbed(cfg, zero_content=True)
    one = shape_of(oracle, cfg, T=1)
    g = -np.logaddexp(0.0, x["f"].astype(np.float64))
    a = np.exp(g) * (1 - 1 / (1 + np.exp(-x["bx"].astype(np.float64))))      # [B,T,H,dk]
    rho = float(a.max())
    S = x["S0"].astype(np.float64)
    n0, M, norms = np.linalg.norm(S), 0.0, []
    for t in range(cfg.T):
        xt = {n: (v[:, t:t + 1] if n in synth.TOKEN_TENSORS else v) for n, v in x.items()}
        xt["S0"] = S
        _, Sn = oracle.fwd(one, xt)
        M = max(M, np.linalg.norm(Sn - S * a[:, t][:, :, None, :]))
        S = Sn
        norms.append(np.linalg.norm(S))
    assert rho < 1.0
    for t, nrm in enumerate(norms, start=1):
        assert nrm <= rho ** t * n0 + M / (1 - rho) + 1e-12
    # and the full call reproduces the stepped state (carried-state interface, l.452)
    _, Sfull = oracle.fwd(shape_of(oracle, cfg), x)
    assert rel(Sfull, S) < 1e-13


def test_gradient_flow_bound(oracle):
    """P7 Thm 5 (l.249): with only dS_final seeded, U=V=0 and beta=0 (homogeneous path),
    |dS0|_F <= |dS_T|_F prod_t rho_t, rho_t = max_j a_t[j]; equality structure
    dS0 = dS_T diag(gamma_T)."""
    cfg = small_cfg(B=1, H=1, T=16, L=4)
    x = perturbed(cfg, zero_content=True)
    x["beta"] = np.zeros_like(x["beta"])
    s = shape_of(oracle, cfg)
    ct = synth.make_cotangents(cfg)
    g_ = oracle.bwd(s, x, np.zeros_like(ct["dO"]), ct["dS_final"])
    g = -np.logaddexp(0.0, x["f"].astype(np.float64))
    a = np.exp(g) * (1 - 1 / (1 + np.exp(-x["bx"].astype(np.float64))))
    prod_rho = np.prod(a.max(-1))
    assert np.linalg.norm(g_["dS0"]) <= np.linalg.norm(ct["dS_final"]) * prod_rho + 1e-15
    want = ct["dS_final"].astype(np.float64) * np.prod(a, axis=1)[:, :, None, :]
    assert rel(g_["dS0"], want) < 1e-12

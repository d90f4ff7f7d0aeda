"""GPU parity: the CUDA path (through the C ABI) vs the fp64 oracle, element by element, on the
same seeded inputs.  Tolerances are north_star's: max|x-ref|/max|ref| <= 1e-4 for fp32 inputs;
<= 2e-2 on O (and S_final) and <= 3e-2 on every gradient for bf16 inputs with fp32 state.
"""
import numpy as np
import pytest

from paper_2606_27229_b200 import carve, synth
from tests.gpu_util import GRADS, oracle_shape, params_of, relerr, run_bwd, run_fwd

pytestmark = pytest.mark.gpu

TOL = {"f32": dict(O=1e-4, S=1e-4, g=1e-4), "bf16": dict(O=2e-2, S=2e-2, g=3e-2)}


def _check_fwd_bwd(oracle, cfg, x, with_bwd=True, path=carve.CARVE_PATH_AUTO, ct=None, tol=None):
    p = params_of(cfg, path=path)
    s = oracle_shape(oracle, cfg)
    O_ref, S_ref = oracle.fwd(s, x)
    O, Sf, handles = run_fwd(p, x, need_bwd=with_bwd)
    tol = tol or TOL[cfg.dtype]
    errs = {"O": relerr(O, O_ref), "S_final": relerr(Sf, S_ref)}
    assert np.isfinite(O).all() and np.isfinite(Sf).all()
    assert errs["O"] <= tol["O"], errs
    assert errs["S_final"] <= tol["S"], errs
    if with_bwd:
        ct = ct or synth.make_cotangents(cfg)
        g_ref = oracle.bwd(s, x, ct["dO"], ct["dS_final"])
        g, _ = run_bwd(p, handles, ct)
        for n in GRADS:
            if x.get(n[1:]) is None and n in ("dA", "dtau"):
                pass  # gradients w.r.t. absent A/tau are still defined (they default to 0)
            assert np.isfinite(g[n]).all(), n
            errs[n] = relerr(g[n], g_ref[n])
            assert errs[n] <= tol.get(n, tol["g"]), (n, errs)
    return errs


# ---- config 0 of BASELINE.json, exactly, plus its U=0 run --------------------------------------
@pytest.mark.parametrize("zero_content", [False, True])
@pytest.mark.parametrize("l2norm", [1, 0])
def test_config0_fp32(oracle, zero_content, l2norm):
    cfg = synth.CFG0.with_(qk_l2norm=l2norm)
    x = synth.make_inputs(cfg, zero_content=zero_content)
    _check_fwd_bwd(oracle, cfg, x)


@pytest.mark.parametrize("l2norm", [1, 0])
def test_config0_fp32_unnormalised_qk(oracle, l2norm):
    """Config 0 with every q, k row rescaled by U(0.5, 2): row a0 (Fig. 2 l.437, Alg. 3 step 3 l.399) on the fp32 path,
    forward (rsqrt scale) and backward (dq = (dq^ - q^<q^,dq^>)/|q|), with and without the in-kernel normalisation."""
    cfg = synth.CFG0.with_(qk_l2norm=l2norm, wstd=0.1)
    x = synth.scale_qk_rows(synth.make_inputs(cfg), cfg)
    _check_fwd_bwd(oracle, cfg, x)


# ---- small cases spanning several sub-chunks, every chunk length, ragged structure -------------
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("L", [16, 32, 64, 128])
def test_chunk_lengths(oracle, dtype, L):
    cfg = synth.Config("t", B=2, H=2, T=256, L=L, dk=64, dv=64, r=8, dtype=dtype, wstd=0.1, s0_std=0.05, seed=L)
    x = synth.make_inputs(cfg, with_decay_params=True)
    _check_fwd_bwd(oracle, cfg, x)


@pytest.mark.parametrize("dk,dv,r", [(128, 128, 16), (64, 128, 8), (128, 64, 32), (64, 256, 16)])
def test_head_dims_bf16(oracle, dk, dv, r):
    cfg = synth.Config("t", B=1, H=3, T=128, L=32, dk=dk, dv=dv, r=r, dtype="bf16", wstd=0.1, s0_std=0.02, seed=7)
    x = synth.make_inputs(cfg)
    _check_fwd_bwd(oracle, cfg, x)


@pytest.mark.parametrize("dk,dv,r", [(128, 256, 16), (256, 64, 8)])
def test_large_heads_forward_only(oracle, dk, dv, r):
    """dk=128, dv=256 (config 3's head shape; tensor path, value channels split over a two-CTA cluster) and dk=256
    (SIMT) are forward-only: bwd must refuse them, not fall back."""
    cfg = synth.Config("t", B=1, H=2, T=128, L=64, dk=dk, dv=dv, r=r, dtype="bf16", s0_std=0.01, seed=5)
    x = synth.make_inputs(cfg)
    _check_fwd_bwd(oracle, cfg, x, with_bwd=False)
    assert carve.carve_workspace_bytes(params_of(cfg), True) == 0
    assert carve.carve_resolved_path(params_of(cfg), False) == (carve.CARVE_PATH_TENSOR if dv == 256 else carve.CARVE_PATH_SIMT)


def test_single_chunk_and_scale(oracle):
    cfg = synth.Config("t", B=1, H=1, T=16, L=16, dk=64, dv=64, r=8, dtype="f32", wstd=0.3, s0_std=0.5,
                       scale=0.125, seed=2)
    x = synth.make_inputs(cfg, with_decay_params=True)
    _check_fwd_bwd(oracle, cfg, x)


def test_stress_conditioning(oracle):
    """Config 4's stress structure at small size: beta = 1 on 10 % of tokens, no decay on 10 % of key dims."""
    cfg = synth.CFG4.with_(B=2, H=2, T=256)
    x = synth.make_inputs(cfg)
    _check_fwd_bwd(oracle, cfg, x)


def test_extreme_decay_no_overflow(oracle):
    """Strong decay/erase (log gamma_L ~ -600 per chunk, |lg| ~ 150 inside one 16-token sub-chunk): every ratio is formed
    as exp(<= 0), nothing overflows.  Not a BASELINE config.  Tolerances per tensor (measured on
    B200 next to each bound): everything that does not pass through d log a keeps north_star's 1e-4 (measured <= 5e-7,
    dUw and dVw included: the write gate is not fed by d log a).  df and dbx ARE d log a times a local factor: an fp32
    prefix sum of magnitude 150 carries ulp/2 ~ 8e-6 absolute error into every exp(lg_a - lg_b), and d log a sums ~1e2
    such terms of both signs: 5e-4 (measured 2.3e-4, 2.5e-4).  dA, dtau (Eq. 9 l.151) and dUb, dVb (the erase gate's
    projections, fed by db_pre = -d log a . b, Alg. 5 l.846) are sums of those over all T tokens that cancel to ~1/10 of
    their terms: 5e-3 (measured 2.9e-3, 2.2e-3, 1.2e-3, 1.5e-3)."""
    cfg = synth.Config("t", B=1, H=1, T=128, L=64, dk=64, dv=64, r=8, dtype="f32", wstd=0.1, s0_std=0.1, seed=4)
    x = synth.make_inputs(cfg)
    x["f"] = x["f"] + 5.0
    x["bx"] = x["bx"] + 5.0
    errs = _check_fwd_bwd(oracle, cfg, x, tol=dict(O=1e-4, S=1e-4, g=1e-4, df=5e-4, dbx=5e-4, dA=5e-3, dtau=5e-3, dUb=5e-3, dVb=5e-3))
    print("extreme decay, measured:", {n: f"{v:.1e}" for n, v in errs.items()})


# ---- invariants that need no oracle -------------------------------------------------------------
def test_split_call_bitwise(oracle):
    """One call over T == two calls over T/2 with S_final -> S0 (Table 2 l.452), bit for bit."""
    cfg = synth.Config("t", B=2, H=2, T=256, L=64, dk=64, dv=64, r=8, dtype="bf16", wstd=0.1, seed=9)
    x = synth.make_inputs(cfg)
    p = params_of(cfg)
    O, Sf, _ = run_fwd(p, x)
    half = cfg.with_(T=128)
    xa = {n: (a[:, :128] if n in synth.TOKEN_TENSORS else a) for n, a in x.items()}
    xb = {n: (a[:, 128:] if n in synth.TOKEN_TENSORS else a) for n, a in x.items()}
    Oa, Sa, _ = run_fwd(params_of(half), xa)
    xb["S0"] = Sa.astype(np.float32)
    Ob, Sb, _ = run_fwd(params_of(half), xb)
    assert np.array_equal(np.concatenate([Oa, Ob], axis=1), O)
    assert np.array_equal(Sb, Sf)


def test_determinism_and_zero_content_grads(oracle):
    cfg = synth.Config("t", B=2, H=4, T=128, L=32, dk=64, dv=64, r=8, dtype="bf16", seed=12)
    x = synth.make_inputs(cfg, zero_content=True)
    ct = synth.make_cotangents(cfg)
    p = params_of(cfg)
    outs = []
    for _ in range(2):
        O, Sf, h = run_fwd(p, x, need_bwd=True)
        g, _ = run_bwd(p, h, ct)
        outs.append((O, Sf, g))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    for n in GRADS:
        assert np.array_equal(outs[0][2][n], outs[1][2][n]), n
    for n in ("dUb", "dUw", "dVb", "dVw"):
        assert np.all(outs[0][2][n] == 0.0), n


@pytest.mark.parametrize("B", [1, 4, 6])
def test_host_entry_point_matches_device_entry_point(oracle, B):
    """carve_fwd_bwd_host cuts the batch into slices on streams of its own: per-chain results are those of the
    device entry points bit for bit; the shared-weight gradients are the slices' sums (another rounding order)."""
    import torch
    cfg = synth.Config("t", B=B, H=2, T=128, L=64, dk=64, dv=64, r=8, dtype="bf16", wstd=0.1, seed=21)
    x = synth.make_inputs(cfg)
    ct = synth.make_cotangents(cfg)
    p = params_of(cfg)
    O, Sf, h = run_fwd(p, x, need_bwd=True)
    g, _ = run_bwd(p, h, ct)
    from tests.gpu_util import alloc_grads, to_device
    xh = {n: (None if t is None else t.pin_memory()) for n, t in to_device(x, torch.bfloat16, "cpu").items()}
    dOh = to_device({"dO": ct["dO"]}, torch.bfloat16, "cpu")["dO"].pin_memory()
    dSfh = torch.from_numpy(ct["dS_final"]).pin_memory()
    Oh = torch.empty(cfg.B, cfg.T, cfg.H, cfg.dv, dtype=torch.bfloat16).pin_memory()
    Sfh = torch.empty(cfg.B, cfg.H, cfg.dv, cfg.dk, dtype=torch.float32).pin_memory()
    gh = {n: (None if t is None else t.pin_memory()) for n, t in alloc_grads(p, torch.bfloat16, "cpu").items()}
    arena = torch.empty(carve.carve_host_arena_bytes(p, True), dtype=torch.uint8, device="cuda")
    carve.carve_fwd_bwd_host(p, True, xh, Oh, Sfh, dOh, dSfh, gh, arena, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert np.array_equal(Oh.float().numpy().astype(np.float64), O)
    assert np.array_equal(Sfh.numpy().astype(np.float64), Sf)
    for n in GRADS:
        got = gh[n].float().numpy().astype(np.float64)
        if B > 1 and n in ("dA", "dtau", "dUb", "dUw", "dVb", "dVw"):
            assert relerr(got, g[n]) < 1e-5, n
        else:
            assert np.array_equal(got, g[n]), n
    # the same call with caller-owned streams and events (carve_host_ctx_create), twice on one context: identical results
    ctx = carve.carve_host_ctx_create()
    first = {n: gh[n].clone() for n in GRADS}
    for _ in range(2):
        Oh.zero_()
        carve.carve_fwd_bwd_host(p, True, xh, Oh, Sfh, dOh, dSfh, gh, arena, torch.cuda.current_stream().cuda_stream, ctx=ctx)
        torch.cuda.synchronize()
        assert np.array_equal(Oh.float().numpy().astype(np.float64), O)
        for n in GRADS:
            assert torch.equal(gh[n], first[n]), n
    carve.carve_host_ctx_destroy(ctx)


# ---- both kernel families against the oracle on the same bf16 case --------------------------------
@pytest.mark.parametrize("path", [carve.CARVE_PATH_SIMT, carve.CARVE_PATH_TENSOR])
@pytest.mark.parametrize("dk,r,L", [(64, 8, 64), (128, 16, 64), (128, 16, 32), (64, 16, 16), (128, 16, 128), (64, 8, 128)])
def test_kernel_families_bf16(oracle, path, dk, r, L):
    """Several chunks, several 16-token anchor blocks, nonzero S0, active content gates, A and tau present."""
    cfg = synth.Config("t", B=2, H=2, T=256, L=L, dk=dk, dv=dk, r=r, dtype="bf16", wstd=0.1, s0_std=0.05, seed=dk + L)
    x = synth.scale_qk_rows(synth.make_inputs(cfg, with_decay_params=True), cfg)   # un-normalised q, k (row a0)
    p = params_of(cfg, path=path)
    assert carve.carve_resolved_path(p, True) == path
    _check_fwd_bwd(oracle, cfg, x, path=path)


@pytest.mark.parametrize("path", [carve.CARVE_PATH_SIMT, carve.CARVE_PATH_TENSOR])
@pytest.mark.parametrize("sigma", [0.3, 3.0])
@pytest.mark.parametrize("l2norm", [1, 0])
def test_unnormalised_qk_both_paths(oracle, path, sigma, l2norm):
    """q, k rows of norm ~ sigma.U(0.5,2) (and, with the normalisation on, four rows of norm ~ sqrt(eps), where the eps
    inside the square root decides the result): pins the rsqrt(|x|^2 + eps) scale and the 1/|x| factor of its backward
    on both kernel families.  With qk_l2norm = 0 the same rows go in as given (a smaller range, so that the un-normalised
    coupling matrix stays well conditioned)."""
    cfg = synth.Config("t", B=2, H=2, T=128, L=64, dk=64, dv=64, r=8, dtype="bf16", wstd=0.1, s0_std=0.05,
                       qk_l2norm=l2norm, seed=int(10 * sigma) + l2norm)
    if l2norm:
        x = synth.scale_qk_rows(synth.make_inputs(cfg), cfg, 0.5 * sigma, 2.0 * sigma, tiny_rows=4)
    else:
        x = synth.scale_qk_rows(synth.make_inputs(cfg), cfg, 0.6, 1.2)
    _check_fwd_bwd(oracle, cfg, x, path=path)


def test_tensor_path_refuses_what_it_does_not_cover(oracle):
    """No silent substitution: an explicit CARVE_PATH_TENSOR request for fp32 tokens, d_k != d_v or r = 32 is an error."""
    for kw in (dict(dk=64, dv=64, r=8, dtype="f32"), dict(dk=64, dv=128, r=8, dtype="bf16"),
               dict(dk=128, dv=128, r=32, dtype="bf16")):
        cfg = synth.Config("t", B=1, H=1, T=128, L=64, seed=1, **kw)
        p = params_of(cfg, path=carve.CARVE_PATH_TENSOR)
        assert carve.carve_resolved_path(p, True) == -1
        assert carve.carve_workspace_bytes(p, True) == 0


def test_tensor_path_scale_and_no_l2norm(oracle):
    cfg = synth.Config("t", B=1, H=2, T=128, L=64, dk=64, dv=64, r=8, dtype="bf16", wstd=0.1, s0_std=0.05,
                       scale=0.125, qk_l2norm=0, seed=31)
    x = synth.make_inputs(cfg)
    _check_fwd_bwd(oracle, cfg, x, path=carve.CARVE_PATH_TENSOR)


@pytest.mark.parametrize("dk,r,L,scale", [(128, 8, 64, 1.0), (128, 8, 16, 1.0), (128, 16, 64, 0.5), (128, 16, 32, 0.5),
                                          (128, 16, 128, 0.5), (64, 16, 64, 1.0), (64, 8, 64, 0.5), (64, 8, 32, 1.0)])
def test_tensor_path_general_instances(oracle, dk, r, L, scale):
    """The tensor-path kernels compile as specialised instances (full 64-token chunks, the configs' rank r = 16 at
    d = 128 / r = 8 at d = 64, scale = 1, chunk lengths 16 and 32 at d = 128) next to general ones of the same source:
    these cases -- another rank, another scale -- run the general instances, forward + backward."""
    cfg = synth.Config("t", B=1, H=2, T=256, L=L, dk=dk, dv=dk, r=r, dtype="bf16", wstd=0.1, s0_std=0.05, scale=scale,
                       seed=dk + r + L)
    x = synth.scale_qk_rows(synth.make_inputs(cfg, with_decay_params=True), cfg)
    _check_fwd_bwd(oracle, cfg, x, path=carve.CARVE_PATH_TENSOR)


@pytest.mark.parametrize("dk,dv,r,L", [(128, 128, 16, 64), (128, 128, 8, 64), (128, 128, 16, 16), (64, 64, 8, 64), (64, 64, 16, 32),
                                       (128, 256, 16, 64), (128, 256, 8, 32)])
def test_tensor_path_inference_instances(oracle, dk, dv, r, L):
    """Forward without workspace (the inference kernel: no T solve, no record code) in its specialised and general
    instances, including the two-CTA value split at d_v = 256."""
    cfg = synth.Config("t", B=1, H=2, T=256, L=L, dk=dk, dv=dv, r=r, dtype="bf16", wstd=0.1, s0_std=0.05, fwd_only=True,
                       seed=dk + dv + r + L)
    x = synth.scale_qk_rows(synth.make_inputs(cfg, with_decay_params=True), cfg)
    p = params_of(cfg, path=carve.CARVE_PATH_TENSOR)
    assert carve.carve_resolved_path(p, False) == carve.CARVE_PATH_TENSOR
    O, Sf, _ = run_fwd(p, x, need_bwd=False)
    O_ref, S_ref = oracle.fwd(oracle_shape(oracle, cfg), x)
    assert relerr(O, O_ref) <= 2e-2 and relerr(Sf, S_ref) <= 2e-2


def test_tensor_path_determinism(oracle):
    cfg = synth.Config("t", B=2, H=3, T=256, L=64, dk=128, dv=128, r=16, dtype="bf16", wstd=0.1, seed=12)
    x, ct = synth.make_inputs(cfg), synth.make_cotangents(cfg)
    p = params_of(cfg, path=carve.CARVE_PATH_TENSOR)
    outs = []
    for _ in range(2):
        O, Sf, h = run_fwd(p, x, need_bwd=True)
        g, _ = run_bwd(p, h, ct)
        outs.append((O, Sf, g))
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    for n in GRADS:
        assert np.array_equal(outs[0][2][n], outs[1][2][n]), n


# ---- BASELINE.json configs at full size, every tensor of every chain: tests/test_gpu_fullsize.py ------------------
@pytest.mark.parametrize("L", [16, 32, 64, 128])
def test_config2_chunk_sweep_reduced_batch(oracle, L):
    """Config 2 (chunk-length sweep, gate projections ~N(0,0.1^2)) at full T = 8192 with B*H reduced to 2 chains."""
    cfg = synth.CFG2[L].with_(B=1, H=2)
    x = synth.make_inputs(cfg)
    _check_fwd_bwd(oracle, cfg, x)


def test_config4_many_short_reduced_batch(oracle):
    """Config 4's shape and stress structure (beta = 1 on 10 %, no decay on 10 % of key dims) at T = 1024, B*H = 4*4."""
    cfg = synth.CFG4.with_(B=4, H=4)
    x = synth.make_inputs(cfg)
    _check_fwd_bwd(oracle, cfg, x)


def test_config3_long_context_forward_reduced_heads(oracle):
    """Config 3 (forward only, T = 65536, d_v = 256, random S0) with H reduced to 2 chains."""
    cfg = synth.CFG3.with_(H=2)
    x = synth.make_inputs(cfg)
    _check_fwd_bwd(oracle, cfg, x, with_bwd=False)


@pytest.mark.parametrize("B,H,T,L,d,r,seed", [(3, 5, 64, 64, 128, 8, 101), (1, 3, 192, 64, 128, 16, 102), (2, 1, 32, 16, 64, 16, 103),
                                              (1, 7, 384, 128, 128, 16, 104), (5, 2, 96, 32, 64, 8, 105)])
def test_tensor_path_odd_shapes(oracle, B, H, T, L, d, r, seed):
    """Single-chunk sequences, odd batch / head counts, every supported r, nonzero S0, A and tau present."""
    cfg = synth.Config("t", B=B, H=H, T=T, L=L, dk=d, dv=d, r=r, dtype="bf16", wstd=0.1, s0_std=0.05, seed=seed)
    x = synth.scale_qk_rows(synth.make_inputs(cfg, with_decay_params=True), cfg)   # un-normalised q, k (row a0)
    _check_fwd_bwd(oracle, cfg, x, path=carve.CARVE_PATH_TENSOR)


def test_tensor_path_repeated_calls_same_workspace(oracle):
    """Back-to-back fwd/bwd pairs on one stream reuse the workspace and the outputs: results must not change."""
    import torch
    cfg = synth.Config("t", B=2, H=3, T=512, L=64, dk=128, dv=128, r=16, dtype="bf16", wstd=0.1, seed=77)
    x, ct = synth.make_inputs(cfg), synth.make_cotangents(cfg)
    p = params_of(cfg, path=carve.CARVE_PATH_TENSOR)
    O, Sf, h = run_fwd(p, x, need_bwd=True)
    g0, gd = run_bwd(p, h, ct)
    xd, ws = h
    from tests.gpu_util import to_device
    dO = to_device({"dO": ct["dO"]}, torch.bfloat16)["dO"]
    dSf = torch.from_numpy(np.ascontiguousarray(ct["dS_final"], dtype=np.float32)).cuda()
    Od = torch.empty(cfg.B, cfg.T, cfg.H, cfg.dv, dtype=torch.bfloat16, device="cuda")
    Sfd = torch.empty(cfg.B, cfg.H, cfg.dv, cfg.dk, dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    for _ in range(3):
        carve.carve_fwd(p, xd, Od, Sfd, ws, st)
        carve.carve_bwd(p, xd, dO, dSf, gd, ws, st)
    torch.cuda.synchronize()
    assert np.array_equal(Od.float().cpu().numpy().astype(np.float64), O)
    for n in GRADS:
        assert np.array_equal(gd[n].float().cpu().numpy().astype(np.float64), g0[n]), n

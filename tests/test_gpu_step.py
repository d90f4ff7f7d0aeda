"""GPU parity of carve_step (the recurrent / decode form; Table 1 l.432, l.450) against
the fp64 oracle: one call of n tokens == the chunked definition with T = L = n and S0 = S; a token-by-token decode
loop (n = 1) == the oracle at L = 1 over the whole sequence, state carried through the in/out buffer."""
import numpy as np
import pytest
import torch

from paper_2606_27229_b200 import carve, synth
from tests.gpu_util import oracle_shape, params_of, relerr, to_device

pytestmark = pytest.mark.gpu


def _step(p, xd, S, n_tok_dtype):
    O = torch.empty(p.B, p.T, p.H, p.dv, dtype=n_tok_dtype, device="cuda")
    carve.carve_step(p, xd, S, O, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return O.float().cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("dtype,tol", [("f32", 1e-4), ("bf16", 2e-2)])
@pytest.mark.parametrize("n", [1, 3, 16])
@pytest.mark.parametrize("dk,dv,r", [(64, 64, 8), (128, 128, 16), (128, 256, 16), (64, 128, 32)])
def test_step_equals_chunked_definition(oracle, dtype, tol, n, dk, dv, r):
    cfg = synth.Config("step", B=3, H=2, T=n, L=16, dk=dk, dv=dv, r=r, dtype=dtype, wstd=0.1, s0_std=0.3, seed=n + dk)
    x = synth.scale_qk_rows(synth.make_inputs(cfg, with_decay_params=True), cfg)
    tok = torch.bfloat16 if dtype == "bf16" else torch.float32
    xd = to_device(x, tok)
    S = xd["S0"].clone()
    p = params_of(cfg)
    O = _step(p, xd, S, tok)
    O_ref, S_ref = oracle.fwd(oracle_shape(oracle, cfg, L=n), x)
    assert relerr(O, O_ref) <= tol
    assert relerr(S.cpu().numpy().astype(np.float64), S_ref) <= tol


def test_decode_loop_is_exact_per_token_gating(oracle):
    """64 single-token calls with the state carried in place == the oracle at L = 1 (no staleness, l.450)."""
    T = 64
    cfg = synth.Config("dec", B=2, H=3, T=T, L=16, dk=128, dv=128, r=16, dtype="f32", wstd=0.1, s0_std=0.2, seed=9)
    x = synth.make_inputs(cfg)
    O_ref, S_ref = oracle.fwd(oracle_shape(oracle, cfg, L=1), x)
    xd = to_device(x, torch.float32)
    S = xd["S0"].clone()
    p1 = params_of(cfg.with_(T=1))
    outs = []
    for t in range(T):
        xt = {n: (v[:, t:t + 1].contiguous() if (v is not None and n in synth.TOKEN_TENSORS) else v) for n, v in xd.items()}
        outs.append(_step(p1, xt, S, torch.float32))
    O = np.concatenate(outs, axis=1)
    assert relerr(O, O_ref) <= 1e-4
    assert relerr(S.cpu().numpy().astype(np.float64), S_ref) <= 1e-4


def test_step_refuses_bad_shapes(oracle):
    cfg = synth.Config("step", B=1, H=1, T=17, L=16, dk=64, dv=64, r=8, dtype="f32", s0_std=0.1)
    x = synth.make_inputs(cfg)
    xd = to_device(x, torch.float32)
    S = xd["S0"].clone()
    O = torch.empty(1, 17, 1, 64, device="cuda")
    with pytest.raises(carve.CarveError) as ei:
        carve.carve_step(params_of(cfg), xd, S, O)
    assert ei.value.status == 2
    with pytest.raises(carve.CarveError) as ei:
        carve.carve_step(params_of(cfg.with_(T=4)), xd, None, O)
    assert ei.value.status == 1


@pytest.mark.parametrize("dtype,tol", [("f32", 1e-4), ("bf16", 2e-2)])
@pytest.mark.parametrize("dk,dv,r", [(64, 64, 8), (128, 128, 16)])
def test_step_varlen_ragged_batch(oracle, dtype, tol, dk, dv, r):
    """carve_step_varlen (cu_seqlens; SURVEY 8(f) NEXT-1 "variable-length batches"): sequences with 0..16 new tokens in one
    packed call == the oracle on every sequence alone (T = L = its length, S0 = its state); the sequence with no new
    token keeps its state bit for bit."""
    lens = [3, 0, 16, 1, 7]
    B, H, Tmax = len(lens), 2, 16
    cfg = synth.Config("ragged", B=B, H=H, T=Tmax, L=16, dk=dk, dv=dv, r=r, dtype=dtype, wstd=0.1, s0_std=0.3, seed=dk + r)
    x = synth.scale_qk_rows(synth.make_inputs(cfg, with_decay_params=True), cfg)
    tok = torch.bfloat16 if dtype == "bf16" else torch.float32
    # pack the first lens[b] tokens of every sequence: [N, H, d]
    packed = {}
    for n, a in x.items():
        if a is not None and n in synth.TOKEN_TENSORS:
            packed[n] = np.concatenate([a[b, :lens[b]] for b in range(B)], axis=0)[None]   # [1, N, H, d]: to_device keeps the layout
        else:
            packed[n] = a
    xd = to_device(packed, tok)
    N = sum(lens)
    cu = torch.tensor(np.concatenate([[0], np.cumsum(lens)]), dtype=torch.int32, device="cuda")
    S = xd["S0"].clone()
    S_in = S.clone()
    O = torch.full((N, H, dv), float("nan"), dtype=tok, device="cuda")
    carve.carve_step_varlen(params_of(cfg), xd, S, O, cu, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    O_np, S_np = O.float().cpu().numpy().astype(np.float64), S.cpu().numpy().astype(np.float64)
    assert np.isfinite(O_np).all()
    off = 0
    for b, n in enumerate(lens):
        if n == 0:
            assert torch.equal(S[b], S_in[b])
            continue
        xb = {m: (a[b:b + 1, :n] if (a is not None and m in synth.TOKEN_TENSORS) else (a[b:b + 1] if m == "S0" else a))
              for m, a in x.items()}
        O_ref, S_ref = oracle.fwd(oracle_shape(oracle, cfg, B=1, T=n, L=n), xb)
        assert relerr(O_np[off:off + n][None], O_ref) <= tol, (b, n)
        assert relerr(S_np[b:b + 1], S_ref) <= tol, (b, n)
        off += n
    with pytest.raises(carve.CarveError) as ei:
        carve.carve_step_varlen(params_of(cfg), xd, S, O, None)
    assert ei.value.status == 1

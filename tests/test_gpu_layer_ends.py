"""GPU parity of the layer ends (Eq. 6 l.125, Alg. 1 line 15 l.194) against
oracle/layer_ends.py: SiLU on q, k, v and RMSNorm of the assembled output, forward and backward, both dtypes, at shapes
that span several grid strides and leave ragged tails (rows not a multiple of the warp count, pieces per row not a
multiple of 32)."""
import numpy as np
import pytest
import torch

from oracle import layer_ends as le
from paper_2606_27229_b200 import carve
from tests.gpu_util import relerr

pytestmark = pytest.mark.gpu

SHAPES = [  # B, T, H, dk, dv
    (2, 64, 2, 64, 64),        # config-0 like: 128 channels per token
    (1, 300, 3, 64, 128),      # ragged: 384 channels = 48 (bf16) / 96 (fp32) pieces per row
    (2, 1536, 16, 128, 128),   # config-1 rows (2048 channels), more rows than warps in the grid
    (1, 64, 16, 128, 256),     # config-3 rows (4096 channels, bf16 only)
]


def _p(B, T, H, dk, dv, dtype):
    return carve.Params(B=B, H=H, T=T, L=min(T, 64), dk=dk, dv=dv, r=8, dtype=carve.CARVE_BF16 if dtype == "bf16" else carve.CARVE_F32)


def _dev(a, tok):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(tok).cuda().contiguous()


def _host(t):
    return t.float().cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("dtype,tol", [("f32", 1e-4), ("bf16", 2e-2)])
@pytest.mark.parametrize("shape", SHAPES[:3], ids=str)
def test_silu_qkv(shape, dtype, tol):
    B, T, H, dk, dv = shape
    tok = torch.bfloat16 if dtype == "bf16" else torch.float32
    rng = np.random.default_rng(sum(shape))
    p = _p(B, T, H, dk, dv, dtype)
    xs = [_dev(rng.normal(0, 2.0, (B, T, H, d)), tok) for d in (dk, dk, dv)]
    dys = [_dev(rng.normal(0, 1.0, (B, T, H, d)), tok) for d in (dk, dk, dv)]
    ys = [torch.empty_like(x) for x in xs]
    carve.carve_silu_qkv_fwd(p, *xs, *ys, torch.cuda.current_stream().cuda_stream)
    g = [d.clone() for d in dys]
    carve.carve_silu_qkv_bwd(p, *xs, *g, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    for x, y, dy, dx in zip(xs, ys, dys, g):
        assert relerr(_host(y), le.silu(_host(x))) <= tol
        assert relerr(_host(dx), le.silu_bwd(_host(x), _host(dy))) <= tol
    # one tensor alone (the other two skipped), in place
    v2 = xs[2].clone()
    carve.carve_silu_qkv_fwd(p, None, None, v2, None, None, v2)
    torch.cuda.synchronize()
    assert torch.equal(v2, ys[2])
    with pytest.raises(carve.CarveError) as ei:
        carve.carve_silu_qkv_fwd(p, xs[0], None, None, None, None, None)
    assert ei.value.status == 1


@pytest.mark.parametrize("dtype,tol", [("f32", 1e-4), ("bf16", 2e-2)])
@pytest.mark.parametrize("shape", SHAPES, ids=str)
def test_out_norm(shape, dtype, tol):
    B, T, H, dk, dv = shape
    if dtype == "f32" and H * dv > 2048:
        pytest.skip("rows above 8 KB are outside the declared shape set")
    tok = torch.bfloat16 if dtype == "bf16" else torch.float32
    rng = np.random.default_rng(sum(shape) + 1)
    p = _p(B, T, H, dk, dv, dtype)
    eps = 1e-5
    o = _dev(rng.normal(0, 1.5, (B, T, H, dv)) * rng.uniform(0.1, 4.0, (B, T, 1, 1)), tok)   # token scales vary
    dy = _dev(rng.normal(0, 1.0, (B, T, H, dv)), tok)
    gain = torch.from_numpy(rng.normal(1.0, 0.3, H * dv).astype(np.float32)).cuda()
    y = torch.empty_like(o)
    st = torch.cuda.current_stream().cuda_stream
    carve.carve_out_norm_fwd(p, o, gain, eps, y, st)
    ws = torch.empty(carve.carve_out_norm_workspace_bytes(p), dtype=torch.uint8, device="cuda")
    outs = []
    for _ in range(2):
        d_o, dgain = torch.empty_like(o), torch.empty_like(gain)
        carve.carve_out_norm_bwd(p, o, gain, eps, dy, d_o, dgain, ws, st)
        outs.append((d_o, dgain))
    torch.cuda.synchronize()
    assert relerr(_host(y), le.out_norm(_host(o), _host(gain), eps)) <= tol
    do_ref, dg_ref = le.out_norm_bwd(_host(o), _host(gain), eps, _host(dy))
    assert relerr(_host(outs[0][0]), do_ref) <= tol
    assert relerr(_host(outs[0][1]), dg_ref) <= tol
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])   # fixed summation order
    with pytest.raises(carve.CarveError) as ei:
        carve.carve_out_norm_bwd(p, o, gain, eps, dy, outs[0][0], outs[0][1], None)
    assert ei.value.status == 5


def test_out_norm_refuses_long_rows():
    p = _p(1, 8, 32, 128, 256, "bf16")   # 8192 channels: 16 KB rows
    assert carve.carve_out_norm_workspace_bytes(p) == 0
    o = torch.zeros(1, 8, 32, 256, dtype=torch.bfloat16, device="cuda")
    with pytest.raises(carve.CarveError) as ei:
        carve.carve_out_norm_fwd(p, o, torch.ones(8192, device="cuda"), 1e-5, o)
    assert ei.value.status == 2

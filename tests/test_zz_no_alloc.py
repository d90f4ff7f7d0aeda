"""carve_fwd_bwd_static (include/carve.h): training forward + backward with the workspace in the library's static device
array -- for callers that cannot allocate (CUDA graph capture, serving loops).  Checked against the existing path
(carve_fwd + carve_bwd with a caller workspace) on two calls in a row with different inputs: the array is shared and
keeps the first call's contents, so the second call shows that nothing depends on a clean start.

The file is named so that pytest collects it last (the suite runs with `pytest -x`); it passes alone in a fresh
process and after the other tests.
"""
import numpy as np
import pytest
import torch

from paper_2606_27229_b200 import carve, synth
from tests.gpu_util import GRADS, alloc_grads, params_of, relerr, to_device

pytestmark = pytest.mark.gpu

# the tolerances of tests/test_gpu_parity.py: bf16 tokens 2e-2 / 3e-2, fp32 1e-4
CASES = [
    (synth.Config("static_bf16_tensor", B=2, H=2, T=256, L=64, dk=128, dv=128, r=16, dtype="bf16", wstd=0.1, seed=11), 2e-2, 3e-2),
    (synth.Config("static_bf16_d64", B=1, H=4, T=256, L=32, dk=64, dv=64, r=8, dtype="bf16", wstd=0.1, seed=12), 2e-2, 3e-2),
    (synth.CFG0, 1e-4, 1e-4),
]


def _both_paths(cfg, seed):
    cfg = cfg.with_(seed=seed)
    x, ct = synth.make_inputs(cfg), synth.make_cotangents(cfg)
    p = params_of(cfg)
    tok = torch.bfloat16 if cfg.dtype == "bf16" else torch.float32
    st = torch.cuda.current_stream().cuda_stream
    xd = to_device(x, tok)
    dO = to_device({"dO": ct["dO"]}, tok)["dO"]
    dSf = torch.from_numpy(np.ascontiguousarray(ct["dS_final"], dtype=np.float32)).cuda()

    def outputs():
        O = torch.empty(cfg.B, cfg.T, cfg.H, cfg.dv, dtype=tok, device="cuda")
        Sf = torch.empty(cfg.B, cfg.H, cfg.dv, cfg.dk, dtype=torch.float32, device="cuda")
        return O, Sf, alloc_grads(p, tok)

    # existing path: caller-allocated workspace
    need = carve.carve_workspace_bytes(p, True)
    assert 0 < need <= carve.carve_static_scratch_bytes()
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    O1, S1, g1 = outputs()
    carve.carve_fwd(p, xd, O1, S1, ws, st)
    carve.carve_bwd(p, xd, dO, dSf, g1, ws, st)
    # new entry point: no workspace argument at all
    O2, S2, g2 = outputs()
    carve.carve_fwd_bwd_static(p, xd, O2, S2, dO, dSf, g2, st)
    torch.cuda.synchronize()
    ref = dict(g1, O=O1, S_final=S1)
    got = dict(g2, O=O2, S_final=S2)
    return ref, got


@pytest.mark.parametrize("cfg,tol_o,tol_g", CASES, ids=lambda c: getattr(c, "name", None))
def test_static_scratch_matches_workspace_path_twice(cfg, tol_o, tol_g):
    for call, seed in enumerate((cfg.seed, cfg.seed + 100)):   # two calls in a row, different inputs
        ref, got = _both_paths(cfg, seed)
        for n in ("O", "S_final") + GRADS:
            a, b = got[n].float().cpu().numpy().astype(np.float64), ref[n].float().cpu().numpy().astype(np.float64)
            assert np.isfinite(a).all(), (call, n)
            assert relerr(a, b) <= (tol_o if n in ("O", "S_final") else tol_g), (call, n, relerr(a, b))
            # same kernels, same launch configuration, no floating-point atomics: the results are in fact identical
            assert torch.equal(got[n], ref[n]), (call, n)


def test_static_scratch_limit_is_an_error():
    """A problem whose workspace exceeds the static array is rejected with CARVE_ERR_STATIC_LIMIT before any launch."""
    cfg = synth.CFG1.with_(B=1, H=2)   # 128 chain-chunks x 262 KB of records > 16 MiB
    p = params_of(cfg)
    assert carve.carve_workspace_bytes(p, True) > carve.carve_static_scratch_bytes()
    tok = torch.bfloat16
    e = lambda *s: torch.zeros(*s, dtype=tok, device="cuda")
    f = lambda *s: torch.zeros(*s, dtype=torch.float32, device="cuda")
    B, H, T, d, r = cfg.B, cfg.H, cfg.T, cfg.dk, cfg.r
    x = {"q": e(B, T, H, d), "k": e(B, T, H, d), "v": e(B, T, H, d), "f": e(B, T, H, d), "bx": e(B, T, H, d),
         "wx": e(B, T, H, d), "beta": e(B, T, H), "A": f(H, d), "tau": f(H, d), "Ub": f(r, d), "Uw": f(r, d),
         "Vb": f(d, r), "Vw": f(d, r), "S0": None}
    O = torch.full((B, T, H, d), 7.0, dtype=tok, device="cuda")
    Sf = f(B, H, d, d)
    with pytest.raises(carve.CarveError) as ei:
        carve.carve_fwd_bwd_static(p, x, O, Sf, e(B, T, H, d), None, alloc_grads(p, tok), torch.cuda.current_stream().cuda_stream)
    assert ei.value.status == 8 and "static" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((O == 7.0).all())   # nothing ran

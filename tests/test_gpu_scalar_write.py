"""GPU parity of the scalar-write variant (section 4.2 l.145, Thm 15 l.762-764): wx = Uw = Vw =
NULL selects the kernels' w == 1 path.  The oracle has no such switch: it computes the same function with wx = +40
(sigmoid(40) rounds to 1 in fp64) and Uw = Vw = 0, which is what the variant means (reading A1: the scalar write gate
multiplies the whole error and is passed inside beta)."""
import numpy as np
import pytest
import torch

from paper_2606_27229_b200 import carve, synth
from tests.gpu_util import GRADS, alloc_grads, oracle_shape, params_of, relerr, to_device

pytestmark = pytest.mark.gpu
SKIP = ("dwx", "dUw", "dVw")


def _oracle_inputs(x):
    xo = dict(x)
    xo["wx"] = np.full_like(x["wx"], 40.0)
    xo["Uw"] = np.zeros_like(x["Uw"])
    xo["Vw"] = np.zeros_like(x["Vw"])
    return xo


@pytest.mark.parametrize("path,dtype,tol_o,tol_g", [(carve.CARVE_PATH_SIMT, "f32", 1e-4, 1e-4), (carve.CARVE_PATH_SIMT, "bf16", 2e-2, 3e-2),
                                                     (carve.CARVE_PATH_TENSOR, "bf16", 2e-2, 3e-2)])
@pytest.mark.parametrize("d,r,L", [(64, 8, 64), (128, 16, 64), (128, 16, 128), (64, 8, 16)])
def test_scalar_write_fwd_bwd(oracle, path, dtype, tol_o, tol_g, d, r, L):
    cfg = synth.Config("sw", B=2, H=2, T=256, L=L, dk=d, dv=d, r=r, dtype=dtype, wstd=0.1, s0_std=0.05, seed=d + L)
    x, ct = synth.scale_qk_rows(synth.make_inputs(cfg, with_decay_params=True), cfg), synth.make_cotangents(cfg)
    s = oracle_shape(oracle, cfg)
    xo = _oracle_inputs(x)
    O_ref, S_ref = oracle.fwd(s, xo)
    g_ref = oracle.bwd(s, xo, ct["dO"], ct["dS_final"])
    for n in SKIP:
        assert np.max(np.abs(g_ref[n])) < 1e-12      # the oracle agrees that nothing flows into the switched-off gate

    p = params_of(cfg, path=path)
    assert carve.carve_resolved_path(p, True) == path
    tok = torch.bfloat16 if dtype == "bf16" else torch.float32
    xd = to_device(dict(x, wx=None, Uw=None, Vw=None), tok)
    O = torch.empty(cfg.B, cfg.T, cfg.H, cfg.dv, dtype=tok, device="cuda")
    Sf = torch.empty(cfg.B, cfg.H, cfg.dv, cfg.dk, dtype=torch.float32, device="cuda")
    ws = torch.empty(carve.carve_workspace_bytes(p, True), dtype=torch.uint8, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    carve.carve_fwd(p, xd, O, Sf, ws, st)
    g = alloc_grads(p, tok)
    for n in SKIP:
        g[n] = None
    carve.carve_bwd(p, xd, to_device({"dO": ct["dO"]}, tok)["dO"], torch.from_numpy(ct["dS_final"]).cuda(), g, ws, st)
    torch.cuda.synchronize()
    assert relerr(O.float().cpu().numpy().astype(np.float64), O_ref) <= tol_o
    assert relerr(Sf.cpu().numpy().astype(np.float64), S_ref) <= tol_o
    for n in GRADS:
        if n in SKIP:
            continue
        got = g[n].float().cpu().numpy().astype(np.float64)
        assert np.isfinite(got).all(), n
        assert relerr(got, g_ref[n]) <= tol_g, (n, relerr(got, g_ref[n]))


def test_scalar_write_step_and_partial_null(oracle):
    cfg = synth.Config("sw", B=2, H=2, T=4, L=16, dk=128, dv=128, r=16, dtype="f32", wstd=0.1, s0_std=0.3, seed=3)
    x = synth.make_inputs(cfg)
    O_ref, S_ref = oracle.fwd(oracle_shape(oracle, cfg, L=cfg.T), _oracle_inputs(x))
    xd = to_device(dict(x, wx=None, Uw=None, Vw=None), torch.float32)
    S = xd["S0"].clone()
    O = torch.empty(cfg.B, cfg.T, cfg.H, cfg.dv, device="cuda")
    carve.carve_step(params_of(cfg), xd, S, O, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert relerr(O.cpu().numpy().astype(np.float64), O_ref) <= 1e-4
    assert relerr(S.cpu().numpy().astype(np.float64), S_ref) <= 1e-4
    # only some of the three NULL: refused
    xbad = to_device(dict(x, wx=None), torch.float32)
    with pytest.raises(carve.CarveError) as ei:
        carve.carve_step(params_of(cfg), xbad, S, O)
    assert ei.value.status == 1

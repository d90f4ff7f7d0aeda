"""Full-size, full-tensor GPU parity for every BASELINE.json config, in the launch configuration bench.py times.

The GPU computes the whole workload in one carve_fwd (+ carve_bwd) call; the oracle recomputes EVERY (batch, head)
chain -- one batch element at a time, to bound host memory; chains are independent (Alg. 2 l.318) -- and every output
tensor is compared element by element: O, S_final, the seven per-token gradients, dS0, and the shared-weight gradients
dUb, dUw, dVb, dVw (and dA, dtau) summed over ALL chains (reduce over heads and batch, Alg. 4 l.816).
SURVEY 8(d): "Parity, unlike timing, is always on the full tensors."
"""
import numpy as np
import pytest
import torch

from paper_2606_27229_b200 import carve, synth
from tests.gpu_util import alloc_grads, oracle_shape, params_of, to_device

pytestmark = pytest.mark.gpu

TOL = dict(O=2e-2, S=2e-2, g=3e-2)
PER_TOKEN = ("dq", "dk", "dv", "df", "dbx", "dwx", "dbeta")
WEIGHTS = ("dA", "dtau", "dUb", "dUw", "dVb", "dVw")


class _MaxErr:
    """Running max|x - ref| and max|ref| of one tensor over the batch slices: relerr of SURVEY 8(c) A12."""

    def __init__(self):
        self.err, self.ref = 0.0, 0.0

    def add(self, got, ref):
        self.err = max(self.err, float(np.max(np.abs(got.astype(np.float64) - ref))))
        self.ref = max(self.ref, float(np.max(np.abs(ref))))

    @property
    def rel(self):
        return self.err / max(self.ref, 1e-30)


def _full_tensor_parity(oracle, cfg):
    x = synth.make_inputs(cfg)
    ct = None if cfg.fwd_only else synth.make_cotangents(cfg)
    p = params_of(cfg)
    assert carve.carve_resolved_path(p, not cfg.fwd_only) == carve.CARVE_PATH_TENSOR
    st = torch.cuda.current_stream().cuda_stream
    xd = to_device(x, torch.bfloat16)
    O = torch.empty(cfg.B, cfg.T, cfg.H, cfg.dv, dtype=torch.bfloat16, device="cuda")
    Sf = torch.empty(cfg.B, cfg.H, cfg.dv, cfg.dk, dtype=torch.float32, device="cuda")
    ws = None if cfg.fwd_only else torch.empty(carve.carve_workspace_bytes(p, True), dtype=torch.uint8, device="cuda")
    carve.carve_fwd(p, xd, O, Sf, ws, st)
    out = {"O": O, "S_final": Sf}
    if not cfg.fwd_only:
        dO = to_device({"dO": ct["dO"]}, torch.bfloat16)["dO"]
        dSf = torch.from_numpy(ct["dS_final"]).cuda()
        g = alloc_grads(p, torch.bfloat16)
        carve.carve_bwd(p, xd, dO, dSf, g, ws, st)
        out.update(g)
    torch.cuda.synchronize()
    host = {n: t.float().cpu().numpy() for n, t in out.items() if t is not None}
    del xd, O, Sf, ws, out
    torch.cuda.empty_cache()
    for n, a in host.items():
        assert np.isfinite(a).all(), n

    errs = {n: _MaxErr() for n in host if n not in WEIGHTS}
    wsum = {n: 0.0 for n in WEIGHTS}
    s1 = oracle_shape(oracle, cfg, B=1)
    for b in range(cfg.B):
        xb = {n: (a[b:b + 1] if (a is not None and n in synth.TOKEN_TENSORS + ("S0",)) else a) for n, a in x.items()}
        O_ref, S_ref = oracle.fwd(s1, xb)
        errs["O"].add(host["O"][b:b + 1], O_ref)
        errs["S_final"].add(host["S_final"][b:b + 1], S_ref)
        if cfg.fwd_only:
            continue
        g_ref = oracle.bwd(s1, xb, ct["dO"][b:b + 1], ct["dS_final"][b:b + 1])
        for n in PER_TOKEN + ("dS0",):
            errs[n].add(host[n][b:b + 1], g_ref[n])
        for n in WEIGHTS:
            wsum[n] = wsum[n] + g_ref[n]
    rel = {n: e.rel for n, e in errs.items()}
    if not cfg.fwd_only:
        for n in WEIGHTS:
            rel[n] = float(np.max(np.abs(host[n].astype(np.float64) - wsum[n])) / max(float(np.max(np.abs(wsum[n]))), 1e-30))
    print(cfg.name, {n: f"{v:.2e}" for n, v in rel.items()})
    assert rel["O"] <= TOL["O"] and rel["S_final"] <= TOL["S"], rel
    for n, v in rel.items():
        if n not in ("O", "S_final"):
            assert v <= TOL["g"], (n, rel)


def test_config1_full_tensors(oracle):
    """Config 1 (1.3B-like, 128 chains x 64 chunks): every tensor, every chain, weight gradients over all chains."""
    _full_tensor_parity(oracle, synth.CFG1)


@pytest.mark.parametrize("L", [16, 32, 64, 128])
def test_config2_full_tensors(oracle, L):
    """Config 2 (64 chains, T = 8192, gate projections ~N(0,0.1^2): content gates active) at every chunk length."""
    _full_tensor_parity(oracle, synth.CFG2[L])


def test_config3_full_tensors(oracle):
    """Config 3 (forward only, 16 chains x 1024 chunks, d_v = 256 split over a CTA cluster, random S0): all 16 chains."""
    _full_tensor_parity(oracle, synth.CFG3)


def test_config4_full_tensors(oracle):
    """Config 4 (2048 chains, d = 64, beta = 1 on 10 % of tokens, no decay on 10 % of key dims): every chain of every wave."""
    _full_tensor_parity(oracle, synth.CFG4)


@pytest.mark.parametrize("cfg", [synth.CFG1, synth.CFG4, synth.CFG2[128]], ids=lambda c: c.name)
def test_full_size_run_to_run_bitwise(cfg):
    """Two back-to-back fwd+bwd calls at full size give bit-identical tensors (no float atomics; and a race between the
    asynchronous copies -- TMA loads, record bulk copies, the staged output store -- and the threads would show here)."""
    x, ct = synth.make_inputs(cfg), synth.make_cotangents(cfg)
    p = params_of(cfg)
    st = torch.cuda.current_stream().cuda_stream
    xd = to_device(x, torch.bfloat16)
    dO = to_device({"dO": ct["dO"]}, torch.bfloat16)["dO"]
    dSf = torch.from_numpy(ct["dS_final"]).cuda()
    ws = torch.empty(carve.carve_workspace_bytes(p, True), dtype=torch.uint8, device="cuda")
    outs = []
    for _ in range(2):
        O = torch.empty(cfg.B, cfg.T, cfg.H, cfg.dv, dtype=torch.bfloat16, device="cuda")
        Sf = torch.empty(cfg.B, cfg.H, cfg.dv, cfg.dk, dtype=torch.float32, device="cuda")
        g = alloc_grads(p, torch.bfloat16)
        carve.carve_fwd(p, xd, O, Sf, ws, st)
        carve.carve_bwd(p, xd, dO, dSf, g, ws, st)
        torch.cuda.synchronize()
        outs.append(dict(g, O=O, S_final=Sf))
    for n in outs[0]:
        assert torch.equal(outs[0][n], outs[1][n]), n

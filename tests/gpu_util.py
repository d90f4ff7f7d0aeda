"""Helpers for the GPU parity tests: numpy inputs -> device tensors -> C ABI -> numpy."""
from __future__ import annotations

import numpy as np
import torch

from paper_2606_27229_b200 import carve, synth

FWD_IN = ("q", "k", "v", "f", "bx", "wx", "beta", "A", "tau", "Ub", "Uw", "Vb", "Vw", "S0")
GRADS = ("dq", "dk", "dv", "df", "dbx", "dwx", "dbeta", "dA", "dtau", "dUb", "dUw", "dVb", "dVw", "dS0")


def params_of(cfg: synth.Config, path=carve.CARVE_PATH_AUTO, **kw) -> carve.Params:
    d = dict(B=cfg.B, H=cfg.H, T=cfg.T, L=cfg.L, dk=cfg.dk, dv=cfg.dv, r=cfg.r,
             dtype=carve.CARVE_BF16 if cfg.dtype == "bf16" else carve.CARVE_F32,
             qk_l2norm=cfg.qk_l2norm, scale=cfg.scale, eps=cfg.eps, path=path)
    d.update(kw)
    return carve.Params(**d)


def to_device(x: dict, tok_dtype: torch.dtype, device="cuda") -> dict:
    out = {}
    for n, a in x.items():
        if a is None:
            out[n] = None
            continue
        t = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32))
        if n in synth.TOKEN_TENSORS or n == "dO":
            t = t.to(tok_dtype)
        out[n] = t.to(device).contiguous()
    return out


def alloc_grads(p: carve.Params, tok_dtype, device="cuda", with_decay=True) -> dict:
    B, H, T, dk, dv, r = p.B, p.H, p.T, p.dk, p.dv, p.r
    e = lambda *s: torch.empty(*s, dtype=tok_dtype, device=device)
    f = lambda *s: torch.empty(*s, dtype=torch.float32, device=device)
    return {"dq": e(B, T, H, dk), "dk": e(B, T, H, dk), "dv": e(B, T, H, dv), "df": e(B, T, H, dk),
            "dbx": e(B, T, H, dk), "dwx": e(B, T, H, dv), "dbeta": e(B, T, H),
            "dA": f(H, dk) if with_decay else None, "dtau": f(H, dk) if with_decay else None,
            "dUb": f(r, dv), "dUw": f(r, dv), "dVb": f(dk, r), "dVw": f(dv, r), "dS0": f(B, H, dv, dk)}


def run_fwd(p: carve.Params, x: dict, need_bwd=False):
    """x: numpy dict.  Returns (O, S_final) as float64 numpy plus the device handles for bwd."""
    tok = torch.bfloat16 if p.dtype == carve.CARVE_BF16 else torch.float32
    xd = to_device(x, tok)
    O = torch.empty(p.B, p.T, p.H, p.dv, dtype=tok, device="cuda")
    Sf = torch.empty(p.B, p.H, p.dv, p.dk, dtype=torch.float32, device="cuda")
    ws = None
    if need_bwd:
        ws = torch.empty(carve.carve_workspace_bytes(p, True), dtype=torch.uint8, device="cuda")
    carve.carve_fwd(p, xd, O, Sf, ws, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return O.float().cpu().numpy().astype(np.float64), Sf.cpu().numpy().astype(np.float64), (xd, ws)


def run_bwd(p: carve.Params, handles, ct: dict):
    xd, ws = handles
    tok = torch.bfloat16 if p.dtype == carve.CARVE_BF16 else torch.float32
    ctd = to_device({"dO": ct["dO"]}, tok)
    dSf = None if ct.get("dS_final") is None else torch.from_numpy(
        np.ascontiguousarray(ct["dS_final"], dtype=np.float32)).cuda()
    g = alloc_grads(p, tok)
    carve.carve_bwd(p, xd, ctd["dO"], dSf, g, ws, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return {n: (None if t is None else t.float().cpu().numpy().astype(np.float64)) for n, t in g.items()}, g


def relerr(a, ref) -> float:
    """Per-tensor error of SURVEY 8(c) A12: max|x - ref| / max|ref|."""
    return float(np.max(np.abs(a - ref)) / max(float(np.max(np.abs(ref))), 1e-30))


def oracle_shape(oracle, cfg: synth.Config, **kw):
    d = dict(B=cfg.B, H=cfg.H, T=cfg.T, L=cfg.L, dk=cfg.dk, dv=cfg.dv, r=cfg.r,
             qk_l2norm=cfg.qk_l2norm, scale=cfg.scale, eps=cfg.eps)
    d.update(kw)
    return oracle.Shape(**d)

"""Seeded synthetic inputs for the CARVE layer operator.

This module serves BOTH the CUDA path's callers (tests, bench.py, smoke) and the oracle's
callers; it holds none of the method's arithmetic -- only the random draws, the value
distributions BASELINE.json's configs prescribe, bf16 rounding of the inputs, and slicing
helpers.  numpy only; it imports neither the oracle nor the CUDA binding.

Recipe: numpy.random.Generator(PCG64(seed)), float32 draws in this
fixed order: q, k, v, f, bx, wx, beta-logit, Ub, Uw, Vb, Vw, S0, [cfg-4 masks], dO, dS_final.
  q, k ~ N(0,1) then L2-normalised per token;  v ~ N(0,1);  beta = sigmoid(N(0,1));
  f ~ N(0,1) with A = tau = NULL, so g = -softplus(f) ("through logsigmoid");
  bx, wx ~ N(0,1);  Ub, Uw, Vb, Vw ~ N(0, wstd^2);  S0 = 0 or N(0, s0_std^2).
Token tensors (q,k,v,f,bx,wx,beta,dO) are rounded to bf16 (round-to-nearest-even) when
dtype == "bf16"; the same rounded values go to the oracle (upcast to fp64) and to the GPU.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace

import numpy as np

TOKEN_TENSORS = ("q", "k", "v", "f", "bx", "wx", "beta")


@dataclass(frozen=True)
class Config:
    name: str
    B: int
    H: int
    T: int
    L: int
    dk: int
    dv: int
    r: int
    dtype: str = "bf16"          # "f32" | "bf16": dtype of token tensors and their grads
    wstd: float = 0.02           # std of Ub,Uw,Vb,Vw
    s0_std: float = 0.0          # 0 => S0 = None (zeros)
    beta_one_frac: float = 0.0   # cfg 4: beta := 1 on this fraction of (b,t,h)
    nodecay_frac: float = 0.0    # cfg 4: f := -12 on this fraction of key dims per head
    fwd_only: bool = False
    qk_l2norm: int = 1
    scale: float = 1.0
    eps: float = 1e-6
    seed: int = 0

    def with_(self, **kw) -> "Config":
        return replace(self, **kw)

    @property
    def tokens(self) -> int:
        return self.B * self.T


# BASELINE.json "configs", in order.
CFG0 = Config("cfg0_tiny_fp32", B=1, H=1, T=256, L=64, dk=64, dv=64, r=8, dtype="f32")
CFG1 = Config("cfg1_1p3b_like", B=8, H=16, T=4096, L=64, dk=128, dv=128, r=16)
CFG2 = {L: Config(f"cfg2_chunk_sweep_L{L}", B=4, H=16, T=8192, L=L, dk=128, dv=128, r=16, wstd=0.1)
        for L in (16, 32, 64, 128)}
CFG3 = Config("cfg3_long_context_fwd", B=1, H=16, T=65536, L=64, dk=128, dv=256, r=16,
              s0_std=0.01, fwd_only=True)
CFG4 = Config("cfg4_many_short", B=64, H=32, T=1024, L=64, dk=64, dv=64, r=8,
              beta_one_frac=0.1, nodecay_frac=0.1)


def bf16_round(x: np.ndarray) -> np.ndarray:
    """Round float32 to the nearest bf16 (ties to even); result stays float32."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32)
    bias = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    r = ((u + bias) & np.uint32(0xFFFF0000)).astype(np.uint32)
    return r.view(np.float32).reshape(x.shape)


def bf16_bits(x: np.ndarray) -> np.ndarray:
    """uint16 bit patterns of an already bf16-representable float32 array."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    return (x.view(np.uint32) >> np.uint32(16)).astype(np.uint16).reshape(x.shape)


def _normal(rng, shape, std=1.0):
    a = rng.standard_normal(size=shape, dtype=np.float32)
    if std != 1.0:
        a *= np.float32(std)
    return a


def make_inputs(cfg: Config, zero_content: bool = False, with_decay_params: bool = False) -> dict:
    """Forward inputs of one config: dict of float32 numpy arrays (None for absent optionals)."""
    rng = np.random.Generator(np.random.PCG64(cfg.seed))
    B, H, T, dk, dv, r = cfg.B, cfg.H, cfg.T, cfg.dk, cfg.dv, cfg.r
    x = {}
    for name in ("q", "k"):
        a = _normal(rng, (B, T, H, dk))
        a /= np.sqrt((a.astype(np.float32) ** 2).sum(-1, keepdims=True))
        x[name] = a
    x["v"] = _normal(rng, (B, T, H, dv))
    x["f"] = _normal(rng, (B, T, H, dk))
    x["bx"] = _normal(rng, (B, T, H, dk))
    x["wx"] = _normal(rng, (B, T, H, dv))
    bl = _normal(rng, (B, T, H))
    x["beta"] = (1.0 / (1.0 + np.exp(-bl))).astype(np.float32)
    x["Ub"] = _normal(rng, (r, dv), cfg.wstd)
    x["Uw"] = _normal(rng, (r, dv), cfg.wstd)
    x["Vb"] = _normal(rng, (dk, r), cfg.wstd)
    x["Vw"] = _normal(rng, (dv, r), cfg.wstd)
    s0 = _normal(rng, (B, H, dv, dk), cfg.s0_std if cfg.s0_std > 0 else 1.0)
    x["S0"] = s0 if cfg.s0_std > 0 else None
    if cfg.beta_one_frac > 0:
        m = rng.random((B, T, H)) < cfg.beta_one_frac
        x["beta"][m] = 1.0
    if cfg.nodecay_frac > 0:
        m = rng.random((H, dk)) < cfg.nodecay_frac
        x["f"][:, :, m] = -12.0
    if with_decay_params:
        x["A"] = _normal(rng, (H, dk), 0.3)
        x["tau"] = _normal(rng, (H, dk), 0.5)
    else:
        x["A"] = None
        x["tau"] = None
    if zero_content:
        for n in ("Ub", "Uw", "Vb", "Vw"):
            x[n] = np.zeros_like(x[n])
    if cfg.dtype == "bf16":
        for n in TOKEN_TENSORS:
            x[n] = bf16_round(x[n])
    return x


def scale_qk_rows(x: dict, cfg: Config, lo: float = 0.5, hi: float = 2.0, tiny_rows: int = 0, seed: int = 11) -> dict:
    """Un-normalise q and k: multiply every token row by its own factor ~ U(lo, hi), so that the operator's
    L2-norm step (and the 1/|x| factor of its backward) has real work to do.  `tiny_rows` rows of each tensor
    get a norm of ~1e-3 = sqrt(eps) instead, where the eps inside the square root matters.  Re-rounds to bf16."""
    rng = np.random.Generator(np.random.PCG64([cfg.seed, seed]))
    out = dict(x)
    for name in ("q", "k"):
        a = np.array(x[name], dtype=np.float32, copy=True)
        sc = rng.uniform(lo, hi, size=a.shape[:-1] + (1,)).astype(np.float32)
        if tiny_rows:
            flat = sc.reshape(-1)
            flat[rng.choice(flat.size, size=min(tiny_rows, flat.size), replace=False)] = np.float32(1e-3)
        a *= sc
        out[name] = bf16_round(a) if cfg.dtype == "bf16" else a
    return out


def make_cotangents(cfg: Config) -> dict:
    """dO ~ N(0,1) in the token dtype and dS_final ~ N(0, 0.01^2) fp32 (drawn after the inputs)."""
    rng = np.random.Generator(np.random.PCG64([cfg.seed, 1]))
    dO = _normal(rng, (cfg.B, cfg.T, cfg.H, cfg.dv))
    dSf = _normal(rng, (cfg.B, cfg.H, cfg.dv, cfg.dk), 0.01)
    if cfg.dtype == "bf16":
        dO = bf16_round(dO)
    return {"dO": dO, "dS_final": dSf}


_PER_TOKEN = ("q", "k", "v", "f", "bx", "wx", "dO",
              "dq", "dk", "dv", "df", "dbx", "dwx", "O")


def slice_chains(x: dict, chains) -> dict:
    """Restrict a dict of [B,T,H,..] / [B,H,..] arrays to the listed (b, h) chains.

    The result is a B'=len(chains), H'=1 problem: every chain of the operator is independent
    (Alg. 2 "all operations are per-head"), the weights are shared.
    """
    out = {}
    bs = [c[0] for c in chains]
    hs = [c[1] for c in chains]
    for n, a in x.items():
        if a is None:
            out[n] = None
        elif n in _PER_TOKEN:
            out[n] = np.stack([a[b, :, h] for b, h in chains])[:, :, None, :]
        elif n in ("beta", "dbeta"):
            out[n] = np.stack([a[b, :, h] for b, h in chains])[:, :, None]
        elif n in ("S0", "dS_final", "S_final", "dS0"):
            out[n] = np.stack([a[b, h] for b, h in chains])[:, None]
        elif n in ("A", "tau"):
            # one head per sliced chain: only valid when all chains share h, else per-chain call
            assert len(set(hs)) == 1, "slice_chains with A/tau needs a single head"
            out[n] = a[hs[0]][None]
        else:
            out[n] = a
    return out

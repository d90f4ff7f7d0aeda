"""Data-parallel sharding of the CARVE operator over ranks: every (batch, head) chain is
independent, so a rank takes a slice of the batch; the only exchange is one sum all-reduce of the shared
weight gradients.  Host logic only -- none of the method's arithmetic."""
from __future__ import annotations

import numpy as np

BATCHED = ("q", "k", "v", "f", "bx", "wx", "beta", "S0", "dO", "dS_final",
           "dq", "dk", "dv", "df", "dbx", "dwx", "dbeta", "dS0", "O", "S_final")
WEIGHT_GRADS = ("dUb", "dUw", "dVb", "dVw", "dA", "dtau")   # order of the packed all-reduce buffer


def batch_range(B: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous, balanced slice [lo, hi) of the batch for `rank` (earlier ranks take the remainder)."""
    base, rem = divmod(B, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def shard_batch(x: dict, rank: int, world: int) -> dict:
    """Slice every batched array of `x` (inputs, cotangents or outputs) along dim 0; weights pass through."""
    out = {}
    for n, a in x.items():
        if a is None or n not in BATCHED:
            out[n] = a
        else:
            lo, hi = batch_range(a.shape[0], rank, world)
            out[n] = a[lo:hi]
    return out


def pack_weight_grads(g: dict) -> np.ndarray:
    return np.concatenate([np.asarray(g[n], dtype=np.float64).ravel() for n in WEIGHT_GRADS])


def unpack_weight_grads(buf: np.ndarray, like: dict) -> dict:
    out, o = {}, 0
    for n in WEIGHT_GRADS:
        k = int(np.prod(like[n].shape))
        out[n] = buf[o:o + k].reshape(like[n].shape)
        o += k
    return out

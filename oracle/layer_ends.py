"""fp64 oracle of the layer ends around the CARVE operator: the SiLU on q, k, v and the RMSNorm of
the assembled output, the two chunk-local "hoisted" launches of PAPER.md Alg. 3 steps 3 and 9 (l.399, l.407).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/ and bench.py's cpu_baseline leg may import this module; it imports
nothing from paper_2606_27229_b200/.

Each function is the plain definition in numpy float64:
  * q = SiLU(W_Q h), k = SiLU(W_K h), v = SiLU(W_V h)                      PAPER.md Eq. 6 l.125-126
    (the projections W h are dense GEMMs outside the path; the oracle starts from the pre-activations)
  * y = W_O RMSNorm(reshape(o))                                           PAPER.md Alg. 1 line 15 l.194
    reshape: [B,T,H,d_v] -> [B,T,H d_v]; RMSNorm over that last axis with a learned gain (the paper does not print the
    RMSNorm formula: the standard one, x / sqrt(mean(x^2) + eps) * gain, is taken -- DESIGN.md section 2, reading A16);
    W_O is a dense GEMM outside the path.
The backward functions are the exact adjoints, written from the chain rule (pinned by central differences and by the
invariants in tests/test_oracle_layer_ends.py).
"""
from __future__ import annotations

import numpy as np


def _sigmoid(x: np.ndarray) -> np.ndarray:
    # 1 / (1 + exp(-x)) without overflow for large |x|
    e = np.exp(-np.abs(x))
    return np.where(x >= 0, 1.0 / (1.0 + e), e / (1.0 + e))


def silu(x: np.ndarray) -> np.ndarray:
    """SiLU(x) = x sigmoid(x)  (Eq. 6 l.125)."""
    x = np.asarray(x, dtype=np.float64)
    return x * _sigmoid(x)


def silu_bwd(x: np.ndarray, dy: np.ndarray) -> np.ndarray:
    """dx = dy d/dx [x s(x)] = dy (s + x s (1 - s)),  s = sigmoid(x)."""
    x = np.asarray(x, dtype=np.float64)
    s = _sigmoid(x)
    return np.asarray(dy, dtype=np.float64) * (s + x * s * (1.0 - s))


def out_norm(o: np.ndarray, gain: np.ndarray, eps: float) -> np.ndarray:
    """RMSNorm(reshape(o)) (Alg. 1 line 15 l.194): o [B,T,H,dv] -> y [B,T,H,dv], normalised over the H*dv channels of a
    token, times gain [H*dv]."""
    o = np.asarray(o, dtype=np.float64)
    B, T, H, dv = o.shape
    x = o.reshape(B, T, H * dv)
    ms = np.mean(x * x, axis=-1, keepdims=True)
    y = x / np.sqrt(ms + eps) * np.asarray(gain, dtype=np.float64).reshape(1, 1, H * dv)
    return y.reshape(B, T, H, dv)


def out_norm_bwd(o: np.ndarray, gain: np.ndarray, eps: float, dy: np.ndarray):
    """Adjoint of out_norm: returns (do [B,T,H,dv], dgain [H*dv]).
    With x the token's channel vector, n = H*dv, r = (mean(x^2) + eps)^(-1/2), y = x r g:
        dgain = sum over tokens of dy x r
        dx    = r g dy - x r^3 mean(x g dy)        (d r / d x_j = -r^3 x_j / n)"""
    o = np.asarray(o, dtype=np.float64)
    B, T, H, dv = o.shape
    n = H * dv
    x = o.reshape(B, T, n)
    g = np.asarray(gain, dtype=np.float64).reshape(1, 1, n)
    d = np.asarray(dy, dtype=np.float64).reshape(B, T, n)
    r = 1.0 / np.sqrt(np.mean(x * x, axis=-1, keepdims=True) + eps)
    dgain = np.sum(d * x * r, axis=(0, 1))
    dx = r * g * d - x * r ** 3 * np.mean(x * g * d, axis=-1, keepdims=True)
    return dx.reshape(B, T, H, dv), dgain

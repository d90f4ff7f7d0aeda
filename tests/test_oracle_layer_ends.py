"""Pins of oracle/layer_ends.py (Eq. 6 l.125, Alg. 1 line 15 l.194) against what the
mathematics fixes: special values, invariants and central differences -- none of them re-types the oracle's formulas."""
import numpy as np

from oracle import layer_ends as le


def test_silu_special_values():
    # SiLU(0) = 0; SiLU(x) -> x for large x, -> 0 for large -x; SiLU(x) - SiLU(-x) = x (sigmoid(x) + sigmoid(-x) = 1)
    assert le.silu(np.array([0.0]))[0] == 0.0
    assert abs(le.silu(np.array([40.0]))[0] - 40.0) < 1e-12
    assert abs(le.silu(np.array([-40.0]))[0]) < 1e-12
    x = np.linspace(-8, 8, 101)
    assert np.max(np.abs(le.silu(x) - le.silu(-x) - x)) < 1e-14
    # printed constants of the function: its minimum -0.27846 at x = -1.27846 (where the derivative vanishes)
    xm = -1.2784645427610737
    assert abs(le.silu(np.array([xm]))[0] + 0.2784645427610738) < 1e-12
    assert abs(le.silu_bwd(np.array([xm]), np.array([1.0]))[0]) < 1e-12
    assert abs(le.silu_bwd(np.array([0.0]), np.array([1.0]))[0] - 0.5) < 1e-15


def test_silu_bwd_central_differences():
    rng = np.random.default_rng(0)
    x, dy = rng.normal(0, 2, 1000), rng.normal(0, 1, 1000)
    h = 1e-6
    fd = (le.silu(x + h) - le.silu(x - h)) / (2 * h) * dy
    assert np.max(np.abs(le.silu_bwd(x, dy) - fd)) < 1e-8


def _case(seed=0, B=2, T=3, H=4, dv=8):
    rng = np.random.default_rng(seed)
    return rng.normal(0, 1.5, (B, T, H, dv)), rng.normal(1, 0.3, H * dv), rng.normal(0, 1, (B, T, H, dv))


def test_out_norm_invariants():
    o, g, _ = _case()
    B, T, H, dv = o.shape
    # gain = 1, eps = 0: every token's output has unit root mean square over its H*dv channels
    y = le.out_norm(o, np.ones(H * dv), 0.0).reshape(B, T, -1)
    assert np.max(np.abs(np.sqrt(np.mean(y * y, axis=-1)) - 1.0)) < 1e-14
    # scale invariance (eps = 0) and linearity in the gain
    assert np.max(np.abs(le.out_norm(3.7 * o, g, 0.0) - le.out_norm(o, g, 0.0))) < 1e-13
    assert np.max(np.abs(le.out_norm(o, 2 * g, 1e-6) - 2 * le.out_norm(o, g, 1e-6))) < 1e-13
    # the normalisation couples heads: it is over all H*dv channels of a token, not per head (reshape, l.194)
    o2 = o.copy()
    o2[:, :, 0] *= 10.0
    assert np.max(np.abs(le.out_norm(o2, g, 0.0)[:, :, 1] - le.out_norm(o, g, 0.0)[:, :, 1])) > 1e-2
    # a constant token x = c: y = sign(c) gain
    y = le.out_norm(np.full((1, 1, H, dv), -2.5), g, 0.0).reshape(-1)
    assert np.max(np.abs(y + g)) < 1e-14
    # eps enters as sqrt(mean + eps): a zero token maps to zero, not NaN
    assert np.all(le.out_norm(np.zeros((1, 1, H, dv)), g, 1e-6) == 0.0)


def test_out_norm_bwd_central_differences_and_orthogonality():
    o, g, dy = _case(1)
    eps = 1e-5
    do, dg = le.out_norm_bwd(o, g, eps, dy)
    f = lambda oo, gg: float(np.sum(le.out_norm(oo, gg, eps) * dy))
    rng = np.random.default_rng(2)
    h = 1e-6
    for _ in range(3):   # directional derivatives along random directions
        u, w = rng.normal(0, 1, o.shape), rng.normal(0, 1, g.shape)
        fd_o = (f(o + h * u, g) - f(o - h * u, g)) / (2 * h)
        fd_g = (f(o, g + h * w) - f(o, g - h * w)) / (2 * h)
        assert abs(fd_o - np.sum(do * u)) < 1e-7 * max(1.0, abs(fd_o))
        assert abs(fd_g - np.sum(dg * w)) < 1e-7 * max(1.0, abs(fd_g))
    # eps = 0: y does not change along o (scale invariance), so the gradient is orthogonal to o token by token
    do0, _ = le.out_norm_bwd(o, g, 0.0, dy)
    B, T, H, dv = o.shape
    assert np.max(np.abs(np.sum((do0 * o).reshape(B, T, -1), axis=-1))) < 1e-12

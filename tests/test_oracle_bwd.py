"""P8: pins for the oracle's backward (Alg. 4/5): central finite differences through the
oracle's own *forward* (which P1-P6 pin), torch autograd through a separately written
per-token recurrence, and a dot-product (adjoint) test at config-0 size.  No GPU.
"""
import numpy as np
import pytest

from paper_2606_27229_b200 import synth
from tests import ref_np
from tests.test_oracle_pins import perturbed, rel, shape_of, small_cfg

IN_NAMES = ["q", "k", "v", "f", "bx", "wx", "beta", "A", "tau", "Ub", "Uw", "Vb", "Vw", "S0"]


def _loss(oracle, s, x, dO, dSf):
    O, Sf = oracle.fwd(s, x)
    return float((O * dO).sum() + (Sf * dSf).sum())


@pytest.mark.parametrize("l2norm", [1, 0])
def test_finite_differences_every_tensor(oracle, l2norm):
    """Central differences (h=1e-6, fp64) for each of the 14 inputs separately, per tensor
    (l.470, l.819: an aggregate check would miss a dw/d-delta mix-up)."""
    cfg = small_cfg(B=1, H=2, T=12, L=4, dk=5, dv=3, r=2, wstd=0.6, s0_std=0.5, qk_l2norm=l2norm)
    x = {n: (None if a is None else a.astype(np.float64))
         for n, a in perturbed(cfg, with_decay_params=True).items()}
    s = shape_of(oracle, cfg, scale=0.9)
    ct = synth.make_cotangents(cfg)
    dO, dSf = ct["dO"].astype(np.float64), ct["dS_final"].astype(np.float64) * 30.0
    g = oracle.bwd(s, x, dO, dSf)
    rng = np.random.default_rng(5)
    h = 1e-6
    for n in IN_NAMES:
        a = x[n]
        fd = np.zeros_like(a)
        idxs = list(np.ndindex(a.shape))
        if len(idxs) > 60:
            idxs = [idxs[i] for i in rng.choice(len(idxs), 60, replace=False)]
        an = np.zeros_like(a)
        for idx in idxs:
            xp, xm = dict(x), dict(x)
            ap, am = a.copy(), a.copy()
            ap[idx] += h
            am[idx] -= h
            xp[n], xm[n] = ap, am
            fd[idx] = (_loss(oracle, s, xp, dO, dSf) - _loss(oracle, s, xm, dO, dSf)) / (2 * h)
            an[idx] = g["d" + n][idx]
        err = np.abs(fd - an).max() / max(np.abs(g["d" + n]).max(), 1e-30)
        assert err < 2e-6, (n, err)


@pytest.mark.parametrize("L", [1, 4, 16])
def test_autograd_every_tensor(oracle, L):
    """torch autograd (fp64) through the per-token recurrence of tests/ref_np.py vs the
    oracle's reverse scan, per tensor, incl. dA, dtau, dS0 and the weight gradients."""
    cfg = small_cfg(B=2, H=2, T=16, L=L, dk=6, dv=4, r=3, wstd=0.5, s0_std=0.4)
    x = perturbed(cfg, with_decay_params=True)
    s = shape_of(oracle, cfg, scale=1.1)
    ct = synth.make_cotangents(cfg)
    g = oracle.bwd(s, x, ct["dO"], ct["dS_final"])
    ga = ref_np.torch_autograd_grads(s, x, ct["dO"], ct["dS_final"], L)
    for n in IN_NAMES:
        assert rel(g["d" + n], ga["d" + n]) < 1e-10, n


def test_autograd_optional_args_absent(oracle):
    """A = tau = S0 = NULL and dS_final = NULL behave as zeros."""
    cfg = small_cfg(B=1, H=2, T=8, L=4, dk=4, dv=3, r=2, s0_std=0.0)
    x = perturbed(cfg)
    s = shape_of(oracle, cfg)
    ct = synth.make_cotangents(cfg)
    g = oracle.bwd(s, x, ct["dO"], None)
    ga = ref_np.torch_autograd_grads(s, x, ct["dO"], np.zeros_like(ct["dS_final"]), 4)
    for n in IN_NAMES:
        assert rel(g["d" + n], ga["d" + n]) < 1e-10, n


def test_dot_product_adjoint_config0(oracle):
    """<dO, J dx> == <J^T dO, dx> at config-0 size (B=1,H=1,T=256,L=64,d=64,r=8) for a random
    direction on all inputs at once; J dx by central differences."""
    cfg = synth.CFG0
    x = {n: (None if a is None else a.astype(np.float64)) for n, a in synth.make_inputs(cfg).items()}
    s = shape_of(oracle, cfg)
    ct = synth.make_cotangents(cfg)
    dO, dSf = ct["dO"].astype(np.float64), ct["dS_final"].astype(np.float64)
    g = oracle.bwd(s, x, dO, dSf)
    rng = np.random.default_rng(9)
    names = [n for n in IN_NAMES if x.get(n) is not None]
    dx = {n: rng.standard_normal(x[n].shape) for n in names}
    h = 1e-6
    xp = dict(x)
    xm = dict(x)
    for n in names:
        xp[n] = x[n] + h * dx[n]
        xm[n] = x[n] - h * dx[n]
    lhs = (_loss(oracle, s, xp, dO, dSf) - _loss(oracle, s, xm, dO, dSf)) / (2 * h)
    rhs = sum(float((g["d" + n] * dx[n]).sum()) for n in names)
    assert abs(lhs - rhs) / abs(rhs) < 1e-6

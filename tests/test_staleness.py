"""The staleness measurement of oracle/staleness.py (Table 4 l.497-510, Prop. 14 l.377-383)
on a tiny case: what must hold whatever the numbers are."""
import numpy as np

from oracle import staleness
from paper_2606_27229_b200 import synth


def _cfg(wstd):
    return synth.Config("t", B=1, H=2, T=128, L=16, dk=16, dv=12, r=4, dtype="f32", wstd=wstd, seed=5)


def test_no_content_gates_no_staleness(oracle):
    """With zero gate projections the chunk length is irrelevant (l.143): deviation exactly ~0 for every L."""
    d = staleness.deviations(_cfg(0.0), Ls=(1, 16, 64))
    for L, v in d.items():
        assert max(v) < 1e-12, (L, v)


def test_staleness_grows_with_gate_strength_and_is_second_order(oracle):
    """The deviation vanishes with the content weights; U and V both scale with wstd, so it scales ~ wstd^2 (Prop. 14:
    the bound is linear in the gate's sensitivity to the state, itself a product of the two projections)."""
    d1 = staleness.deviations(_cfg(0.05), Ls=(16,))[16][0]
    d2 = staleness.deviations(_cfg(0.1), Ls=(16,))[16][0]
    assert 0 < d1 < d2
    assert 3.0 < d2 / d1 < 5.0, d2 / d1
    assert staleness.deviations(_cfg(0.1), Ls=(1,))[1][0] == 0.0

"""Staleness of the chunk-level gate readout, measured with the fp64 oracle on synthetic inputs.

TEST / MEASUREMENT INFRASTRUCTURE: calls only oracle/ and the seeded input generator; nothing of the CUDA path.

CARVE's gates read the state once per chunk, S_{c-1} (Eq. 7 l.134-136), instead of the exact per-token
S_{t-1}; Prop. 14 (l.377-383) bounds the deviation and Table 4 (l.497-510) reports 0.18 %, flat in L, on trained
125M activations.  Those activations are not available here, so this script measures the same quantity on the
synthetic config-2 distributions (gate projections ~N(0, 0.1^2): content gates active) -- context, not a
reproduction: the chunked definition at L in {16, 32, 64, 128} against the same definition at L = 1, where the gate of
token t reads S_{t-1} exactly (the oracle's L = 1 mode is pinned by tests/test_oracle_pins.py::test_L1_is_exact_content_gating).

    python -m oracle.staleness [--B 1 --H 4 --T 2048 --wstd 0.1]      # prints a markdown table

Reported per L: ||O_L - O_1||_F / ||O_1||_F (the paper's "relative deviation"), the max-norm version of it, and the
same two for the final state.
"""
from __future__ import annotations

import argparse

import numpy as np

from oracle import carve_oracle as orc
from paper_2606_27229_b200 import synth


def deviations(cfg: synth.Config, Ls=(16, 32, 64, 128)):
    """Returns {L: (fro_O, max_O, fro_S, max_S)} of the chunked definition at chunk length L against L = 1."""
    x = synth.make_inputs(cfg)
    base = dict(B=cfg.B, H=cfg.H, T=cfg.T, dk=cfg.dk, dv=cfg.dv, r=cfg.r, qk_l2norm=cfg.qk_l2norm, scale=cfg.scale, eps=cfg.eps)
    O1, S1 = orc.fwd(orc.Shape(L=1, **base), x)
    out = {}
    for L in Ls:
        OL, SL = orc.fwd(orc.Shape(L=L, **base), x)
        out[L] = (float(np.linalg.norm(OL - O1) / np.linalg.norm(O1)),
                  float(np.max(np.abs(OL - O1)) / np.max(np.abs(O1))),
                  float(np.linalg.norm(SL - S1) / max(np.linalg.norm(S1), 1e-300)),
                  float(np.max(np.abs(SL - S1)) / max(np.max(np.abs(S1)), 1e-300)))
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--B", type=int, default=1)
    ap.add_argument("--H", type=int, default=4)
    ap.add_argument("--T", type=int, default=2048)
    ap.add_argument("--wstd", type=float, nargs="*", default=[0.02, 0.1, 0.3])
    args = ap.parse_args()
    print("| gate projections | L | rel. deviation of O (Frobenius) | (max norm) | of S_final (Frobenius) | (max norm) |")
    print("|---|---|---|---|---|---|")
    for w in args.wstd:
        cfg = synth.CFG2[64].with_(B=args.B, H=args.H, T=args.T, wstd=w, dtype="f32")
        for L, d in deviations(cfg).items():
            print(f"| N(0, {w}^2) | {L} | {100 * d[0]:.3f} % | {100 * d[1]:.3f} % | {100 * d[2]:.3f} % | {100 * d[3]:.3f} % |")


if __name__ == "__main__":
    main()

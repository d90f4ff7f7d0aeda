"""Independent restatements used ONLY to pin the oracle (tests/test_oracle_*.py).

Everything here is written from the paper's *per-token* equations (Eq. 5 l.108, Eq. 7-9
l.134-151) or from a dense library solve -- never from oracle/carve_oracle.c's chunked WY
code.  numpy / torch CPU, float64.
"""
from __future__ import annotations

import numpy as np


def _sig(x):
    return 1.0 / (1.0 + np.exp(-x))


def _softplus(x):
    return np.logaddexp(0.0, x)


def _prep(x, s, b, h):
    """Per-chain views: normalised q,k, decay g, raw gates."""
    q = np.asarray(x["q"], np.float64)[b, :, h]
    k = np.asarray(x["k"], np.float64)[b, :, h]
    if s.qk_l2norm:
        q = q / np.sqrt((q * q).sum(-1, keepdims=True) + s.eps)
        k = k / np.sqrt((k * k).sum(-1, keepdims=True) + s.eps)
    A = 0.0 if x.get("A") is None else np.asarray(x["A"], np.float64)[h]
    tau = 0.0 if x.get("tau") is None else np.asarray(x["tau"], np.float64)[h]
    g = -np.exp(A) * _softplus(np.asarray(x["f"], np.float64)[b, :, h] + tau)
    return (q, k, np.asarray(x["v"], np.float64)[b, :, h], g,
            np.asarray(x["bx"], np.float64)[b, :, h], np.asarray(x["wx"], np.float64)[b, :, h],
            np.asarray(x["beta"], np.float64)[b, :, h])


def recurrence_memory_blind(s, x):
    """Key-axis-gated delta rule with NO content path at all (Thm 1's memory-blind class,
    l.206): S_t = S_{t-1} diag(exp(g) (1-sigma(bx))) + beta (sigma(wx) v - S_{t-1} k) k^T."""
    O = np.zeros((s.B, s.T, s.H, s.dv))
    Sf = np.zeros((s.B, s.H, s.dv, s.dk))
    for b in range(s.B):
        for h in range(s.H):
            q, k, v, g, bx, wx, beta = _prep(x, s, b, h)
            S = np.zeros((s.dv, s.dk)) if x.get("S0") is None else np.array(x["S0"][b, h], np.float64)
            for t in range(s.T):
                a = np.exp(g[t]) * (1.0 - _sig(bx[t]))
                u = beta[t] * (_sig(wx[t]) * v[t] - S @ k[t])
                S = S * a[None, :] + np.outer(u, k[t])
                O[b, t, h] = s.scale * (S @ q[t])
            Sf[b, h] = S
    return O, Sf


def recurrence_content(s, x, L):
    """Eq. 5 token by token; the gates of token t read the state at the start of its
    chunk of length L (Eq. 7-8).  L=1 is exact per-token content gating."""
    Ub, Uw = np.asarray(x["Ub"], np.float64), np.asarray(x["Uw"], np.float64)
    Vb, Vw = np.asarray(x["Vb"], np.float64), np.asarray(x["Vw"], np.float64)
    O = np.zeros((s.B, s.T, s.H, s.dv))
    Sf = np.zeros((s.B, s.H, s.dv, s.dk))
    for b in range(s.B):
        for h in range(s.H):
            q, k, v, g, bx, wx, beta = _prep(x, s, b, h)
            S = np.zeros((s.dv, s.dk)) if x.get("S0") is None else np.array(x["S0"][b, h], np.float64)
            Sc = S
            for t in range(s.T):
                if t % L == 0:
                    Sc = S.copy()
                m = Sc @ q[t]                       # per-token readout m_{c,t} = S_{c-1} q_t (l.50)
                tb, tw = np.tanh(Ub @ m), np.tanh(Uw @ m)
                bt = _sig(bx[t] + Vb @ tb)
                wt = _sig(wx[t] + Vw @ tw)
                a = np.exp(g[t]) * (1.0 - bt)
                u = beta[t] * (wt * v[t] - S @ k[t])
                S = S * a[None, :] + np.outer(u, k[t])
                O[b, t, h] = s.scale * (S @ q[t])
            Sf[b, h] = S
    return O, Sf


def chunk_dense_solve(s, x):
    """Chunked form with the coupling matrix built by broadcasting and the triangular
    system solved by numpy's dense LU (np.linalg.solve)."""
    Ub, Uw = np.asarray(x["Ub"], np.float64), np.asarray(x["Uw"], np.float64)
    Vb, Vw = np.asarray(x["Vb"], np.float64), np.asarray(x["Vw"], np.float64)
    L = s.L
    O = np.zeros((s.B, s.T, s.H, s.dv))
    Sf = np.zeros((s.B, s.H, s.dv, s.dk))
    for b in range(s.B):
        for h in range(s.H):
            q, k, v, g, bx, wx, beta = _prep(x, s, b, h)
            S = np.zeros((s.dv, s.dk)) if x.get("S0") is None else np.array(x["S0"][b, h], np.float64)
            for c in range(s.T // L):
                sl = slice(c * L, (c + 1) * L)
                qc, kc, vc = q[sl], k[sl], v[sl]
                tt_b = np.tanh((qc @ S.T) @ Ub.T)
                tt_w = np.tanh((qc @ S.T) @ Uw.T)
                bg = _sig(bx[sl] + tt_b @ Vb.T)
                wg = _sig(wx[sl] + tt_w @ Vw.T)
                lg = np.cumsum(g[sl] + np.log1p(-bg), axis=0)
                lgm1 = np.vstack([np.zeros((1, s.dk)), lg[:-1]])
                # A[t,s] = sum_j k_t k_s exp(lg_{t-1} - lg_s), s<t
                Efull = np.exp(np.minimum(lgm1[:, None, :] - lg[None, :, :], 50.0))
                Am = np.tril(np.einsum("tj,sj,tsj->ts", kc, kc, Efull), -1)
                R = wg * vc - (kc * np.exp(lgm1)) @ S.T
                bt = beta[sl]
                U = np.linalg.solve(np.eye(L) + bt[:, None] * Am, bt[:, None] * R)
                Pfull = np.exp(np.minimum(lg[:, None, :] - lg[None, :, :], 50.0))
                P = np.tril(np.einsum("tj,sj,tsj->ts", qc, kc, Pfull), 0)
                O[b, sl, h] = s.scale * ((qc * np.exp(lg)) @ S.T + P @ U)
                S = S * np.exp(lg[-1])[None, :] + U.T @ (kc * np.exp(lg[-1][None, :] - lg))
            Sf[b, h] = S
    return O, Sf


def torch_autograd_grads(s, x, dO, dSf, L):
    """Gradients of <dO,O> + <dS_final,S_final> by torch autograd through the per-token
    recurrence (float64, CPU)."""
    import torch

    names = ["q", "k", "v", "f", "bx", "wx", "beta", "A", "tau", "Ub", "Uw", "Vb", "Vw", "S0"]
    tt = {}
    for n in names:
        a = x.get(n)
        if a is None:
            shp = {"A": (s.H, s.dk), "tau": (s.H, s.dk), "S0": (s.B, s.H, s.dv, s.dk)}[n]
            a = np.zeros(shp)
        tt[n] = torch.tensor(np.asarray(a, np.float64), requires_grad=True)
    q, k = tt["q"], tt["k"]
    if s.qk_l2norm:
        q = q / torch.sqrt((q * q).sum(-1, keepdim=True) + s.eps)
        k = k / torch.sqrt((k * k).sum(-1, keepdim=True) + s.eps)
    g = -torch.exp(tt["A"])[None, None] * torch.nn.functional.softplus(tt["f"] + tt["tau"][None, None])
    loss = 0.0
    dO_t, dSf_t = torch.tensor(np.asarray(dO, np.float64)), torch.tensor(np.asarray(dSf, np.float64))
    for b in range(s.B):
        for h in range(s.H):
            S = tt["S0"][b, h]
            Sc = S
            for t in range(s.T):
                if t % L == 0:
                    Sc = S
                m = Sc @ q[b, t, h]
                bt = torch.sigmoid(tt["bx"][b, t, h] + tt["Vb"] @ torch.tanh(tt["Ub"] @ m))
                wt = torch.sigmoid(tt["wx"][b, t, h] + tt["Vw"] @ torch.tanh(tt["Uw"] @ m))
                a = torch.exp(g[b, t, h]) * (1.0 - bt)
                u = tt["beta"][b, t, h] * (wt * tt["v"][b, t, h] - S @ k[b, t, h])
                S = S * a[None, :] + torch.outer(u, k[b, t, h])
                loss = loss + s.scale * (dO_t[b, t, h] * (S @ q[b, t, h])).sum()
            loss = loss + (dSf_t[b, h] * S).sum()
    loss.backward()
    out = {"d" + n: tt[n].grad.numpy() for n in names}
    return out

"""ctypes binding of the fp64 CPU oracle (oracle/carve_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It imports
nothing from paper_2606_27229_b200/ and the CUDA path imports nothing from here.

The arithmetic lives in carve_oracle.c (each step cites PAPER.md); this file only
builds the shared object with gcc and marshals numpy float64 arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "carve_oracle.c")
_SO = os.path.join(_HERE, "libcarve_oracle.so")


def build(force: bool = False) -> str:
    """Compile carve_oracle.c -> libcarve_oracle.so: gcc -O3 -fopenmp.  No -march=native (the object built on the CPU box
    also has to run on the host cores of the GPU box) and no fast-math (the fp64 arithmetic is that of the source)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O3", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-Wall", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _SO)
    return _SO


class _Params(ctypes.Structure):
    _fields_ = [
        ("B", ctypes.c_int), ("H", ctypes.c_int), ("T", ctypes.c_int), ("L", ctypes.c_int),
        ("dk", ctypes.c_int), ("dv", ctypes.c_int), ("r", ctypes.c_int),
        ("qk_l2norm", ctypes.c_int), ("scale", ctypes.c_double), ("eps", ctypes.c_double),
    ]


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.carve_ref_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(_load().carve_ref_num_threads())


@dataclass
class Shape:
    B: int
    H: int
    T: int
    L: int
    dk: int
    dv: int
    r: int
    qk_l2norm: int = 1
    scale: float = 1.0
    eps: float = 1e-6

    def c(self) -> _Params:
        return _Params(self.B, self.H, self.T, self.L, self.dk, self.dv, self.r,
                       self.qk_l2norm, self.scale, self.eps)


def _p(a, shape=None):
    if a is None:
        return None
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        assert a.shape == tuple(shape), (a.shape, shape)
    return a


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _inputs(s: Shape, x: dict):
    B, H, T, dk, dv, r = s.B, s.H, s.T, s.dk, s.dv, s.r
    arrs = [
        _p(x["q"], (B, T, H, dk)), _p(x["k"], (B, T, H, dk)), _p(x["v"], (B, T, H, dv)),
        _p(x["f"], (B, T, H, dk)), _p(x["bx"], (B, T, H, dk)), _p(x["wx"], (B, T, H, dv)),
        _p(x["beta"], (B, T, H)),
        _p(x.get("A"), (H, dk)) if x.get("A") is not None else None,
        _p(x.get("tau"), (H, dk)) if x.get("tau") is not None else None,
        _p(x["Ub"], (r, dv)), _p(x["Uw"], (r, dv)), _p(x["Vb"], (dk, r)), _p(x["Vw"], (dv, r)),
        _p(x.get("S0"), (B, H, dv, dk)) if x.get("S0") is not None else None,
    ]
    return arrs


def _fwd(fn_name: str, s: Shape, x: dict):
    lib = _load()
    arrs = _inputs(s, x)
    O = np.empty((s.B, s.T, s.H, s.dv), dtype=np.float64)
    Sf = np.empty((s.B, s.H, s.dv, s.dk), dtype=np.float64)
    p = s.c()
    rc = getattr(lib, fn_name)(ctypes.byref(p), *[_ptr(a) for a in arrs], _ptr(O), _ptr(Sf))
    if rc != 0:
        raise RuntimeError(f"{fn_name} failed with code {rc}")
    return O, Sf


def fwd(s: Shape, x: dict):
    """Chunked definition (Alg. 1 + Alg. 2).  Returns (O, S_final)."""
    return _fwd("carve_ref_fwd", s, x)


def fwd_sequential(s: Shape, x: dict):
    """Per-token Eq. 5 with chunk-stale gates.  Returns (O, S_final)."""
    return _fwd("carve_ref_fwd_sequential", s, x)


GRAD_NAMES = ("dq", "dk", "dv", "df", "dbx", "dwx", "dbeta", "dA", "dtau",
              "dUb", "dUw", "dVb", "dVw", "dS0")


def bwd(s: Shape, x: dict, dO, dS_final=None) -> dict:
    """Per-token adjoint (Alg. 4 + Alg. 5 glue).  Returns a dict of the 14 gradients."""
    lib = _load()
    arrs = _inputs(s, x)
    B, H, T, dk, dv, r = s.B, s.H, s.T, s.dk, s.dv, s.r
    dO = _p(dO, (B, T, H, dv))
    dSf = _p(dS_final, (B, H, dv, dk)) if dS_final is not None else None
    out = {
        "dq": np.empty((B, T, H, dk)), "dk": np.empty((B, T, H, dk)), "dv": np.empty((B, T, H, dv)),
        "df": np.empty((B, T, H, dk)), "dbx": np.empty((B, T, H, dk)), "dwx": np.empty((B, T, H, dv)),
        "dbeta": np.empty((B, T, H)), "dA": np.empty((H, dk)), "dtau": np.empty((H, dk)),
        "dUb": np.empty((r, dv)), "dUw": np.empty((r, dv)), "dVb": np.empty((dk, r)),
        "dVw": np.empty((dv, r)), "dS0": np.empty((B, H, dv, dk)),
    }
    p = s.c()
    rc = lib.carve_ref_bwd(ctypes.byref(p), *[_ptr(a) for a in arrs], _ptr(dO), _ptr(dSf),
                           *[_ptr(out[n]) for n in GRAD_NAMES])
    if rc != 0:
        raise RuntimeError(f"carve_ref_bwd failed with code {rc}")
    return out

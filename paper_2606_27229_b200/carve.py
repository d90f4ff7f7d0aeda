"""Thin Python binding of include/carve.h (ctypes).  Argument marshalling only: every step of
the operator runs inside csrc/libcarve.so.  There is no fallback of any kind -- if the shared
library is missing or a call returns a non-zero status this module raises.

Arguments are objects with a `.data_ptr()` method (torch tensors: CUDA tensors for carve_fwd /
carve_bwd, pinned CPU tensors for carve_fwd_bwd_host), raw integer addresses, or None where the
header allows NULL.  The caller owns all memory; nothing is allocated here.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libcarve.so")

CARVE_F32, CARVE_BF16 = 0, 1
CARVE_PATH_AUTO, CARVE_PATH_SIMT, CARVE_PATH_TENSOR = 0, 1, 2

# Every symbol include/carve.h declares (tests check the library exports them all).
SYMBOLS = ("carve_workspace_bytes", "carve_fwd", "carve_bwd", "carve_step", "carve_host_arena_bytes", "carve_fwd_bwd_host",
           "carve_host_ctx_create", "carve_host_ctx_destroy", "carve_fwd_bwd_host_ctx",
           "carve_fwd_bwd_static", "carve_static_scratch_bytes", "carve_step_varlen",
           "carve_silu_qkv_fwd", "carve_silu_qkv_bwd", "carve_out_norm_fwd", "carve_out_norm_bwd",
           "carve_out_norm_workspace_bytes",
           "carve_num_launches", "carve_resolved_path", "carve_status_string", "carve_version")


class CarveError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"carve status {status}: {msg}")
        self.status = status


class _Params(ctypes.Structure):
    _fields_ = [("B", ctypes.c_int), ("H", ctypes.c_int), ("T", ctypes.c_int), ("L", ctypes.c_int),
                ("dk", ctypes.c_int), ("dv", ctypes.c_int), ("r", ctypes.c_int), ("dtype", ctypes.c_int),
                ("qk_l2norm", ctypes.c_int), ("scale", ctypes.c_float), ("eps", ctypes.c_float),
                ("path", ctypes.c_int)]


@dataclass
class Params:
    B: int
    H: int
    T: int
    L: int
    dk: int
    dv: int
    r: int
    dtype: int = CARVE_BF16
    qk_l2norm: int = 1
    scale: float = 1.0
    eps: float = 1e-6
    path: int = CARVE_PATH_AUTO

    def c(self) -> _Params:
        return _Params(self.B, self.H, self.T, self.L, self.dk, self.dv, self.r, self.dtype, self.qk_l2norm,
                       self.scale, self.eps, self.path)


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen csrc/libcarve.so (built by `python -m paper_2606_27229_b200.build`); raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2606_27229_b200.build` "
                "(there is no CPU or PyTorch fallback)")
        lib = ctypes.CDLL(LIB_PATH)
        vp, sz, ci = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int
        pp = ctypes.POINTER(_Params)
        lib.carve_workspace_bytes.restype = sz
        lib.carve_workspace_bytes.argtypes = [pp, ci]
        lib.carve_host_arena_bytes.restype = sz
        lib.carve_host_arena_bytes.argtypes = [pp, ci]
        lib.carve_num_launches.restype = ci
        lib.carve_num_launches.argtypes = [pp, ci]
        lib.carve_resolved_path.restype = ci
        lib.carve_resolved_path.argtypes = [pp, ci]
        lib.carve_status_string.restype = ctypes.c_char_p
        lib.carve_status_string.argtypes = [ci]
        lib.carve_version.restype = ctypes.c_char_p
        lib.carve_fwd.restype = ci
        lib.carve_fwd.argtypes = [pp] + [vp] * 16 + [vp, sz, vp]
        lib.carve_step.restype = ci
        lib.carve_step.argtypes = [pp] + [vp] * 15 + [vp]
        lib.carve_step_varlen.restype = ci
        lib.carve_step_varlen.argtypes = [pp] + [vp] * 15 + [vp, vp]
        lib.carve_silu_qkv_fwd.restype = ci
        lib.carve_silu_qkv_fwd.argtypes = [pp] + [vp] * 6 + [vp]
        lib.carve_silu_qkv_bwd.restype = ci
        lib.carve_silu_qkv_bwd.argtypes = [pp] + [vp] * 6 + [vp]
        lib.carve_out_norm_fwd.restype = ci
        lib.carve_out_norm_fwd.argtypes = [pp, vp, vp, ctypes.c_float, vp, vp]
        lib.carve_out_norm_workspace_bytes.restype = sz
        lib.carve_out_norm_workspace_bytes.argtypes = [pp]
        lib.carve_out_norm_bwd.restype = ci
        lib.carve_out_norm_bwd.argtypes = [pp, vp, vp, ctypes.c_float, vp, vp, vp, vp, sz, vp]
        lib.carve_bwd.restype = ci
        lib.carve_bwd.argtypes = [pp] + [vp] * 30 + [vp, sz, vp]
        lib.carve_fwd_bwd_host.restype = ci
        lib.carve_fwd_bwd_host.argtypes = [pp, ci] + [vp] * 32 + [vp, sz, vp]
        lib.carve_fwd_bwd_host_ctx.restype = ci
        lib.carve_fwd_bwd_host_ctx.argtypes = [vp, pp, ci] + [vp] * 32 + [vp, sz, vp]
        lib.carve_host_ctx_create.restype = ci
        lib.carve_host_ctx_create.argtypes = [ctypes.POINTER(vp)]
        lib.carve_fwd_bwd_static.restype = ci
        lib.carve_fwd_bwd_static.argtypes = [pp] + [vp] * 32 + [vp]
        lib.carve_static_scratch_bytes.restype = sz
        lib.carve_static_scratch_bytes.argtypes = []
        lib.carve_host_ctx_destroy.restype = None
        lib.carve_host_ctx_destroy.argtypes = [vp]
        _lib = lib
    return _lib


def _ptr(x):
    if x is None:
        return None
    if isinstance(x, int):
        return ctypes.c_void_p(x)
    return ctypes.c_void_p(x.data_ptr())


def _nbytes(x) -> int:
    return 0 if x is None else x.numel() * x.element_size()


def _check(status: int):
    if status != 0:
        raise CarveError(status, load_library().carve_status_string(status).decode())


def carve_version() -> str:
    return load_library().carve_version().decode()


def carve_workspace_bytes(p: Params, need_bwd: bool = True) -> int:
    cp = p.c()
    return int(load_library().carve_workspace_bytes(ctypes.byref(cp), int(need_bwd)))


def carve_host_arena_bytes(p: Params, with_bwd: bool = True) -> int:
    cp = p.c()
    return int(load_library().carve_host_arena_bytes(ctypes.byref(cp), int(with_bwd)))


def carve_num_launches(p: Params, bwd: bool) -> int:
    cp = p.c()
    return int(load_library().carve_num_launches(ctypes.byref(cp), int(bwd)))


def carve_resolved_path(p: Params, bwd: bool) -> int:
    cp = p.c()
    return int(load_library().carve_resolved_path(ctypes.byref(cp), int(bwd)))


_FWD_IN = ("q", "k", "v", "f", "bx", "wx", "beta", "A", "tau", "Ub", "Uw", "Vb", "Vw", "S0")
_GRADS = ("dq", "dk", "dv", "df", "dbx", "dwx", "dbeta", "dA", "dtau", "dUb", "dUw", "dVb", "dVw", "dS0")


def carve_fwd(p: Params, x: dict, O, S_final, workspace=None, stream: int = 0) -> None:
    """carve_fwd of carve.h.  `x` maps the names q,k,v,f,bx,wx,beta,A,tau,Ub,Uw,Vb,Vw,S0 to device
    tensors (A, tau, S0 may be None); O, S_final are written; workspace (a device byte tensor of
    carve_workspace_bytes(p) bytes) is filled for carve_bwd, or None for inference."""
    cp = p.c()
    _check(load_library().carve_fwd(ctypes.byref(cp), *[_ptr(x.get(n)) for n in _FWD_IN], _ptr(O), _ptr(S_final),
                                    _ptr(workspace), _nbytes(workspace), ctypes.c_void_p(stream)))


def carve_step(p: Params, x: dict, S, O, stream: int = 0) -> None:
    """carve_step of carve.h: p.T = n <= 16 new tokens per sequence; `x` as for carve_fwd (S0 is not used);
    S [B,H,dv,dk] float32 is read and overwritten in place; O [B,n,H,dv] is written."""
    cp = p.c()
    _check(load_library().carve_step(ctypes.byref(cp), *[_ptr(x.get(n)) for n in _FWD_IN[:-1]], _ptr(S), _ptr(O),
                                     ctypes.c_void_p(stream)))


def carve_silu_qkv_fwd(p: Params, qx, kx, vx, q, k, v, stream: int = 0) -> None:
    """carve_silu_qkv_fwd of carve.h: q, k, v = SiLU(qx), SiLU(kx), SiLU(vx) in one launch (None pairs are skipped)."""
    cp = p.c()
    _check(load_library().carve_silu_qkv_fwd(ctypes.byref(cp), _ptr(qx), _ptr(kx), _ptr(vx), _ptr(q), _ptr(k), _ptr(v),
                                             ctypes.c_void_p(stream)))


def carve_silu_qkv_bwd(p: Params, qx, kx, vx, dq, dk, dv, stream: int = 0) -> None:
    """carve_silu_qkv_bwd of carve.h: dq, dk, dv (gradients w.r.t. q, k, v) become those w.r.t. qx, kx, vx, in place."""
    cp = p.c()
    _check(load_library().carve_silu_qkv_bwd(ctypes.byref(cp), _ptr(qx), _ptr(kx), _ptr(vx), _ptr(dq), _ptr(dk), _ptr(dv),
                                             ctypes.c_void_p(stream)))


def carve_out_norm_workspace_bytes(p: Params) -> int:
    cp = p.c()
    return int(load_library().carve_out_norm_workspace_bytes(ctypes.byref(cp)))


def carve_out_norm_fwd(p: Params, o, gain, eps: float, y, stream: int = 0) -> None:
    """carve_out_norm_fwd of carve.h: y = RMSNorm over the H*dv channels of every token of o, times gain."""
    cp = p.c()
    _check(load_library().carve_out_norm_fwd(ctypes.byref(cp), _ptr(o), _ptr(gain), ctypes.c_float(eps), _ptr(y),
                                             ctypes.c_void_p(stream)))


def carve_out_norm_bwd(p: Params, o, gain, eps: float, dy, d_o, dgain, workspace, stream: int = 0) -> None:
    """carve_out_norm_bwd of carve.h."""
    cp = p.c()
    _check(load_library().carve_out_norm_bwd(ctypes.byref(cp), _ptr(o), _ptr(gain), ctypes.c_float(eps), _ptr(dy), _ptr(d_o),
                                             _ptr(dgain), _ptr(workspace), _nbytes(workspace), ctypes.c_void_p(stream)))


def carve_step_varlen(p: Params, x: dict, S, O, cu_seqlens, stream: int = 0) -> None:
    """carve_step_varlen of carve.h: packed token tensors [N,H,d] with N = cu_seqlens[B]; `cu_seqlens` is a device int32
    tensor of B + 1 entries; p.T = the maximum number of new tokens of any sequence (<= 16)."""
    cp = p.c()
    _check(load_library().carve_step_varlen(ctypes.byref(cp), *[_ptr(x.get(n)) for n in _FWD_IN[:-1]], _ptr(S), _ptr(O),
                                            _ptr(cu_seqlens), ctypes.c_void_p(stream)))


def carve_bwd(p: Params, x: dict, dO, dS_final, grads: dict, workspace, stream: int = 0) -> None:
    """carve_bwd of carve.h.  `grads` maps dq,dk,dv,df,dbx,dwx,dbeta,dA,dtau,dUb,dUw,dVb,dVw,dS0 to
    preallocated device tensors (dA, dtau may be None); they are overwritten."""
    cp = p.c()
    _check(load_library().carve_bwd(ctypes.byref(cp), *[_ptr(x.get(n)) for n in _FWD_IN], _ptr(dO), _ptr(dS_final),
                                    *[_ptr(grads.get(n)) for n in _GRADS], _ptr(workspace), _nbytes(workspace),
                                    ctypes.c_void_p(stream)))


def carve_static_scratch_bytes() -> int:
    return int(load_library().carve_static_scratch_bytes())


def carve_fwd_bwd_static(p: Params, x: dict, O, S_final, dO, dS_final, grads: dict, stream: int = 0) -> None:
    """carve_fwd_bwd_static of carve.h: training forward + backward with the workspace in the library's static device
    array (no allocation; problems beyond carve_static_scratch_bytes() raise CarveError with CARVE_ERR_STATIC_LIMIT)."""
    cp = p.c()
    _check(load_library().carve_fwd_bwd_static(ctypes.byref(cp), *[_ptr(x.get(n)) for n in _FWD_IN], _ptr(O), _ptr(S_final),
                                               _ptr(dO), _ptr(dS_final), *[_ptr(grads.get(n)) for n in _GRADS],
                                               ctypes.c_void_p(stream)))


def carve_host_ctx_create() -> ctypes.c_void_p:
    """carve_host_ctx_create of carve.h: the side streams and events of the host entry point, owned by the caller."""
    h = ctypes.c_void_p()
    _check(load_library().carve_host_ctx_create(ctypes.byref(h)))
    return h


def carve_host_ctx_destroy(ctx) -> None:
    load_library().carve_host_ctx_destroy(ctx)


def carve_fwd_bwd_host(p: Params, with_bwd: bool, x: dict, O, S_final, dO, dS_final, grads: dict, arena,
                       stream: int = 0, ctx=None) -> None:
    """carve_fwd_bwd_host (ctx None) / carve_fwd_bwd_host_ctx of carve.h: all tensors are HOST (pinned) tensors, `arena`
    is a device byte tensor of carve_host_arena_bytes(p, with_bwd) bytes."""
    cp = p.c()
    g = grads or {}
    args = [ctypes.byref(cp), int(with_bwd), *[_ptr(x.get(n)) for n in _FWD_IN], _ptr(O), _ptr(S_final), _ptr(dO),
            _ptr(dS_final), *[_ptr(g.get(n)) for n in _GRADS], _ptr(arena), _nbytes(arena), ctypes.c_void_p(stream)]
    if ctx is None:
        _check(load_library().carve_fwd_bwd_host(*args))
    else:
        _check(load_library().carve_fwd_bwd_host_ctx(ctx, *args))

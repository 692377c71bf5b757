"""ctypes loader for the CPU oracle (oracle/sla_oracle.cpp).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package never imports this module.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sla_oracle.cpp")
_LIB = os.path.join(_HERE, "libsla_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no CUDA, no third-party code)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-pthread", _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        p = ctypes.c_void_p
        i = ctypes.c_int
        for suf in ("f32", "f64"):
            getattr(L, f"sla_oracle_forward_{suf}").argtypes = [p, p, p, p, i, i, i, p, p, p, i, i, ctypes.c_double]
            getattr(L, f"sla_oracle_forward_{suf}").restype = None
            getattr(L, f"sla_oracle_backward_{suf}").argtypes = [p, p, p, p, p, i, i, i, p, p, p, i, i, ctypes.c_double]
            getattr(L, f"sla_oracle_backward_{suf}").restype = None
        L.sla_oracle_offsets.argtypes = [p, ctypes.c_int64, i, p]
        L.sla_oracle_offsets.restype = None
        L.sla_oracle_hw_threads.restype = i
        _lib = L
    return _lib


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _prep(x):
    x = np.asarray(x)
    if x.dtype not in (np.float32, np.float64):
        x = x.astype(np.float64)
    return np.ascontiguousarray(x)


PHI_KINDS = {"elu1": 0, "relu": 1}


def forward(q, k, v, offsets, *, return_state: bool = False, nthreads: int = 1, phi: str = "elu1", eps: float = 0.0):
    """q,k,v: [N,H,d] float32 or float64 numpy; offsets int32[W+1].  Returns float64 out [N,H,d]
    (and S [W,H,d,d], z [W,H,d] if return_state).  phi: "elu1" (default, eps 0) or "relu" (epsilon `eps` in the
    denominator, reading A15)."""
    L = _load()
    q, k, v = _prep(q), _prep(k), _prep(v)
    assert q.dtype == k.dtype == v.dtype and q.shape == k.shape == v.shape and q.ndim == 3
    off = np.ascontiguousarray(offsets, dtype=np.int32)
    N, H, d = q.shape
    W = off.shape[0] - 1
    assert off[0] == 0 and off[-1] == N and np.all(np.diff(off) >= 0)
    out = np.full((N, H, d), np.nan, dtype=np.float64)
    S = np.zeros((W, H, d, d), dtype=np.float64) if return_state else None
    z = np.zeros((W, H, d), dtype=np.float64) if return_state else None
    fn = L.sla_oracle_forward_f32 if q.dtype == np.float32 else L.sla_oracle_forward_f64
    fn(_ptr(q), _ptr(k), _ptr(v), _ptr(off), W, H, d, _ptr(out), _ptr(S), _ptr(z), int(nthreads), PHI_KINDS[phi],
       float(eps))
    return (out, S, z) if return_state else out


def backward(q, k, v, d_out, offsets, *, nthreads: int = 1, phi: str = "elu1", eps: float = 0.0):
    """Analytic gradients of L = sum(d_out * SLA(q,k,v)).  Returns float64 dq, dk, dv."""
    L = _load()
    q, k, v, g = _prep(q), _prep(k), _prep(v), _prep(d_out)
    assert q.dtype == k.dtype == v.dtype == g.dtype and q.shape == k.shape == v.shape == g.shape
    off = np.ascontiguousarray(offsets, dtype=np.int32)
    N, H, d = q.shape
    W = off.shape[0] - 1
    assert off[0] == 0 and off[-1] == N and np.all(np.diff(off) >= 0)
    dq = np.full((N, H, d), np.nan, dtype=np.float64)
    dk = np.full((N, H, d), np.nan, dtype=np.float64)
    dv = np.full((N, H, d), np.nan, dtype=np.float64)
    fn = L.sla_oracle_backward_f32 if q.dtype == np.float32 else L.sla_oracle_backward_f64
    fn(_ptr(q), _ptr(k), _ptr(v), _ptr(g), _ptr(off), W, H, d, _ptr(dq), _ptr(dk), _ptr(dv), int(nthreads),
       PHI_KINDS[phi], float(eps))
    return dq, dk, dv


def offsets_from_window_ids(win_id, W: int):
    """off[w] = #{i : win_id[i] < w}, w = 0..W (int32[W+1])."""
    L = _load()
    ids = np.ascontiguousarray(win_id, dtype=np.int32)
    assert ids.ndim == 1
    if ids.size:
        assert ids.min() >= 0 and ids.max() < W and np.all(np.diff(ids) >= 0)
    off = np.zeros(W + 1, dtype=np.int32)
    L.sla_oracle_offsets(_ptr(ids), ids.shape[0], int(W), _ptr(off))
    return off


def hw_threads() -> int:
    return int(_load().sla_oracle_hw_threads())

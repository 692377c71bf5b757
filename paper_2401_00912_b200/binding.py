"""Thin Python binding of the C-ABI library declared in include/sla.h.

Argument marshalling only: torch supplies device memory and the current stream; every step of the SLA
path runs in the library's CUDA kernels.  There is NO fallback: if the library is missing or a call
fails, an exception is raised.  This module never imports anything under oracle/.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsla_b200.so")

SLA_OK = 0
SLA_F32, SLA_F16, SLA_BF16 = 0, 1, 2
SLA_PHI_ELU1, SLA_PHI_RELU = 0, 1
_PHI = {"elu1": SLA_PHI_ELU1, "relu": SLA_PHI_RELU}

# Every symbol include/sla.h declares (tests check the library exports exactly these).
SYMBOLS = (
    "sla_status_string", "sla_version", "sla_workspace_bytes", "sla_offsets_from_window_ids",
    "sla_forward", "sla_forward_phi", "sla_backward_phi", "sla_forward_tcgen05", "sla_forward_static", "sla_forward_bounded", "sla_span_table_bytes", "sla_build_span_table", "sla_forward_planned", "sla_backward", "sla_backward_bounded", "sla_forward_host",
    "sla_bench_stream_ceiling",
    "sla_window_count", "sla_window_keys", "sla_sort_workspace_bytes", "sla_sort_by_window", "sla_gather_rows",
    "sla_scatter_rows", "sla_sequence_workspace_bytes", "sla_sequence_from_coords",
    "sla_qkv_projection", "sla_linear", "sla_module_forward", "sla_cwi_workspace_bytes", "sla_cwi_forward",
)

_lib = None


class SlaError(RuntimeError):
    pass


def load_library(path: str | None = None) -> ctypes.CDLL:
    """dlopen the in-tree library and declare the C signatures.  Fails loudly if it is not built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or os.environ.get("SLA_LIB_PATH") or LIB_PATH   # SLA_LIB_PATH: A/B-test another build
    if not os.path.exists(p):
        raise SlaError(f"{p} not found: build it with `python -m paper_2401_00912_b200.build` "
                       "(there is no CPU or PyTorch fallback)")
    L = ctypes.CDLL(p)
    vp, i32, i64, sz, ci = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_size_t, ctypes.c_int
    L.sla_status_string.argtypes = [ci]
    L.sla_status_string.restype = ctypes.c_char_p
    L.sla_version.argtypes = []
    L.sla_version.restype = ctypes.c_char_p
    L.sla_workspace_bytes.argtypes = [i64, i32, i32, i32, ci, ci]
    L.sla_workspace_bytes.restype = sz
    L.sla_offsets_from_window_ids.argtypes = [vp, i64, i32, vp, vp]
    L.sla_offsets_from_window_ids.restype = ci
    L.sla_forward.argtypes = [vp, vp, vp, vp, i64, i32, i32, i32, ci, vp, vp, sz, vp]
    L.sla_forward.restype = ci
    L.sla_forward_phi.argtypes = [vp, vp, vp, vp, i64, i32, i32, i32, ci, ci, ctypes.c_float, vp, vp, sz, vp]
    L.sla_forward_phi.restype = ci
    L.sla_backward_phi.argtypes = [vp, vp, vp, vp, i64, i32, i32, i32, ci, ci, ctypes.c_float, vp, vp, vp, vp, vp, sz, vp]
    L.sla_backward_phi.restype = ci
    L.sla_forward_tcgen05.argtypes = [vp, vp, vp, vp, i64, i32, i32, i32, ci, vp, vp, sz, vp]
    L.sla_forward_tcgen05.restype = ci
    L.sla_forward_static.argtypes = [vp, vp, vp, vp, i64, i32, i32, i32, ci, vp, vp]
    L.sla_forward_static.restype = ci
    L.sla_forward_bounded.argtypes = [vp, vp, vp, vp, i64, i32, i32, i32, ci, vp, i32, vp]
    L.sla_forward_bounded.restype = ci
    L.sla_span_table_bytes.argtypes = [i64, i32, i32]
    L.sla_span_table_bytes.restype = sz
    L.sla_build_span_table.argtypes = [vp, i64, i32, i32, i32, vp, sz, vp]
    L.sla_build_span_table.restype = ci
    L.sla_forward_planned.argtypes = [vp, vp, vp, vp, i64, i32, i32, i32, ci, vp, i32, vp, sz, vp]
    L.sla_forward_planned.restype = ci
    L.sla_backward.argtypes = [vp, vp, vp, vp, i64, i32, i32, i32, ci, vp, vp, vp, vp, vp, sz, vp]
    L.sla_backward.restype = ci
    L.sla_backward_bounded.argtypes = [vp, vp, vp, vp, i64, i32, i32, i32, ci, vp, vp, vp, vp, i32, vp]
    L.sla_backward_bounded.restype = ci
    L.sla_forward_host.argtypes = [vp, vp, vp, vp, i64, i32, i32, i32, ci, vp, vp]
    L.sla_forward_host.restype = ci
    L.sla_bench_stream_ceiling.argtypes = [vp, vp, vp, vp, sz, vp]
    L.sla_bench_stream_ceiling.restype = ci
    L.sla_window_count.argtypes = [i32, i32, i32, i32, i32]
    L.sla_window_count.restype = i64
    L.sla_window_keys.argtypes = [vp, i64, i32, i32, i32, i32, i32, vp, vp]
    L.sla_window_keys.restype = ci
    L.sla_sort_workspace_bytes.argtypes = [i64]
    L.sla_sort_workspace_bytes.restype = sz
    L.sla_sort_by_window.argtypes = [vp, i64, i32, vp, vp, vp, sz, vp]
    L.sla_sort_by_window.restype = ci
    L.sla_gather_rows.argtypes = [vp, vp, i64, sz, vp, vp]
    L.sla_gather_rows.restype = ci
    L.sla_scatter_rows.argtypes = [vp, vp, i64, sz, vp, vp]
    L.sla_scatter_rows.restype = ci
    L.sla_sequence_workspace_bytes.argtypes = [i64]
    L.sla_sequence_workspace_bytes.restype = sz
    L.sla_sequence_from_coords.argtypes = [vp, i64, i32, i32, i32, i32, i32, vp, vp, vp, vp, sz, vp]
    L.sla_sequence_from_coords.restype = ci
    L.sla_qkv_projection.argtypes = [vp, vp, vp, i64, i32, ci, vp, vp, vp, vp]
    L.sla_qkv_projection.restype = ci
    L.sla_linear.argtypes = [vp, vp, vp, i64, i32, ci, vp, vp]
    L.sla_linear.restype = ci
    L.sla_module_forward.argtypes = [vp, vp, vp, vp, i64, i32, i32, i32, ci, vp, vp, vp, vp, vp, sz, vp]
    L.sla_module_forward.restype = ci
    L.sla_cwi_workspace_bytes.argtypes = [i32, i32, i32, i32]
    L.sla_cwi_workspace_bytes.restype = sz
    L.sla_cwi_forward.argtypes = [vp, vp, i64, i32, ci, i32, i32, i32, i32, i32, i32, vp, vp, vp, vp, vp, sz, vp]
    L.sla_cwi_forward.restype = ci
    if path is None:
        _lib = L
    return L


def _check(rc: int, what: str):
    if rc != SLA_OK:
        raise SlaError(f"{what} failed: {load_library().sla_status_string(rc).decode()} ({rc})")


def _dt(t) -> int:
    import torch
    try:
        return {torch.float32: SLA_F32, torch.float16: SLA_F16, torch.bfloat16: SLA_BF16}[t.dtype]
    except KeyError:
        raise SlaError(f"unsupported dtype {t.dtype}") from None


def _stream(stream=None) -> int:
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def _chk_dev(*ts):
    for t in ts:
        if not t.is_cuda:
            raise SlaError("device entry points need CUDA tensors (no CPU fallback)")
        if not t.is_contiguous():
            raise SlaError("tensors must be contiguous [N,H,d_h]")


def workspace_bytes(N: int, W: int, H: int, d_h: int, dt: int, for_backward: bool = False) -> int:
    return int(load_library().sla_workspace_bytes(N, W, H, d_h, dt, 1 if for_backward else 0))


def _workspace(like, N, W, H, d_h, dt, for_backward, workspace):
    import torch
    need = workspace_bytes(N, W, H, d_h, dt, for_backward)
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=like.device)
    return workspace, workspace.numel() * workspace.element_size()


def sla_offsets_from_window_ids(win_id, W: int, out=None, stream=None):
    """win_id: CUDA int32[N] non-decreasing in [0,W) -> CUDA int32[W+1] offsets (include/sla.h)."""
    import torch
    L = load_library()
    _chk_dev(win_id)
    if win_id.dtype != torch.int32:
        raise SlaError("win_id must be int32")
    N = win_id.numel()
    if out is None:
        out = torch.empty(W + 1, dtype=torch.int32, device=win_id.device)
    _check(L.sla_offsets_from_window_ids(win_id.data_ptr(), N, W, out.data_ptr(), _stream(stream)),
           "sla_offsets_from_window_ids")
    return out


def sla_forward(q, k, v, window_offsets, out=None, workspace=None, stream=None, max_window_len=0, tcgen05=False,
                phi="elu1", eps=0.0):
    """q,k,v: CUDA [N,H,d_h] (fp32/fp16/bf16); window_offsets: CUDA int32[W+1] -> out [N,H,d_h].
    max_window_len > 0 (a promise that no window is longer; <= 256) takes sla_forward_bounded: one
    kernel launch, no workspace.  tcgen05=True takes sla_forward_tcgen05 (fp16, d_h = 16, H*d_h % 128 == 0).
    phi="relu" (with eps > 0 in the denominator) takes sla_forward_phi."""
    import torch
    L = load_library()
    _chk_dev(q, k, v, window_offsets)
    if not (q.shape == k.shape == v.shape and q.dim() == 3 and q.dtype == k.dtype == v.dtype):
        raise SlaError("q,k,v must share shape [N,H,d_h] and dtype")
    if window_offsets.dtype != torch.int32:
        raise SlaError("window_offsets must be int32")
    N, H, d = q.shape
    W = window_offsets.numel() - 1
    dt = _dt(q)
    if out is None:
        out = torch.empty_like(q)
    if max_window_len:
        _check(L.sla_forward_bounded(q.data_ptr(), k.data_ptr(), v.data_ptr(), window_offsets.data_ptr(), N, W,
                                     H, d, dt, out.data_ptr(), int(max_window_len), _stream(stream)),
               "sla_forward_bounded")
        return out
    workspace, wsb = _workspace(q, N, W, H, d, dt, False, workspace)
    if phi != "elu1":
        _check(L.sla_forward_phi(q.data_ptr(), k.data_ptr(), v.data_ptr(), window_offsets.data_ptr(), N, W, H, d, dt,
                                 _PHI[phi], float(eps), out.data_ptr(), workspace.data_ptr(), wsb, _stream(stream)),
               "sla_forward_phi")
        return out
    fn, name = (L.sla_forward_tcgen05, "sla_forward_tcgen05") if tcgen05 else (L.sla_forward, "sla_forward")
    _check(fn(q.data_ptr(), k.data_ptr(), v.data_ptr(), window_offsets.data_ptr(), N, W, H, d,
              dt, out.data_ptr(), workspace.data_ptr(), wsb, _stream(stream)), name)
    return out


def sla_backward(q, k, v, window_offsets, d_out, dq=None, dk=None, dv=None, workspace=None, stream=None,
                 phi="elu1", eps=0.0, max_window_len=0):
    """Gradients of sum(d_out * SLA(q,k,v)) -> (dq, dk, dv), each [N,H,d_h] of the input dtype.
    max_window_len > 0 (a promise that no window is longer; <= 256) takes sla_backward_bounded: one kernel
    launch, no workspace."""
    import torch
    L = load_library()
    _chk_dev(q, k, v, window_offsets, d_out)
    if not (q.shape == k.shape == v.shape == d_out.shape and q.dim() == 3
            and q.dtype == k.dtype == v.dtype == d_out.dtype):
        raise SlaError("q,k,v,d_out must share shape [N,H,d_h] and dtype")
    if window_offsets.dtype != torch.int32:
        raise SlaError("window_offsets must be int32")
    N, H, d = q.shape
    W = window_offsets.numel() - 1
    dt = _dt(q)
    dq = torch.empty_like(q) if dq is None else dq
    dk = torch.empty_like(q) if dk is None else dk
    dv = torch.empty_like(q) if dv is None else dv
    if max_window_len:
        if phi != "elu1":
            raise SlaError("sla_backward_bounded computes the elu+1 map only")
        _check(L.sla_backward_bounded(q.data_ptr(), k.data_ptr(), v.data_ptr(), window_offsets.data_ptr(), N, W, H, d,
                                      dt, d_out.data_ptr(), dq.data_ptr(), dk.data_ptr(), dv.data_ptr(),
                                      int(max_window_len), _stream(stream)), "sla_backward_bounded")
        return dq, dk, dv
    workspace, wsb = _workspace(q, N, W, H, d, dt, True, workspace)
    if phi != "elu1":
        _check(L.sla_backward_phi(q.data_ptr(), k.data_ptr(), v.data_ptr(), window_offsets.data_ptr(), N, W, H, d, dt,
                                  _PHI[phi], float(eps), d_out.data_ptr(), dq.data_ptr(), dk.data_ptr(), dv.data_ptr(),
                                  workspace.data_ptr(), wsb, _stream(stream)), "sla_backward_phi")
        return dq, dk, dv
    _check(L.sla_backward(q.data_ptr(), k.data_ptr(), v.data_ptr(), window_offsets.data_ptr(), N, W, H, d,
                          dt, d_out.data_ptr(), dq.data_ptr(), dk.data_ptr(), dv.data_ptr(),
                          workspace.data_ptr(), wsb, _stream(stream)), "sla_backward")
    return dq, dk, dv


def sla_forward_host(q, k, v, win_id, W: int, out=None, stream=None):
    """End-to-end host entry: q,k,v,win_id are HOST (CPU, ideally pinned) torch tensors; returns a
    HOST tensor.  H2D copies, prep, forward and the D2H copy all happen inside the C call."""
    import torch
    L = load_library()
    for t in (q, k, v, win_id):
        if t.is_cuda or not t.is_contiguous():
            raise SlaError("sla_forward_host takes contiguous host tensors")
    if not (q.shape == k.shape == v.shape and q.dim() == 3 and q.dtype == k.dtype == v.dtype):
        raise SlaError("q,k,v must share shape [N,H,d_h] and dtype")
    if win_id.dtype != torch.int32 or win_id.numel() != q.shape[0]:
        raise SlaError("win_id must be int32[N]")
    N, H, d = q.shape
    if out is None:
        out = torch.empty_like(q, pin_memory=q.is_pinned())
    _check(L.sla_forward_host(q.data_ptr(), k.data_ptr(), v.data_ptr(), win_id.data_ptr(), N, W, H, d,
                              _dt(q), out.data_ptr(), _stream(stream)), "sla_forward_host")
    return out


def sla_bench_stream_ceiling(a, b, c, out, stream=None):
    """Measurement aid (include/sla.h): out = a ^ b ^ c bytewise, 128-bit streaming accesses."""
    L = load_library()
    _chk_dev(a, b, c, out)
    nbytes = a.numel() * a.element_size()
    for t in (b, c, out):
        if t.numel() * t.element_size() != nbytes:
            raise SlaError("a, b, c, out must have the same size in bytes")
    _check(L.sla_bench_stream_ceiling(a.data_ptr(), b.data_ptr(), c.data_ptr(), out.data_ptr(), nbytes,
                                      _stream(stream)), "sla_bench_stream_ceiling")
    return out


# ---- sequence preparation (include/sla.h) ----

def sla_window_count(batch: int, grid_h: int, grid_w: int, S_h: int, S_w: int) -> int:
    W = int(load_library().sla_window_count(batch, grid_h, grid_w, S_h, S_w))
    if W < 0:
        raise SlaError("sla_window_count: arguments must be >= 1 and W must fit in int32")
    return W


def _chk_i32(t, what):
    import torch
    _chk_dev(t)
    if t.dtype != torch.int32:
        raise SlaError(f"{what} must be int32")


def sla_window_keys(coords, batch: int, grid_h: int, grid_w: int, S_h: int, S_w: int, out=None, stream=None):
    """coords: CUDA int32[N,4] rows (b, z, y, x) -> CUDA int32[N] window keys in [0, W]."""
    import torch
    _chk_i32(coords, "coords")
    if coords.dim() != 2 or coords.shape[1] != 4:
        raise SlaError("coords must be [N,4]")
    N = coords.shape[0]
    if out is None:
        out = torch.empty(N, dtype=torch.int32, device=coords.device)
    _check(load_library().sla_window_keys(coords.data_ptr(), N, batch, grid_h, grid_w, S_h, S_w, out.data_ptr(),
                                          _stream(stream)), "sla_window_keys")
    return out


def sla_sort_by_window(key, W: int, workspace=None, stream=None):
    """key: CUDA int32[N] in [0, W] -> (perm, key_sorted), the stable sort by key."""
    import torch
    L = load_library()
    _chk_i32(key, "key")
    N = key.numel()
    perm = torch.empty(N, dtype=torch.int32, device=key.device)
    ks = torch.empty(N, dtype=torch.int32, device=key.device)
    if workspace is None:
        workspace = torch.empty(max(int(L.sla_sort_workspace_bytes(N)), 16), dtype=torch.uint8, device=key.device)
    _check(L.sla_sort_by_window(key.data_ptr(), N, W, perm.data_ptr(), ks.data_ptr(), workspace.data_ptr(),
                                workspace.numel(), _stream(stream)), "sla_sort_by_window")
    return perm, ks


def _permute_rows(fn, name, src, perm, out, stream):
    import torch
    _chk_dev(src)
    _chk_i32(perm, "perm")
    N = perm.numel()
    if src.shape[0] != N:
        raise SlaError("src must have one row per entry of perm")
    if out is None:
        out = torch.empty_like(src)
    row_bytes = (src.numel() // N) * src.element_size() if N else 0
    _check(fn(src.data_ptr(), perm.data_ptr(), N, row_bytes, out.data_ptr(), _stream(stream)), name)
    return out


def sla_gather_rows(src, perm, out=None, stream=None):
    """out[j] = src[perm[j]] (rows of any shape and dtype whose size is a multiple of 4 bytes)."""
    return _permute_rows(load_library().sla_gather_rows, "sla_gather_rows", src, perm, out, stream)


def sla_scatter_rows(src, perm, out=None, stream=None):
    """out[perm[j]] = src[j]: undoes sla_gather_rows."""
    return _permute_rows(load_library().sla_scatter_rows, "sla_scatter_rows", src, perm, out, stream)


def sla_sequence_from_coords(coords, batch: int, grid_h: int, grid_w: int, S_h: int, S_w: int, workspace=None,
                             stream=None):
    """coords: CUDA int32[N,4] -> (perm int32[N], key_sorted int32[N], window_offsets int32[W+1]) in one C call."""
    import torch
    L = load_library()
    _chk_i32(coords, "coords")
    if coords.dim() != 2 or coords.shape[1] != 4:
        raise SlaError("coords must be [N,4]")
    N = coords.shape[0]
    W = sla_window_count(batch, grid_h, grid_w, S_h, S_w)
    dev = coords.device
    perm = torch.empty(N, dtype=torch.int32, device=dev)
    ks = torch.empty(N, dtype=torch.int32, device=dev)
    off = torch.empty(W + 1, dtype=torch.int32, device=dev)
    if workspace is None:
        workspace = torch.empty(max(int(L.sla_sequence_workspace_bytes(N)), 16), dtype=torch.uint8, device=dev)
    _check(L.sla_sequence_from_coords(coords.data_ptr(), N, batch, grid_h, grid_w, S_h, S_w, perm.data_ptr(),
                                      ks.data_ptr(), off.data_ptr(), workspace.data_ptr(), workspace.numel(),
                                      _stream(stream)), "sla_sequence_from_coords")
    return perm, ks, off


def sla_forward_static(q, k, v, window_offsets, out=None, stream=None):
    """sla_forward with the workspace in the library's static device array (include/sla.h): the C call allocates
    nothing; problems whose workspace exceeds 4 MiB raise SLA_ERR_TOO_LARGE.  `out` may be passed in so that this
    wrapper allocates nothing either."""
    import torch
    L = load_library()
    _chk_dev(q, k, v, window_offsets)
    if not (q.shape == k.shape == v.shape and q.dim() == 3 and q.dtype == k.dtype == v.dtype):
        raise SlaError("q,k,v must share shape [N,H,d_h] and dtype")
    if window_offsets.dtype != torch.int32:
        raise SlaError("window_offsets must be int32")
    N, H, d = q.shape
    if out is None:
        out = torch.empty_like(q)
    _check(L.sla_forward_static(q.data_ptr(), k.data_ptr(), v.data_ptr(), window_offsets.data_ptr(), N,
                                window_offsets.numel() - 1, H, d, _dt(q), out.data_ptr(), _stream(stream)),
           "sla_forward_static")
    return out


# ---- shared Q/K/V projection and the module (include/sla.h) ----

def _chk_proj(x, w, bias):
    import torch
    _chk_dev(x, w)
    if x.dim() != 2 or w.dim() != 2 or w.shape != (3 * x.shape[1], x.shape[1]) or w.dtype != x.dtype:
        raise SlaError("x must be [N, C] and w_qkv [3C, C] of the same dtype")
    if bias is not None:
        _chk_dev(bias)
        if bias.dtype != torch.float32 or bias.numel() != 3 * x.shape[1]:
            raise SlaError("bias must be fp32 [3C]")


def sla_qkv_projection(x, w_qkv, bias=None, q=None, k=None, v=None, stream=None):
    """x: CUDA [N, C], w_qkv: [3C, C] (row j = weights of output feature j; Q, K, V blocks) -> (q, k, v), each
    [N, C]: y = x w^T (+ bias); fp16/bf16 with C in {128, 256} on tcgen05, everything else on a generic kernel."""
    import torch
    L = load_library()
    _chk_proj(x, w_qkv, bias)
    N, C = x.shape
    q, k, v = (torch.empty_like(x) if t is None else t for t in (q, k, v))
    _check(L.sla_qkv_projection(x.data_ptr(), w_qkv.data_ptr(), bias.data_ptr() if bias is not None else None, N, C,
                                _dt(x), q.data_ptr(), k.data_ptr(), v.data_ptr(), _stream(stream)),
           "sla_qkv_projection")
    return q, k, v


def sla_linear(x, w, bias=None, out=None, stream=None):
    """y = x w^T (+ bias): x CUDA [N, C] fp16/bf16, w [C, C] (row j = weights of output feature j), bias fp32 [C]."""
    import torch
    L = load_library()
    _chk_dev(x, w)
    if x.dim() != 2 or tuple(w.shape) != (x.shape[1], x.shape[1]) or w.dtype != x.dtype:
        raise SlaError("x must be [N, C] and w [C, C] of the same dtype")
    if bias is not None:
        _chk_dev(bias)
        if bias.dtype != torch.float32 or bias.numel() != x.shape[1]:
            raise SlaError("bias must be fp32 [C]")
    out = torch.empty_like(x) if out is None else out
    _check(L.sla_linear(x.data_ptr(), w.data_ptr(), bias.data_ptr() if bias is not None else None, x.shape[0],
                        x.shape[1], _dt(x), out.data_ptr(), _stream(stream)), "sla_linear")
    return out


def sla_module_forward(x, w_qkv, window_offsets, H: int, bias=None, q=None, k=None, v=None, out=None, workspace=None,
                       stream=None):
    """Projection, then SLA on its results, in one C call -> (out [N, H, d_h], q, k, v)."""
    import torch
    L = load_library()
    _chk_proj(x, w_qkv, bias)
    _chk_dev(window_offsets)
    if window_offsets.dtype != torch.int32:
        raise SlaError("window_offsets must be int32")
    N, C = x.shape
    if C % H:
        raise SlaError("C must be H * d_h")
    d = C // H
    W = window_offsets.numel() - 1
    dt = _dt(x)
    q, k, v = (torch.empty(N, H, d, dtype=x.dtype, device=x.device) if t is None else t for t in (q, k, v))
    out = torch.empty(N, H, d, dtype=x.dtype, device=x.device) if out is None else out
    workspace, wsb = _workspace(x, N, W, H, d, dt, False, workspace)
    _check(L.sla_module_forward(x.data_ptr(), w_qkv.data_ptr(), bias.data_ptr() if bias is not None else None,
                                window_offsets.data_ptr(), N, W, H, d, dt, q.data_ptr(), k.data_ptr(), v.data_ptr(),
                                out.data_ptr(), workspace.data_ptr(), wsb, _stream(stream)), "sla_module_forward")
    return out, q, k, v


# ---- Cross-Window Interaction (include/sla.h) ----

def sla_cwi_forward(x, coords, grid, S_h: int, S_w: int, w_h, w_w, w_3, out=None, workspace=None, stream=None):
    """x: CUDA [N, 4c]; coords: CUDA int32 [N,4] rows (b, z, y, x); grid = (batch, grid_z, grid_h, grid_w);
    w_h [c, S_h+1], w_w [c, S_w+1], w_3 [c, 27] fp32 -> out [N, 4c] (Eq. 4-7)."""
    import torch
    L = load_library()
    _chk_dev(x, w_h, w_w, w_3)
    _chk_i32(coords, "coords")
    if x.dim() != 2 or coords.shape != (x.shape[0], 4):
        raise SlaError("x must be [N, C] and coords [N, 4]")
    N, C = x.shape
    c = C // 4
    for w, taps in ((w_h, S_h + 1), (w_w, S_w + 1), (w_3, 27)):
        if w.dtype != torch.float32 or tuple(w.shape) != (c, taps):
            raise SlaError("weights must be fp32 [c, taps]")
    batch, gz, gh, gw = (int(v) for v in grid)
    need = int(L.sla_cwi_workspace_bytes(batch, gz, gh, gw))
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=x.device)
    if out is None:
        out = torch.empty_like(x)
    dt = {torch.float32: SLA_F32, torch.float16: SLA_F16, torch.bfloat16: SLA_BF16}.get(x.dtype)
    if dt is None:
        raise SlaError(f"unsupported dtype {x.dtype}")
    _check(L.sla_cwi_forward(x.data_ptr(), coords.data_ptr(), N, C, dt, batch, gz, gh, gw, S_h, S_w, w_h.data_ptr(),
                             w_w.data_ptr(), w_3.data_ptr(), out.data_ptr(), workspace.data_ptr(), workspace.numel(),
                             _stream(stream)), "sla_cwi_forward")
    return out


# ---- span table ----

def sla_build_span_table(window_offsets, N: int, H: int, d_h: int, table=None, stream=None):
    """The work list of a scene for sla_forward_planned: CUDA uint8 buffer of sla_span_table_bytes(N, H, d_h)."""
    import torch
    L = load_library()
    _chk_i32(window_offsets, "window_offsets")
    need = int(L.sla_span_table_bytes(N, H, d_h))
    if table is None:
        table = torch.empty(max(need, 16), dtype=torch.uint8, device=window_offsets.device)
    _check(L.sla_build_span_table(window_offsets.data_ptr(), N, window_offsets.numel() - 1, H, d_h, table.data_ptr(),
                                  table.numel(), _stream(stream)), "sla_build_span_table")
    return table


def sla_forward_planned(q, k, v, window_offsets, table, max_window_len: int, out=None, stream=None):
    """sla_forward_bounded with the scene's span table (built once by sla_build_span_table)."""
    import torch
    L = load_library()
    _chk_dev(q, k, v, window_offsets, table)
    if not (q.shape == k.shape == v.shape and q.dim() == 3 and q.dtype == k.dtype == v.dtype):
        raise SlaError("q,k,v must share shape [N,H,d_h] and dtype")
    N, H, d = q.shape
    if out is None:
        out = torch.empty_like(q)
    _check(L.sla_forward_planned(q.data_ptr(), k.data_ptr(), v.data_ptr(), window_offsets.data_ptr(), N,
                                 window_offsets.numel() - 1, H, d, _dt(q), out.data_ptr(), int(max_window_len),
                                 table.data_ptr(), table.numel(), _stream(stream)), "sla_forward_planned")
    return out

"""Thin Python binding of libgspn (include/gspn.h): argument marshalling only.

Every function here has the name of the C entry point it calls and does no arithmetic of the
method: tensors are checked (dtype, device, contiguity, shape), their data pointers and the
current CUDA stream are handed to the C ABI, outputs are allocated with torch (device memory
only).  There is no fallback: if libgspn.so is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgspn.so")

DIR_TB, DIR_BT, DIR_LR, DIR_RL, DIR_ALL = 1, 2, 4, 8, 15
F32, BF16 = 0, 1
IMPL_AUTO, IMPL_NAIVE, IMPL_FUSED, IMPL_FLAT, IMPL_CHAIN, IMPL_PAIR, IMPL_PLANE, IMPL_LINE = 0, 1, 2, 3, 4, 5, 6, 7
STATUS = {0: "GSPN_OK", 1: "GSPN_EINVAL", 2: "GSPN_EUNSUPPORTED", 3: "GSPN_EALIGN",
          4: "GSPN_EWORKSPACE", 5: "GSPN_ECUDA"}

EXPORTS = ("gspn_scan_fwd", "gspn_scan_bwd", "gspn_merge", "gspn_scan_fwd_ex", "gspn_scan_bwd_ex",
           "gspn_scan_fwd_host", "gspn_scan_bwd_host", "gspn_scan_fwd_bwd_host", "gspn_debug_chunk_copy",
           "gspn_normalize_fwd", "gspn_normalize_bwd",
           "gspn_workspace_bytes",
           "gspn_last_launch_count", "gspn_last_variant", "gspn_last_error", "gspn_version")


class GspnError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


class _Args(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_size_t),
                ("x", ctypes.c_void_p), ("w3", ctypes.c_void_p), ("lam", ctypes.c_void_p),
                ("u", ctypes.c_void_p), ("h0", ctypes.c_void_p), ("dy", ctypes.c_void_p),
                ("y", ctypes.c_void_p),
                ("dx", ctypes.c_void_p), ("dlambda", ctypes.c_void_p), ("du", ctypes.c_void_p),
                ("dw3", ctypes.c_void_p), ("dh0", ctypes.c_void_p),
                ("B", ctypes.c_int), ("C", ctypes.c_int), ("H", ctypes.c_int), ("W", ctypes.c_int),
                ("G", ctypes.c_int), ("dir_mask", ctypes.c_uint), ("dtype", ctypes.c_int),
                ("impl", ctypes.c_int), ("stream", ctypes.c_void_p),
                ("dir_stride_w3", ctypes.c_size_t), ("dir_stride_lambda", ctypes.c_size_t),
                ("dir_stride_u", ctypes.c_size_t), ("k_chunk", ctypes.c_int), ("flags", ctypes.c_uint),
                ("workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_size_t)]


FLAG_W3_LOGITS = 1


DIR_STRIDE_DENSE = ctypes.c_size_t(-1).value       # GSPN_DIR_STRIDE_DENSE
SHAREABLE = ("w3", "lam", "u")


def _strides(shared) -> dict:
    """gspn_args_t.dir_stride_*: 0 for the operands named in `shared` (one slab read by every direction), else dense."""
    bad = set(shared) - set(SHAREABLE)
    if bad:
        raise ValueError(f"shared: unknown operand(s) {sorted(bad)} (choose from {SHAREABLE})")
    return {"dir_stride_w3": 0 if "w3" in shared else DIR_STRIDE_DENSE,
            "dir_stride_lambda": 0 if "lam" in shared else DIR_STRIDE_DENSE,
            "dir_stride_u": 0 if "u" in shared else DIR_STRIDE_DENSE}


_lib = None


def lib() -> ctypes.CDLL:
    """Load libgspn.so (built in-tree by paper_2606_00746_b200.build); raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise GspnError(5, f"{LIB_PATH} not found: run `python -m paper_2606_00746_b200.build` "
                               "(there is no CPU or PyTorch fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, ci, cu = ctypes.c_void_p, ctypes.c_int, ctypes.c_uint
        L.gspn_scan_fwd.argtypes = [vp] * 5 + [ci] * 5 + [cu, ci, vp]
        L.gspn_scan_bwd.argtypes = [vp] * 10 + [ci] * 5 + [cu, ci, vp]
        L.gspn_merge.argtypes = [vp] * 3 + [ci] * 4 + [cu, ci, vp]
        L.gspn_normalize_fwd.argtypes = [vp] * 2 + [ci] * 4 + [cu, ci, vp]
        L.gspn_normalize_bwd.argtypes = [vp] * 3 + [ci] * 4 + [cu, ci, vp]
        L.gspn_scan_fwd_host.argtypes = L.gspn_scan_fwd.argtypes
        L.gspn_scan_bwd_host.argtypes = L.gspn_scan_bwd.argtypes
        L.gspn_scan_fwd_bwd_host.argtypes = [vp] * 11 + [ci] * 5 + [cu, ci, vp]
        L.gspn_debug_chunk_copy.argtypes = [vp, vp, ctypes.c_size_t] + [ci] * 5
        L.gspn_scan_fwd_ex.argtypes = [ctypes.POINTER(_Args)]
        L.gspn_scan_bwd_ex.argtypes = [ctypes.POINTER(_Args)]
        L.gspn_workspace_bytes.argtypes = [ci] * 5 + [cu, ci, ci]
        L.gspn_workspace_bytes.restype = ctypes.c_size_t
        L.gspn_last_error.restype = ctypes.c_char_p
        L.gspn_last_variant.restype = ctypes.c_char_p
        _lib = L
    return _lib


def _check(rc: int) -> None:
    if rc != 0:
        raise GspnError(rc, lib().gspn_last_error().decode())


def _dtype_code(t: torch.Tensor) -> int:
    if t.dtype == torch.float32:
        return F32
    if t.dtype == torch.bfloat16:
        return BF16
    raise TypeError(f"unsupported storage dtype {t.dtype}")


def _popcount(mask: int) -> int:
    return bin(mask & 15).count("1")


def _dev(t, name, shape, like):
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous() or t.dtype != like.dtype or t.device != like.device:
        raise ValueError(f"{name}: need a contiguous CUDA tensor of dtype {like.dtype} on {like.device}")
    if tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: shape {tuple(t.shape)} != {tuple(shape)}")
    return t


def _p(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(t):
    return ctypes.c_void_p(torch.cuda.current_stream(t.device).cuda_stream)


def _workspace(x, B, C, H, W, G, dir_mask, is_bwd, impl):
    """Scratch for planes beyond shared memory (gspn_args_t.workspace): allocated here, as every other tensor is, when
    gspn_workspace_bytes asks for it and the call can reach the kernels that use it."""
    if impl not in (IMPL_AUTO, IMPL_NAIVE):
        return None
    n = lib().gspn_workspace_bytes(B, C, H, W, G, dir_mask, _dtype_code(x), is_bwd)
    return torch.empty(n, dtype=torch.uint8, device=x.device) if n else None


def _shapes(x, G, dir_mask):
    B, C, H, W = x.shape
    D = _popcount(dir_mask)
    return B, C, H, W, D, (D, B, C, H, W), (D, B, G, 3, H, W), (D, B, C, max(H, W))


def gspn_scan_fwd(x, w3, lam, u, G: int, dir_mask: int = DIR_ALL, h0=None, out=None,
                  impl: int = IMPL_AUTO, shared=(), k_chunk: int = 0, w3_logits: bool = False):
    """y = sum_d u_d * scan_d(x); see include/gspn.h gspn_scan_fwd / gspn_scan_fwd_ex.
    k_chunk > 1: the chunked scan (bands of ceil(L / k_chunk) lines, independent scans; gspn_args_t.k_chunk).
    w3_logits: w3 holds the raw tap logits, Eq. 3 is applied where the taps are loaded (GSPN_FLAG_W3_LOGITS).
    shared: operands among ("w3", "lam", "u") that hold ONE slab ([B,G,3,H,W] / [B,C,H,W], no D axis) read by every
    direction (gspn_args_t.dir_stride_* = 0)."""
    if not x.is_cuda:
        raise ValueError("x: need a CUDA tensor (there is no CPU path)")
    B, C, H, W, D, s_bc, s_w, s_h0 = _shapes(x, G, dir_mask)
    _dev(x, "x", x.shape, x); _dev(w3, "w3", s_w[1:] if "w3" in shared else s_w, x)
    _dev(lam, "lam", s_bc[1:] if "lam" in shared else s_bc, x); _dev(u, "u", s_bc[1:] if "u" in shared else s_bc, x)
    _dev(h0, "h0", s_h0, x)
    y = torch.empty_like(x) if out is None else _dev(out, "out", x.shape, x)
    ws = _workspace(x, B, C, H, W, G, dir_mask, 0, impl)
    with torch.cuda.device(x.device):
        if h0 is None and impl == IMPL_AUTO and not shared and k_chunk <= 1 and not w3_logits and ws is None:
            rc = lib().gspn_scan_fwd(_p(x), _p(w3), _p(lam), _p(u), _p(y), B, C, H, W, G, dir_mask,
                                     _dtype_code(x), _stream(x))
        else:
            a = _Args(struct_size=ctypes.sizeof(_Args), x=x.data_ptr(), w3=w3.data_ptr(),
                      lam=lam.data_ptr(), u=u.data_ptr(), h0=None if h0 is None else h0.data_ptr(),
                      y=y.data_ptr(), B=B, C=C, H=H, W=W, G=G, dir_mask=dir_mask,
                      dtype=_dtype_code(x), impl=impl, workspace=None if ws is None else ws.data_ptr(),
                      workspace_bytes=0 if ws is None else ws.numel(),
                      stream=torch.cuda.current_stream(x.device).cuda_stream, k_chunk=k_chunk, flags=FLAG_W3_LOGITS if w3_logits else 0, **_strides(shared))
            rc = lib().gspn_scan_fwd_ex(ctypes.byref(a))
    _check(rc)
    return y


def gspn_scan_bwd(x, w3, lam, u, dy, G: int, dir_mask: int = DIR_ALL, h0=None,
                  need=("dx", "dlambda", "du", "dw3", "dh0"), impl: int = IMPL_AUTO, shared=(), k_chunk: int = 0,
                  w3_logits: bool = False) -> dict:
    """Adjoint of gspn_scan_fwd; returns the requested gradients (include/gspn.h gspn_scan_bwd).
    shared: as in gspn_scan_fwd; the gradients keep one slab per direction (the gradient of a shared slab is their sum).
    w3_logits: w3 holds logits; "dw3" is then the gradient of the logits."""
    if not x.is_cuda:
        raise ValueError("x: need a CUDA tensor (there is no CPU path)")
    B, C, H, W, D, s_bc, s_w, s_h0 = _shapes(x, G, dir_mask)
    _dev(x, "x", x.shape, x); _dev(w3, "w3", s_w[1:] if "w3" in shared else s_w, x)
    _dev(lam, "lam", s_bc[1:] if "lam" in shared else s_bc, x); _dev(u, "u", s_bc[1:] if "u" in shared else s_bc, x)
    _dev(dy, "dy", x.shape, x); _dev(h0, "h0", s_h0, x)
    shapes = {"dx": x.shape, "dlambda": s_bc, "du": s_bc, "dw3": s_w, "dh0": s_h0}
    out = {k: torch.empty(shapes[k], dtype=x.dtype, device=x.device) for k in need}
    g = lambda k: out[k].data_ptr() if k in out else None
    ws = _workspace(x, B, C, H, W, G, dir_mask, 1, impl)
    with torch.cuda.device(x.device):
        if h0 is None and impl == IMPL_AUTO and not shared and k_chunk <= 1 and not w3_logits and ws is None:
            rc = lib().gspn_scan_bwd(_p(x), _p(w3), _p(lam), _p(u), _p(dy), g("dx"), g("dlambda"),
                                     g("du"), g("dw3"), g("dh0"), B, C, H, W, G, dir_mask,
                                     _dtype_code(x), _stream(x))
        else:
            a = _Args(struct_size=ctypes.sizeof(_Args), x=x.data_ptr(), w3=w3.data_ptr(),
                      lam=lam.data_ptr(), u=u.data_ptr(), h0=None if h0 is None else h0.data_ptr(),
                      dy=dy.data_ptr(), dx=g("dx"), dlambda=g("dlambda"), du=g("du"), dw3=g("dw3"),
                      dh0=g("dh0"), B=B, C=C, H=H, W=W, G=G, dir_mask=dir_mask,
                      dtype=_dtype_code(x), impl=impl, workspace=None if ws is None else ws.data_ptr(),
                      workspace_bytes=0 if ws is None else ws.numel(),
                      stream=torch.cuda.current_stream(x.device).cuda_stream, k_chunk=k_chunk, flags=FLAG_W3_LOGITS if w3_logits else 0, **_strides(shared))
            rc = lib().gspn_scan_bwd_ex(ctypes.byref(a))
    _check(rc)
    return out


def gspn_merge(y_dirs, m=None, dir_mask: int = DIR_ALL, out=None):
    """y = sum_q m[q,c] * y_dirs[q]  (include/gspn.h gspn_merge)."""
    D, B, C, H, W = y_dirs.shape
    if D != _popcount(dir_mask):
        raise ValueError("y_dirs: leading dim != popcount(dir_mask)")
    if not y_dirs.is_cuda or not y_dirs.is_contiguous():
        raise ValueError("y_dirs: need a contiguous CUDA tensor")
    if m is not None and (m.dtype != torch.float32 or tuple(m.shape) != (D, C) or not m.is_cuda
                          or not m.is_contiguous()):
        raise ValueError("m: need a contiguous CUDA fp32 tensor [D,C]")
    y = torch.empty((B, C, H, W), dtype=y_dirs.dtype, device=y_dirs.device) if out is None else out
    with torch.cuda.device(y_dirs.device):
        rc = lib().gspn_merge(_p(y_dirs), _p(m), _p(y), B, C, H, W, dir_mask, _dtype_code(y_dirs),
                              _stream(y_dirs))
    _check(rc)
    return y


def _norm_shape(wt, dir_mask):
    if not wt.is_cuda or not wt.is_contiguous() or wt.dim() != 6 or wt.shape[3] != 3:
        raise ValueError("wt: need a contiguous CUDA tensor [D,B,G,3,H,W] (there is no CPU path)")
    D, B, G, _, H, W = wt.shape
    if D != _popcount(dir_mask):
        raise ValueError(f"wt: {D} direction slabs but dir_mask={dir_mask}")
    return B, G, H, W


def gspn_normalize_fwd(wt, dir_mask: int = DIR_ALL, out=None):
    """w3 = Eq. (3) of the tap logits wt [D,B,G,3,H,W]; see include/gspn.h gspn_normalize_fwd."""
    B, G, H, W = _norm_shape(wt, dir_mask)
    w3 = torch.empty_like(wt) if out is None else _dev(out, "out", wt.shape, wt)
    with torch.cuda.device(wt.device):
        rc = lib().gspn_normalize_fwd(_p(wt), _p(w3), B, G, H, W, dir_mask, _dtype_code(wt), _stream(wt))
    _check(rc)
    return w3


def gspn_normalize_bwd(wt, dw3, dir_mask: int = DIR_ALL, out=None):
    """dwt = adjoint of gspn_normalize_fwd at wt applied to dw3; see include/gspn.h gspn_normalize_bwd."""
    B, G, H, W = _norm_shape(wt, dir_mask)
    _dev(dw3, "dw3", wt.shape, wt)
    dwt = torch.empty_like(wt) if out is None else _dev(out, "out", wt.shape, wt)
    with torch.cuda.device(wt.device):
        rc = lib().gspn_normalize_bwd(_p(wt), _p(dw3), _p(dwt), B, G, H, W, dir_mask, _dtype_code(wt),
                                      _stream(wt))
    _check(rc)
    return dwt


def _host(t, name):
    if t is None:
        return None
    if t.is_cuda or not t.is_contiguous():
        raise ValueError(f"{name}: need a contiguous HOST tensor")
    return t


def gspn_scan_fwd_host(x, w3, lam, u, y, G: int, dir_mask: int = DIR_ALL, stream=None) -> None:
    """Host-buffer forward (include/gspn.h gspn_scan_fwd_host): H2D, scan, D2H, synchronised."""
    B, C, H, W = x.shape
    for t, n in ((x, "x"), (w3, "w3"), (lam, "lam"), (u, "u"), (y, "y")):
        _host(t, n)
    st = torch.cuda.current_stream().cuda_stream if stream is None else stream
    _check(lib().gspn_scan_fwd_host(_p(x), _p(w3), _p(lam), _p(u), _p(y), B, C, H, W, G, dir_mask,
                                    _dtype_code(x), ctypes.c_void_p(st)))


def gspn_scan_bwd_host(x, w3, lam, u, dy, dx, dlambda, du, dw3, dh0, G: int,
                       dir_mask: int = DIR_ALL, stream=None) -> None:
    """Host-buffer backward (include/gspn.h gspn_scan_bwd_host)."""
    B, C, H, W = x.shape
    for t, n in ((x, "x"), (w3, "w3"), (lam, "lam"), (u, "u"), (dy, "dy"), (dx, "dx"),
                 (dlambda, "dlambda"), (du, "du"), (dw3, "dw3"), (dh0, "dh0")):
        _host(t, n)
    st = torch.cuda.current_stream().cuda_stream if stream is None else stream
    _check(lib().gspn_scan_bwd_host(_p(x), _p(w3), _p(lam), _p(u), _p(dy), _p(dx), _p(dlambda), _p(du),
                                    _p(dw3), _p(dh0), B, C, H, W, G, dir_mask, _dtype_code(x),
                                    ctypes.c_void_p(st)))


def gspn_scan_fwd_bwd_host(x, w3, lam, u, dy, y, dx, dlambda, du, dw3, dh0, G: int,
                           dir_mask: int = DIR_ALL, stream=None) -> None:
    """One forward + backward step through host buffers, operands uploaded once, pipelined over batch chunks
    (include/gspn.h gspn_scan_fwd_bwd_host).  y and every gradient may be None."""
    B, C, H, W = x.shape
    for t, n in ((x, "x"), (w3, "w3"), (lam, "lam"), (u, "u"), (dy, "dy"), (y, "y"), (dx, "dx"),
                 (dlambda, "dlambda"), (du, "du"), (dw3, "dw3"), (dh0, "dh0")):
        _host(t, n)
    st = torch.cuda.current_stream().cuda_stream if stream is None else stream
    _check(lib().gspn_scan_fwd_bwd_host(_p(x), _p(w3), _p(lam), _p(u), _p(dy), _p(y), _p(dx), _p(dlambda), _p(du),
                                        _p(dw3), _p(dh0), B, C, H, W, G, dir_mask, _dtype_code(x),
                                        ctypes.c_void_p(st)))


def gspn_last_launch_count() -> int:
    return int(lib().gspn_last_launch_count())


def gspn_last_variant() -> str:
    return lib().gspn_last_variant().decode()


def gspn_version() -> int:
    return int(lib().gspn_version())

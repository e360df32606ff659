"""CPU-side checks of the C-ABI boundary: the library builds, loads, exports every symbol that
include/gspn.h declares, and rejects bad arguments before touching a GPU (no compute calls)."""
import ctypes
import os
import re

import pytest

import paper_2606_00746_b200 as gspn
from paper_2606_00746_b200 import build as gbuild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    gbuild.build()
    return gspn.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "gspn.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gspn_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(L):
    names = declared_symbols()
    assert {"gspn_scan_fwd", "gspn_scan_bwd", "gspn_merge"} <= set(names)
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/gspn.h but not exported by libgspn.so"
    assert set(names) == set(gspn.EXPORTS)


def test_version_and_workspace(L):
    assert gspn.gspn_version() >= 100
    assert L.gspn_workspace_bytes(4, 256, 128, 128, 64, 15, 1, 0) == 0
    assert L.gspn_workspace_bytes(32, 128, 73, 73, 32, 15, 1, 1) == 0
    # planes beyond shared memory: the fp32 planes the fall-back kernels move to the caller's workspace
    assert L.gspn_workspace_bytes(16, 8, 1024, 1024, 2, 15, 1, 0) == 16 * 8 * 1024 * 1024 * 4
    assert L.gspn_workspace_bytes(1, 2, 200, 200, 1, 15, 0, 0) == 0                       # 160 KB: still on chip
    assert L.gspn_workspace_bytes(1, 2, 200, 200, 1, 15, 0, 1) == max(2 * 2, 4 * 4 * 1) * 200 * 200 * 4
    assert L.gspn_workspace_bytes(4, 256, 128, 128, 64, 15, 1, 1) == 4 * 4 * 4 * 64 * 128 * 128 * 4   # cfg4 backward: the dw3 launch
    assert L.gspn_workspace_bytes(1, 1, 2000, 8, 1, 15, 0, 0) == 0                        # lines beyond 1024: not held at all


def test_argument_validation_without_gpu(L):
    buf = ctypes.create_string_buffer(4096 + 16)
    base = (ctypes.addressof(buf) + 15) & ~15
    p = ctypes.c_void_p(base)
    odd = ctypes.c_void_p(base + 2)

    def fwd(B=1, C=4, H=4, W=4, G=2, mask=15, dtype=0, x=p, y=p):
        return L.gspn_scan_fwd(x, p, p, p, y, B, C, H, W, G, mask, dtype, None)

    assert fwd(B=0) == 1 and b"shape" in L.gspn_last_error()
    assert fwd(C=4, G=3) == 1 and b"multiple" in L.gspn_last_error()
    assert fwd(mask=0) == 1 and fwd(mask=16) == 1
    assert fwd(dtype=7) == 1
    assert fwd(x=None) == 1 and b"NULL" in L.gspn_last_error()
    assert fwd(x=odd) == 3 and b"aligned" in L.gspn_last_error()
    assert L.gspn_scan_bwd(p, p, p, p, None, p, p, p, p, p, 1, 4, 4, 4, 2, 15, 0, None) == 1
    assert L.gspn_merge(None, None, p, 1, 4, 4, 4, 15, 0, None) == 1
    # Eq. 3 normalisation: same validation rules
    assert L.gspn_normalize_fwd(p, p, 0, 2, 4, 4, 15, 0, None) == 1
    assert L.gspn_normalize_fwd(p, p, 1, 2, 4, 4, 0, 0, None) == 1
    assert L.gspn_normalize_fwd(None, p, 1, 2, 4, 4, 15, 0, None) == 1 and b"NULL" in L.gspn_last_error()
    assert L.gspn_normalize_fwd(p, odd, 1, 2, 4, 4, 15, 1, None) == 3
    assert L.gspn_normalize_bwd(p, None, p, 1, 2, 4, 4, 15, 0, None) == 1
    assert L.gspn_normalize_bwd(p, p, p, 1, 2, 4, 4, 15, 9, None) == 1
    # a backward call that asks for no output is a no-op
    assert L.gspn_scan_bwd(p, p, p, p, p, None, None, None, None, None, 1, 4, 4, 4, 2, 15, 0, None) == 0
    assert L.gspn_last_launch_count() == 0


def test_binding_refuses_cpu_tensors():
    import torch
    x = torch.zeros(1, 2, 3, 3)
    with pytest.raises(ValueError):
        gspn.gspn_scan_fwd(x, x, x, x, 1)


def test_sources_do_not_reference_the_oracle():
    """The product path and the oracle share no code and neither imports the other."""
    pkg = os.path.join(ROOT, "paper_2606_00746_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in s.lower() or f == "README.md", f"{f} mentions the oracle"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            s = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2606_00746_b200" not in s and "libgspn.so" not in s


def test_chunk_walk_of_the_fused_host_call_matches_numpy_slicing():
    """gspn_scan_fwd_bwd_host cuts the batch into chunks: a chunk of a [D, B, ...] tensor is [D, bc, ...].  The walk it
    uses for its copies (exported as gspn_debug_chunk_copy, memcpy host to host) against numpy slicing, both ways."""
    import ctypes
    import numpy as np
    import paper_2606_00746_b200 as gspn
    L = gspn.lib()
    rng = np.random.default_rng(5)
    for D, B, per in ((1, 5, 7), (4, 9, 12), (3, 4, 1), (2, 32, 40)):
        t = rng.integers(0, 255, size=(D, B, per), dtype=np.uint8)
        for b0, bc in ((0, 1), (0, B), (B - 1, 1), (B // 2, B - B // 2), (1, max(1, B // 3))):
            chunk = np.zeros((D, bc, per), dtype=np.uint8)
            rc = L.gspn_debug_chunk_copy(chunk.ctypes.data_as(ctypes.c_void_p), t.ctypes.data_as(ctypes.c_void_p), per, D, B, b0, bc, 1)
            assert rc == 0
            np.testing.assert_array_equal(chunk, t[:, b0:b0 + bc])
            back = np.zeros_like(t)
            rc = L.gspn_debug_chunk_copy(chunk.ctypes.data_as(ctypes.c_void_p), back.ctypes.data_as(ctypes.c_void_p), per, D, B, b0, bc, 0)
            assert rc == 0
            np.testing.assert_array_equal(back[:, b0:b0 + bc], t[:, b0:b0 + bc])
            assert back[:, :b0].sum() == 0 and back[:, b0 + bc:].sum() == 0
    assert L.gspn_debug_chunk_copy(None, None, 4, 1, 1, 0, 1, 1) != 0
    assert L.gspn_debug_chunk_copy(chunk.ctypes.data_as(ctypes.c_void_p), t.ctypes.data_as(ctypes.c_void_p), 4, 1, 4, 3, 2, 1) != 0


def test_dir_stride_fields_are_validated_without_gpu(L):
    """gspn_args_t.dir_stride_* (include/gspn.h, reading 6): 0 = one slab shared by every direction,
    GSPN_DIR_STRIDE_DENSE or the dense element count = one slab per direction, anything else GSPN_EINVAL; the round-1
    struct (without the fields) is still accepted.  A backward call that asks for no output validates and returns."""
    from paper_2606_00746_b200 import binding as bd
    buf = ctypes.create_string_buffer(4096 + 16)
    p = (ctypes.addressof(buf) + 15) & ~15
    B, C, H, W, G = 2, 4, 5, 6, 2

    def call(size=None, **kw):
        a = bd._Args(struct_size=ctypes.sizeof(bd._Args) if size is None else size, x=p, w3=p, lam=p, u=p, dy=p,
                     B=B, C=C, H=H, W=W, G=G, dir_mask=15, dtype=0, impl=0,
                     dir_stride_w3=bd.DIR_STRIDE_DENSE, dir_stride_lambda=bd.DIR_STRIDE_DENSE, dir_stride_u=bd.DIR_STRIDE_DENSE)
        for k, v in kw.items():
            setattr(a, k, v)
        return L.gspn_scan_bwd_ex(ctypes.byref(a))

    assert call() == 0
    assert call(dir_stride_w3=0) == 0 and call(dir_stride_lambda=0, dir_stride_u=0) == 0
    assert call(dir_stride_w3=3 * B * G * H * W, dir_stride_lambda=B * C * H * W, dir_stride_u=B * C * H * W) == 0
    assert call(dir_stride_w3=B * C * H * W) == 1 and b"dir_stride_w3" in L.gspn_last_error()
    assert call(dir_stride_u=7) == 1 and b"dir_stride_u" in L.gspn_last_error()
    r1 = bd._Args.dir_stride_w3.offset                      # GSPN_ARGS_SIZE_R1: the struct up to `stream`
    assert r1 == bd._Args.stream.offset + ctypes.sizeof(ctypes.c_void_p)
    assert call(size=r1, dir_stride_w3=12345) == 0          # fields beyond struct_size are not read
    assert call(size=r1 + 8) == 1 and b"struct_size" in L.gspn_last_error()
    # k_chunk (chunked scan): 0 / 1 = global scan, > 1 accepted, negative refused
    assert call(k_chunk=0) == 0 and call(k_chunk=1) == 0 and call(k_chunk=5) == 0
    assert call(k_chunk=-1) == 1 and b"k_chunk" in L.gspn_last_error()
    # flags: GSPN_FLAG_W3_LOGITS accepted, unknown bits refused
    assert call(flags=1) == 0
    assert call(flags=2) == 1 and b"flags" in L.gspn_last_error()
    # the options the naive kernels alone serve are refused by a forced fused kernel before anything is launched
    def fwd_forced(**kw):
        a = bd._Args(struct_size=ctypes.sizeof(bd._Args), x=p, w3=p, lam=p, u=p, y=p, B=B, C=C, H=H, W=W, G=G, dir_mask=15, dtype=0,
                     impl=gspn.IMPL_CHAIN, dir_stride_w3=bd.DIR_STRIDE_DENSE, dir_stride_lambda=bd.DIR_STRIDE_DENSE,
                     dir_stride_u=bd.DIR_STRIDE_DENSE)
        for k, v in kw.items():
            setattr(a, k, v)
        return L.gspn_scan_fwd_ex(ctypes.byref(a))
    assert fwd_forced(dir_stride_w3=0) == 2 and b"naive kernels only" in L.gspn_last_error()
    assert fwd_forced(k_chunk=3) == 2 and fwd_forced(flags=1) == 2
    assert fwd_forced(workspace=p + 8) == 3 and b"workspace" in L.gspn_last_error()
    # the binding's helper: names -> strides
    assert bd._strides(("w3",)) == {"dir_stride_w3": 0, "dir_stride_lambda": bd.DIR_STRIDE_DENSE, "dir_stride_u": bd.DIR_STRIDE_DENSE}
    with pytest.raises(ValueError):
        bd._strides(("x",))

"""pytest plugin used by tests/test_gpu_tests_dryrun_cpu.py (in a child process): runs GPU test files on the CPU with
torch.cuda stubbed and the binding's entry points replaced by the ORACLE's values rounded to the storage type -- the best
result any kernel could return.  What it checks is the tests, not the kernels: fixtures, helper signatures, indexing,
and that the gates accept an exactly rounded result (which is how the element-count condition of the bf16 norm-wise
gate was found to be wrong).  TEST INFRASTRUCTURE; nothing outside that test loads it."""
import sys, os, types, ctypes
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path[:0] = [ROOT, ROOT + "/tests"]
import numpy as np, torch
import gspn_inputs as gi
from oracle import gspn_oracle as orc
import parity_util as pu
import paper_2606_00746_b200 as gspn

cuda = torch.cuda
cuda.is_available = lambda: True
cuda.synchronize = lambda *a, **k: None
cuda.empty_cache = lambda: None
_to = torch.Tensor.to
def to(self, *a, **k):
    a = tuple("cpu" if isinstance(x, str) and x.startswith("cuda") else x for x in a)
    k = {kk: ("cpu" if isinstance(vv, str) and vv.startswith("cuda") else vv) for kk, vv in k.items()}
    return _to(self, *a, **k)
torch.Tensor.to = to
torch.Tensor.cuda = lambda self, *a, **k: self
torch.Tensor.pin_memory = lambda self: self
_mi = gi.make_inputs
gi.make_inputs = lambda cfg, dtype, device="cpu", **k: _mi(cfg, dtype, device="cpu", **k)
_ml = gi.make_logits
gi.make_logits = lambda cfg, dtype, device="cpu", **k: _ml(cfg, dtype, device="cpu", **k)
_full, _empty = torch.full, torch.empty
state = {"v": ""}
n64 = pu.np64
def expand(t, D, shared, name):
    return t.unsqueeze(0).expand(D, *t.shape).contiguous() if name in shared else t
def _naive_only(impl, shared, k_chunk, w3_logits):
    if (shared or k_chunk > 1 or w3_logits) and impl not in (gspn.IMPL_AUTO, gspn.IMPL_NAIVE):
        raise gspn.GspnError(2, "served by the naive kernels only")          # as csrc/gspn_api.cu
def fwd(x, w3, lam, u, G, mask=15, h0=None, out=None, impl=0, shared=(), k_chunk=0, w3_logits=False):
    _naive_only(impl, shared, k_chunk, w3_logits)
    D = bin(mask).count("1")
    w3, lam, u = expand(w3, D, shared, "w3"), expand(lam, D, shared, "lam"), expand(u, D, shared, "u")
    w = orc.normalize(n64(w3), mask) if w3_logits else n64(w3)
    hh = None if h0 is None else n64(h0)
    y = orc.fwd_chunked(n64(x), w, n64(lam), n64(u), G, mask, k_chunk, h0=hh) if k_chunk > 1 else orc.fwd(n64(x), w, n64(lam), n64(u), G, mask, h0=hh)
    t = torch.from_numpy(y).to(x.dtype)
    if out is not None: out.copy_(t); t = out
    state["v"] = "naive_fwd" if (shared or k_chunk > 1 or w3_logits or impl == gspn.IMPL_NAIVE) else {gspn.IMPL_LINE: "line_fwd", gspn.IMPL_CHAIN: "chain_fwd", gspn.IMPL_PLANE: "plane_fwd", gspn.IMPL_FUSED: "fused_fwd_tile", gspn.IMPL_FLAT: "flat_fwd"}.get(impl, "stub_fwd")
    return t
def bwd(x, w3, lam, u, dy, G, mask=15, h0=None, need=("dx", "dlambda", "du", "dw3", "dh0"), impl=0, shared=(), k_chunk=0, w3_logits=False):
    _naive_only(impl, shared, k_chunk, w3_logits)
    D = bin(mask).count("1")
    w3, lam, u = expand(w3, D, shared, "w3"), expand(lam, D, shared, "lam"), expand(u, D, shared, "u")
    w = orc.normalize(n64(w3), mask) if w3_logits else n64(w3)
    hh = None if h0 is None else n64(h0)
    g = orc.bwd_chunked(n64(x), w, n64(lam), n64(u), n64(dy), G, mask, k_chunk, h0=hh) if k_chunk > 1 else orc.bwd(n64(x), w, n64(lam), n64(u), n64(dy), G, mask, h0=hh)
    if w3_logits: g["dw3"] = orc.normalize_bwd(n64(w3), g["dw3"], mask)
    state["v"] = "naive_bwd" if (shared or k_chunk > 1 or w3_logits or impl == gspn.IMPL_NAIVE) else {gspn.IMPL_LINE: "line_bwd", gspn.IMPL_FUSED: "fused_bwd_group", gspn.IMPL_CHAIN: "chain_bwd", gspn.IMPL_PLANE: "plane_bwd"}.get(impl, "stub_bwd")
    return {k: torch.from_numpy(g[k]).to(x.dtype) for k in need}
def fwd_host(x, w3, lam, u, y, G, mask=15, stream=None): y.copy_(fwd(x, w3, lam, u, G, mask))
def bwd_host(x, w3, lam, u, dy, dx, dlambda, du, dw3, dh0, G, mask=15, stream=None):
    g = bwd(x, w3, lam, u, dy, G, mask)
    for k, t in (("dx", dx), ("dlambda", dlambda), ("du", du), ("dw3", dw3), ("dh0", dh0)):
        if t is not None: t.copy_(g[k])
def fb_host(x, w3, lam, u, dy, y, dx, dlambda, du, dw3, dh0, G, mask=15, stream=None):
    if y is not None: fwd_host(x, w3, lam, u, y, G, mask)
    bwd_host(x, w3, lam, u, dy, dx, dlambda, du, dw3, dh0, G, mask)
def norm_fwd(wt, mask=15, out=None):
    r = torch.from_numpy(orc.normalize(n64(wt), mask)).to(wt.dtype); state["v"] = "normalize_fwd_stub"
    if out is not None: out.copy_(r); r = out
    return r
def norm_bwd(wt, dw3, mask=15, out=None):
    r = torch.from_numpy(orc.normalize_bwd(n64(wt), n64(dw3), mask)).to(wt.dtype); state["v"] = "normalize_bwd_stub"
    if out is not None: out.copy_(r); r = out
    return r
for name, f in (("gspn_scan_fwd", fwd), ("gspn_scan_bwd", bwd), ("gspn_scan_fwd_host", fwd_host), ("gspn_scan_bwd_host", bwd_host),
                ("gspn_scan_fwd_bwd_host", fb_host), ("gspn_normalize_fwd", norm_fwd), ("gspn_normalize_bwd", norm_bwd)):
    setattr(gspn, name, f)
    if hasattr(gspn, "binding"): setattr(gspn.binding, name, f)
gspn.gspn_last_variant = lambda: state["v"]
gspn.gspn_last_launch_count = lambda: 1

# log the largest bf16 rel-L2 among gated tensors (n_eff >= 32) and the smallest n_eff that was L2-gated
_gate = pu.gate
_log = {"max_rel_l2": 0.0, "where": None, "count": 0}
def gate_logged(a, b, A, dtype):
    r = _gate(a, b, A, dtype)
    if dtype != "f32" and r.get("n_eff", 0) >= pu.MIN_L2_EFFECTIVE:
        _log["count"] += 1
        if r["rel_l2"] > _log["max_rel_l2"]:
            _log["max_rel_l2"] = r["rel_l2"]; _log["where"] = (tuple(np.shape(b)), round(r["n_eff"], 1))
    return r
pu.gate = gate_logged
def pytest_sessionfinish(session, exitstatus):
    print("\nDRYRUN bf16 L2-gated tensors:", _log)

"""CPU dry run of bench.py main(), run as a script by tests/test_bench_dryrun_cpu.py in a process of its own: torch.cuda
and the binding's entry points are replaced by stand-ins (the 'kernels' call the oracle on shrunken configs), so that
every Python path of the bench -- the timing loop with its L2 flush, roofline, sampled parity, both end-to-end legs and
their fall-back, the other configs, the Table 1 planes, the cpu baseline, the JSON line -- executes once without a GPU.
It checks the bench's bookkeeping, never a number.  BAD=raise / BAD=parity make the fused host call fail / miss parity and
one config's backward unsupported, to walk the fall-back paths.  TEST INFRASTRUCTURE."""
import sys, os, time, types, json
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path[:0] = [ROOT, ROOT + "/tests"]
import torch, numpy as np
import gspn_inputs as gi
from oracle import gspn_oracle as orc
import parity_util as pu

# shrink the configs so that the oracle-backed fake kernels are fast
from dataclasses import replace
for k, c in list(gi.CONFIGS.items()):
    gi.CONFIGS[k] = replace(c, B=min(c.B, 2), C=c.G * 1 if c.C // c.G == 1 else (c.C // c.G) * 2, G=2 if c.C // c.G > 1 else c.G)
    c2 = gi.CONFIGS[k]
    gi.CONFIGS[k] = replace(c2, H=min(c2.H, 12), W=min(c2.W, 12))
gi.CONFIGS["cfg4_2k"] = replace(gi.CONFIGS["cfg4_2k"], H=10, W=16)
_small = gi.small_config
gi.small_config = lambda name, B, C, H, W, G, *a, **kw: _small(name, min(B, 1), C, min(H, 10), min(W, 10), G, *a, **kw)

class Ev:
    def __init__(self, enable_timing=True): self.t = None
    def record(self): self.t = time.perf_counter()
    def elapsed_time(self, o): return (o.t - self.t) * 1e3 + 1e-3
cuda = torch.cuda
cuda.is_available = lambda: True
cuda.set_device = lambda d: None
cuda.current_device = lambda: 0
cuda.synchronize = lambda *a, **k: None
cuda.empty_cache = lambda: None
cuda.Event = Ev
cuda.get_device_properties = lambda d: types.SimpleNamespace(L2_cache_size=1 << 16, name="fake")
class _Stream: cuda_stream = 0
cuda.current_stream = lambda *a, **k: _Stream()
_dev = torch.device
torch.device = lambda *a, **k: _dev("cpu")
_empty = torch.empty
torch.empty = lambda *a, **k: _empty(*a, **{kk: vv for kk, vv in k.items() if kk != "device"})
_mi = gi.make_inputs
gi.make_inputs = lambda cfg, dtype, device="cpu", **k: _mi(cfg, dtype, device="cpu", **k)
_ml = gi.make_logits
gi.make_logits = lambda cfg, dtype, device="cpu", **k: _ml(cfg, dtype, device="cpu", **k)
torch.Tensor.pin_memory = lambda self: self
torch.Tensor.cuda = lambda self, *a, **k: self

import paper_2606_00746_b200 as gspn
state = {"variant": "fake", "n": 0}
def np_(t): return pu.np64(t)
def fake_fwd(x, w3, lam, u, G, mask=15, h0=None, out=None, impl=0, **kw):
    y = orc.fwd(np_(x), np_(w3), np_(lam), np_(u), G, mask)
    t = torch.from_numpy(y).to(x.dtype)
    if out is not None: out.copy_(t); t = out
    state["variant"] = "fake_fwd"; return t
def fake_bwd(x, w3, lam, u, dy, G, mask=15, h0=None, need=("dx","dlambda","du","dw3","dh0"), impl=0, **kw):
    if os.environ.get("BAD") and tuple(x.shape) == UNSUP: raise gspn.GspnError(2, "no kernel holds it")
    g = orc.bwd(np_(x), np_(w3), np_(lam), np_(u), np_(dy), G, mask)
    state["variant"] = "fake_bwd"
    return {k: torch.from_numpy(g[k]).to(x.dtype) for k in need}
def fake_fwd_host(x, w3, lam, u, y, G, mask=15, stream=None): y.copy_(fake_fwd(x, w3, lam, u, G, mask))
def fake_bwd_host(x, w3, lam, u, dy, dx, dlambda, du, dw3, dh0, G, mask=15, stream=None):
    g = fake_bwd(x, w3, lam, u, dy, G, mask)
    for k, t in (("dx", dx), ("dlambda", dlambda), ("du", du), ("dw3", dw3), ("dh0", dh0)): t.copy_(g[k])
def fake_fb_host(x, w3, lam, u, dy, y, dx, dlambda, du, dw3, dh0, G, mask=15, stream=None):
    if os.environ.get("BAD") == "raise": raise gspn.GspnError(5, "fake failure")
    fake_fwd_host(x, w3, lam, u, y, G, mask); fake_bwd_host(x, w3, lam, u, dy, dx, dlambda, du, dw3, dh0, G, mask)
    if os.environ.get("BAD") == "parity": dx.zero_()
def fake_norm_fwd(wt, mask=15, out=None):
    r = torch.from_numpy(orc.normalize(np_(wt), mask)).to(wt.dtype); state["variant"] = "fake_norm"
    if out is not None: out.copy_(r)
    return r
def fake_norm_bwd(wt, dw3, mask=15, out=None):
    r = torch.from_numpy(orc.normalize_bwd(np_(wt), np_(dw3), mask)).to(wt.dtype)
    if out is not None: out.copy_(r)
    return r
gspn.gspn_scan_fwd = fake_fwd; gspn.gspn_scan_bwd = fake_bwd
gspn.gspn_scan_fwd_host = fake_fwd_host; gspn.gspn_scan_bwd_host = fake_bwd_host; gspn.gspn_scan_fwd_bwd_host = fake_fb_host
gspn.gspn_normalize_fwd = fake_norm_fwd; gspn.gspn_normalize_bwd = fake_norm_bwd
gspn.gspn_last_launch_count = lambda: 1
gspn.gspn_last_variant = lambda: state["variant"]
gspn.lib = lambda: None

UNSUP = tuple([gi.CONFIGS["cfg4_2k"].B, gi.CONFIGS["cfg4_2k"].C, gi.CONFIGS["cfg4_2k"].H, gi.CONFIGS["cfg4_2k"].W])
import bench
bench.line_bwd_probe = lambda limit_s=150: {"rc": 0, "results": {"stub": True}}
sys.argv = ["bench.py", "--steps", "3", "--warmup", "3"] + sys.argv[1:]
bench.main()

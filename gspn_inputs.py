"""Seeded synthetic inputs for the GSPN line scan (shared by tests, bench and smoke).

This module holds NONE of the method's arithmetic (no recurrence, no gating, no
merge).  It only draws the operands the method consumes, with the shapes and
value distributions BASELINE.json's five configs state (recipe restated in
DESIGN.md "Input recipe"):

  x, u, dy      ~ N(0,1)
  lambda        ~ U(0,1) (cfg 1) or sigmoid(N(0,1)) (cfg 2-5)
  w3            softmax over the 3 taps of N(0,sigma) logits, out-of-grid taps
                masked to 0, remaining taps renormalised (row-stochastic,
                PAPER.md:94-99); one tap set per channel group, per direction
  h0            zeros (not materialised) unless asked for

Every value is a pure function of (seed, tensor id, direction slab, linear
index in the FULL tensor): a counter-based generator (splitmix64 finaliser ->
24-bit uniforms -> Box-Muller), so any batch slice can be drawn on its own and
equals the same slice of the full tensor.  Values are drawn in fp32 and, for
bf16 storage, rounded once (RNE) -- the oracle and the CUDA path both receive
those rounded values.

The paper's kernel measurements use real activations of trained networks
(PAPER.md:259-290); none are available offline, so these synthetic tensors
stand in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace

import torch

DIR_TB, DIR_BT, DIR_LR, DIR_RL, DIR_ALL = 1, 2, 4, 8, 15

_T_X, _T_W, _T_LAM, _T_U, _T_DY, _T_H0, _T_DW = 1, 2, 3, 4, 5, 6, 7
_MASK63 = (1 << 63) - 1


@dataclass(frozen=True)
class ScanConfig:
    name: str
    B: int
    C: int
    H: int
    W: int
    G: int
    dir_mask: int
    dtypes: tuple          # storage dtypes the config is quoted on
    seed: int
    lam_dist: str = "sigmoid"   # "uniform" | "sigmoid"
    logit_std: float = 1.0
    backward: bool = False

    @property
    def D(self) -> int:
        return bin(self.dir_mask).count("1")

    @property
    def n(self) -> int:
        return self.B * self.C * self.H * self.W

    @property
    def n_w(self) -> int:
        return 3 * self.B * self.G * self.H * self.W

    def fwd_bytes(self, s: int) -> int:
        """Algorithmic bytes of one forward call: x, y once; lambda,u,w3 per direction."""
        return s * (2 * self.n + self.D * (2 * self.n + self.n_w))

    def bwd_bytes(self, s: int) -> int:
        """Algorithmic bytes of one backward call: x,dy read, dx written; per direction
        lambda,u,w3 read and dlambda,du,dw3 written; dh0 written."""
        return (s * (3 * self.n + 2 * self.D * (2 * self.n + self.n_w))
                + s * self.D * self.B * self.C * max(self.H, self.W))


CONFIGS = {
    "cfg1_tiny": ScanConfig("cfg1_tiny", 1, 8, 16, 16, 8, DIR_TB, ("f32",), 0, lam_dist="uniform"),
    "cfg2_cls56": ScanConfig("cfg2_cls56", 64, 192, 56, 56, 24, DIR_ALL, ("f32", "bf16"), 1),
    "cfg3_enc378": ScanConfig("cfg3_enc378", 256, 128, 27, 27, 32, DIR_ALL, ("bf16",), 2),
    "cfg4_2k": ScanConfig("cfg4_2k", 4, 256, 128, 128, 64, DIR_ALL, ("bf16",), 3, logit_std=2.0),
    "cfg5_1k": ScanConfig("cfg5_1k", 32, 128, 73, 73, 32, DIR_ALL, ("bf16",), 4, backward=True),
}


def torch_dtype(name: str):
    return {"f32": torch.float32, "bf16": torch.bfloat16}[name]


def _lsr(z: torch.Tensor, k: int) -> torch.Tensor:
    """Logical shift right of int64 bit patterns."""
    return (z >> k) & ((1 << (64 - k)) - 1)


def _mix(z: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser on int64 bit patterns (wrap-around arithmetic)."""
    z = (z ^ _lsr(z, 30)) * -4658895280553007687      # 0xBF58476D1CE4E5B9
    z = (z ^ _lsr(z, 27)) * -7723592293110705685      # 0x94D049BB133111EB
    return z ^ _lsr(z, 31)


def _key(seed: int, tensor_id: int, slab: int, stream: int) -> int:
    k = (seed * 0x9E3779B97F4A7C15 + tensor_id * 0xD1B54A32D192ED03
         + slab * 0x8CB92BA72F3D8DD7 + stream * 0xABC98388FB8FAC03) & ((1 << 64) - 1)
    return k - (1 << 64) if k >= (1 << 63) else k


def _uniform(idx: torch.Tensor, seed: int, tensor_id: int, slab: int, stream: int) -> torch.Tensor:
    """24-bit uniforms in (0,1), fp32, one per int64 counter in idx."""
    bits = _mix(_mix(idx + _key(seed, tensor_id, slab, stream)) ^ 0x2545F4914F6CDD1D)
    return (_lsr(bits, 40).to(torch.float32) + 0.5) * (1.0 / 16777216.0)


_CHUNK = 1 << 23


def _draw(kind: str, offset: int, count: int, seed: int, tensor_id: int, slab: int,
          device) -> torch.Tensor:
    """count values for linear indices [offset, offset+count) of one slab, fp32."""
    out = torch.empty(count, dtype=torch.float32, device=device)
    for c0 in range(0, count, _CHUNK):
        c1 = min(count, c0 + _CHUNK)
        idx = torch.arange(offset + c0, offset + c1, dtype=torch.int64, device=device)
        u1 = _uniform(idx, seed, tensor_id, slab, 0)
        if kind == "uniform":
            out[c0:c1] = u1
        else:
            u2 = _uniform(idx, seed, tensor_id, slab, 1)
            out[c0:c1] = torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)
    return out


def dir_list(mask: int):
    """Direction ids (0 TB, 1 BT, 2 LR, 3 RL) present in mask, in slab order."""
    return [d for d in range(4) if mask >> d & 1]


def make_inputs(cfg: ScanConfig, dtype: str, device="cpu", batch_slice=None,
                with_dy: bool | None = None, with_h0: bool = False) -> dict:
    """Draw the operands of cfg (optionally only batches [b0,b1)).

    Returns storage-dtype tensors: x [b,C,H,W], w3 [D,b,G,3,H,W], lam,u [D,b,C,H,W],
    optionally dy [b,C,H,W] and h0 [D,b,C,max(H,W)] (N(0,1), entries past the
    direction's cross length left as drawn; consumers ignore them).
    """
    B, C, H, W, G = cfg.B, cfg.C, cfg.H, cfg.W, cfg.G
    b0, b1 = (0, B) if batch_slice is None else batch_slice
    assert 0 <= b0 < b1 <= B
    nb = b1 - b0
    dirs = dir_list(cfg.dir_mask)
    st = torch_dtype(dtype)
    plane = H * W
    out = {}
    out["x"] = _draw("normal", b0 * C * plane, nb * C * plane, cfg.seed, _T_X, 0,
                     device).view(nb, C, H, W).to(st)
    lam, u, w3 = [], [], []
    for q, d in enumerate(dirs):
        off = b0 * C * plane
        cnt = nb * C * plane
        if cfg.lam_dist == "uniform":
            lq = _draw("uniform", off, cnt, cfg.seed, _T_LAM, d, device)
        else:
            lq = torch.sigmoid(_draw("normal", off, cnt, cfg.seed, _T_LAM, d, device))
        lam.append(lq.view(nb, C, H, W))
        u.append(_draw("normal", off, cnt, cfg.seed, _T_U, d, device).view(nb, C, H, W))
        logits = _draw("normal", b0 * G * 3 * plane, nb * G * 3 * plane, cfg.seed, _T_W, d,
                       device).view(nb, G, 3, H, W) * cfg.logit_std
        taps = torch.softmax(logits, dim=2)
        # out-of-grid taps (neighbour -1 at cross position 0, +1 at the last one) -> 0
        if d < 2:       # vertical scan: taps run along j
            taps[:, :, 0, :, 0] = 0.0
            taps[:, :, 2, :, W - 1] = 0.0
        else:           # horizontal scan: taps run along i
            taps[:, :, 0, 0, :] = 0.0
            taps[:, :, 2, H - 1, :] = 0.0
        taps = taps / taps.sum(dim=2, keepdim=True)
        w3.append(taps)
    out["lam"] = torch.stack(lam).to(st).contiguous()
    out["u"] = torch.stack(u).to(st).contiguous()
    out["w3"] = torch.stack(w3).to(st).contiguous()
    if with_dy if with_dy is not None else cfg.backward:
        out["dy"] = _draw("normal", b0 * C * plane, nb * C * plane, cfg.seed, _T_DY, 0,
                          device).view(nb, C, H, W).to(st)
    if with_h0:
        L = max(H, W)
        h0 = [_draw("normal", b0 * C * L, nb * C * L, cfg.seed, _T_H0, d, device).view(nb, C, L)
              for d in dirs]
        out["h0"] = torch.stack(h0).to(st).contiguous()
    return out


def make_logits(cfg: ScanConfig, dtype: str, device="cpu", batch_slice=None, with_dw: bool = False) -> dict:
    """Raw tap logits wt [D,b,G,3,H,W] ~ N(0, logit_std) for the Eq. (3) normalisation (the same draws that
    make_inputs turns into w3), optionally with an upstream gradient dw3 ~ N(0,1) of the same shape."""
    B, G, H, W = cfg.B, cfg.G, cfg.H, cfg.W
    b0, b1 = (0, B) if batch_slice is None else batch_slice
    nb = b1 - b0
    st = torch_dtype(dtype)
    plane = H * W
    wt, dw = [], []
    for d in dir_list(cfg.dir_mask):
        wt.append(_draw("normal", b0 * G * 3 * plane, nb * G * 3 * plane, cfg.seed, _T_W, d,
                        device).view(nb, G, 3, H, W) * cfg.logit_std)
        if with_dw:
            dw.append(_draw("normal", b0 * G * 3 * plane, nb * G * 3 * plane, cfg.seed, _T_DW, d,
                            device).view(nb, G, 3, H, W))
    out = {"wt": torch.stack(wt).to(st).contiguous()}
    if with_dw:
        out["dw3"] = torch.stack(dw).to(st).contiguous()
    return out


def small_config(name: str, B: int, C: int, H: int, W: int, G: int, dir_mask: int = DIR_ALL,
                 seed: int = 100, **kw) -> ScanConfig:
    """Ad-hoc config for parity / edge-case tests."""
    return ScanConfig(name, B, C, H, W, G, dir_mask, ("f32", "bf16"), seed, **kw)


def with_batch(cfg: ScanConfig, B: int) -> ScanConfig:
    return replace(cfg, B=B)

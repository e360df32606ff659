"""Parity gates and case runners shared by the GPU parity tests, smoke() and bench.py's checks.

Tolerances (BASELINE.json north_star: fp32 max relative error <= 1e-5 with
absolute floor 1e-6; bf16 storage + fp32 accumulation <= 3e-3 relative).  `b` is the fp64 oracle on
the SAME (already storage-rounded) inputs, `A` the oracle's magnitude run (sum of |terms| behind
each output), i.e. the scale rounding errors are relative to:

  fp32 : |a-b| <= max(1e-5*A, 1e-6)                                   elementwise
  bf16 : ||a-b||_2 / ||b||_2 <= 3e-3  (tensors of more than 16 elements)  and, elementwise,
         |a-b| <= 0.5*ulp_bf16(max(|a|,|b|))*(1+2^-6) + 1e-5*max(A,1e-6)
         (the fp32 tolerance plus the one unavoidable storage rounding)
"""
from __future__ import annotations

import numpy as np
import torch

import gspn_inputs as gi
from oracle import gspn_oracle as orc


# bf16: the norm-wise gate needs enough elements that carry the norm.  One storage rounding is up to
# 2^-8 relative (3.9e-3) and 1.66e-3 in the root mean square; over n_eff = (sum b^2)^2 / sum b^4 elements of comparable
# weight the ratio |a-b|/|b| of a correctly rounded result scatters around 1.66e-3 by about 2e-3 / sqrt(n_eff), so 3e-3 is
# beyond ten standard deviations from n_eff = 32 on; below that the norm is reported and the elementwise gate -- which
# bounds every element by half an ulp -- decides alone.
MIN_L2_EFFECTIVE = 32.0


def np64(t: torch.Tensor) -> np.ndarray:
    return t.detach().to("cpu", torch.float64).numpy()


def half_ulp_bf16(v: np.ndarray) -> np.ndarray:
    """0.5 ulp of bfloat16 (8 significand bits) at magnitude v."""
    _, ex = np.frexp(np.maximum(np.abs(v), 1e-38))      # |v| = m * 2^ex, m in [0.5,1)
    return np.ldexp(1.0, ex - 9)                        # ulp = 2^(ex-8); half of it


def gate(a: np.ndarray, b: np.ndarray, A: np.ndarray, dtype: str) -> dict:
    """Score GPU result a against oracle b with magnitude A.  Returns metrics + 'ok'."""
    a = np.asarray(a, dtype=np.float64)
    err = np.abs(a - b)
    out = {
        "max_abs_err": float(err.max(initial=0.0)),
        "max_err_over_A": float((err / np.maximum(A, 1e-30)).max(initial=0.0)),
        "literal_rel_max": float((err / np.maximum(np.abs(b), 1e-6)).max(initial=0.0)),
    }
    if dtype == "f32":
        tol = np.maximum(1e-5 * A, 1e-6)
        viol = err > tol
        out["violations"] = int(viol.sum())
        out["ok"] = out["violations"] == 0
    else:
        nb = float(np.linalg.norm(b.ravel()))
        out["rel_l2"] = float(np.linalg.norm((a - b).ravel()) / nb) if nb > 0 else float(err.max(initial=0.0))
        tol = half_ulp_bf16(np.maximum(np.abs(a), np.abs(b))) * (1 + 2.0 ** -6) + 1e-5 * np.maximum(A, 1e-6)
        viol = err > tol
        out["violations"] = int(viol.sum())
        b2 = np.square(b.ravel())
        out["n_eff"] = float(b2.sum() ** 2 / np.square(b2).sum()) if nb > 0 else 0.0
        out["ok"] = out["violations"] == 0 and (out["rel_l2"] <= 3e-3 or out["n_eff"] < MIN_L2_EFFECTIVE)
    out["nonfinite"] = int((~np.isfinite(a)).sum())
    out["ok"] = bool(out["ok"] and out["nonfinite"] == 0)
    return out


def oracle_fwd(t: dict, cfg: gi.ScanConfig):
    """fp64 oracle + magnitude run on the storage-rounded operands of t."""
    x, w3, lam, u = (np64(t[k]) for k in ("x", "w3", "lam", "u"))
    h0 = np64(t["h0"]) if "h0" in t else None
    y = orc.fwd(x, w3, lam, u, cfg.G, cfg.dir_mask, h0=h0)
    A = orc.fwd_magnitude(x, w3, lam, u, cfg.G, cfg.dir_mask, h0=h0)
    return y, A


def oracle_bwd(t: dict, cfg: gi.ScanConfig):
    x, w3, lam, u, dy = (np64(t[k]) for k in ("x", "w3", "lam", "u", "dy"))
    h0 = np64(t["h0"]) if "h0" in t else None
    g = orc.bwd(x, w3, lam, u, dy, cfg.G, cfg.dir_mask, h0=h0)
    A = orc.bwd_magnitude(x, w3, lam, u, dy, cfg.G, cfg.dir_mask, h0=h0)
    return g, A


def check_fwd(cfg: gi.ScanConfig, dtype: str, impl: int = 0, with_h0: bool = False,
              device: str = "cuda:0") -> dict:
    """Whole-tensor forward parity of one (small) config through the C ABI."""
    import paper_2606_00746_b200 as gspn
    t = gi.make_inputs(cfg, dtype, device="cpu", with_h0=with_h0)
    d = {k: v.to(device) for k, v in t.items()}
    y = gspn.gspn_scan_fwd(d["x"], d["w3"], d["lam"], d["u"], cfg.G, cfg.dir_mask,
                           h0=d.get("h0"), impl=impl)
    torch.cuda.synchronize()
    yo, A = oracle_fwd(t, cfg)
    r = gate(np64(y), yo, A, dtype)
    r["variant"] = gspn.gspn_last_variant()
    return r


def check_bwd(cfg: gi.ScanConfig, dtype: str, impl: int = 0, with_h0: bool = False,
              device: str = "cuda:0") -> dict:
    """Whole-tensor backward parity (all five gradients) of one (small) config."""
    import paper_2606_00746_b200 as gspn
    t = gi.make_inputs(cfg, dtype, device="cpu", with_dy=True, with_h0=with_h0)
    d = {k: v.to(device) for k, v in t.items()}
    g = gspn.gspn_scan_bwd(d["x"], d["w3"], d["lam"], d["u"], d["dy"], cfg.G, cfg.dir_mask,
                           h0=d.get("h0"), impl=impl)
    torch.cuda.synchronize()
    variant = gspn.gspn_last_variant()
    go, A = oracle_bwd(t, cfg)
    res = {"variant": variant, "ok": True}
    for k in ("dx", "dlambda", "du", "dw3", "dh0"):
        res[k] = gate(np64(g[k]), go[k], A[k], dtype)
        res["ok"] = res["ok"] and res[k]["ok"]
    return res


def batch_slices(B: int, width: int = 1):
    """First, middle and last batch windows (deduplicated)."""
    starts = sorted({0, max(0, B // 2 - width // 2), max(0, B - width)})
    return [(s, min(B, s + width)) for s in starts]


def _slice(tensors: dict, b0: int, b1: int) -> dict:
    """Images [b0,b1) of the operands the GPU consumed, copied to the host for the oracle."""
    return {k: (v[b0:b1] if k in ("x", "dy") else v[:, b0:b1]).cpu() for k, v in tensors.items()}


def check_fwd_sampled(cfg: gi.ScanConfig, dtype: str, tensors: dict, y: torch.Tensor,
                      width: int = 1) -> dict:
    """Full-size parity on sampled batches: the oracle recomputes whole images b (every (b,group)
    unit is independent) from the very operands the GPU call consumed and is
    compared with those images of the GPU's full output."""
    res = {"ok": True, "slices": []}
    for b0, b1 in batch_slices(cfg.B, width):
        t = _slice(tensors, b0, b1)
        sub = gi.with_batch(cfg, b1 - b0)
        yo, A = oracle_fwd(t, sub)
        r = gate(np64(y[b0:b1]), yo, A, dtype)
        r["batch"] = (b0, b1)
        res["slices"].append(r)
        res["ok"] = res["ok"] and r["ok"]
    return res


def check_bwd_sampled(cfg: gi.ScanConfig, dtype: str, tensors: dict, grads: dict,
                      width: int = 1) -> dict:
    res = {"ok": True, "slices": []}
    for b0, b1 in batch_slices(cfg.B, width):
        t = _slice(tensors, b0, b1)
        sub = gi.with_batch(cfg, b1 - b0)
        go, A = oracle_bwd(t, sub)
        entry = {"batch": (b0, b1)}
        for k in ("dx", "dlambda", "du", "dw3", "dh0"):
            gk = grads[k][b0:b1] if k == "dx" else grads[k][:, b0:b1]
            entry[k] = gate(np64(gk), go[k], A[k], dtype)
            res["ok"] = res["ok"] and entry[k]["ok"]
        res["slices"].append(entry)
    return res


# ---- Eq. (3) normalisation ------------------------------------------------------------
def norm_bwd_magnitude(wt: np.ndarray, dw3: np.ndarray, mask: int) -> np.ndarray:
    """Sum of the absolute values of the terms behind dwt (the oracle's magnitude run)."""
    return orc.normalize_bwd(wt, dw3, mask, magnitude=True)


def check_norm(cfg: gi.ScanConfig, dtype: str, device: str = "cuda:0", batch_slice=None, backward: bool = True) -> dict:
    """Whole-tensor parity of gspn_normalize_fwd / _bwd through the C ABI against the fp64 oracle."""
    import paper_2606_00746_b200 as gspn
    t = gi.make_logits(cfg, dtype, device="cpu", batch_slice=batch_slice, with_dw=backward)
    d = {k: v.to(device) for k, v in t.items()}
    w3 = gspn.gspn_normalize_fwd(d["wt"], cfg.dir_mask)
    variant = gspn.gspn_last_variant()
    wt64 = np64(t["wt"])
    ref = orc.normalize(wt64, cfg.dir_mask)
    out = {"fwd": gate(np64(w3), ref, np.abs(ref), dtype), "variant": variant}
    out["ok"] = out["fwd"]["ok"]
    if backward:
        dwt = gspn.gspn_normalize_bwd(d["wt"], d["dw3"], cfg.dir_mask)
        dw64 = np64(t["dw3"])
        gref = orc.normalize_bwd(wt64, dw64, cfg.dir_mask)
        out["bwd"] = gate(np64(dwt), gref, norm_bwd_magnitude(wt64, dw64, cfg.dir_mask), dtype)
        out["ok"] = bool(out["ok"] and out["bwd"]["ok"])
    return out


def oracle_logits(t: dict, wt: torch.Tensor, cfg: gi.ScanConfig, backward: bool = True):
    """Oracle of the scan fed with tap LOGITS (GSPN_FLAG_W3_LOGITS, second half): the composition of two
    pinned oracle functions, Eq. 3 (normalize) then the scan, and backwards the scan's adjoint then Eq. 3's adjoint.
    Everything in fp64 from the storage-rounded logits; the normalised taps are never rounded (the kernel keeps them in
    fp32 on chip).  Returns (y, A_y, grads, A_grads) with grads["dw3"] = the gradient of the logits."""
    x, lam, u = (np64(t[k]) for k in ("x", "lam", "u"))
    h0 = np64(t["h0"]) if "h0" in t else None
    wl = np64(wt)
    w3 = orc.normalize(wl, cfg.dir_mask)
    y = orc.fwd(x, w3, lam, u, cfg.G, cfg.dir_mask, h0=h0)
    A = orc.fwd_magnitude(x, w3, lam, u, cfg.G, cfg.dir_mask, h0=h0)
    if not backward:
        return y, A, None, None
    dy = np64(t["dy"])
    g = orc.bwd(x, w3, lam, u, dy, cfg.G, cfg.dir_mask, h0=h0)
    Ag = orc.bwd_magnitude(x, w3, lam, u, dy, cfg.G, cfg.dir_mask, h0=h0)
    g["dw3"], Ag["dw3"] = (orc.normalize_bwd(wl, g["dw3"], cfg.dir_mask),
                           orc.normalize_bwd(wl, Ag["dw3"], cfg.dir_mask, magnitude=True))
    return y, A, g, Ag

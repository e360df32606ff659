"""Properties of the seeded synthetic input generator (CPU)."""
import numpy as np
import torch

import gspn_inputs as gi


def test_configs_match_baseline_shapes_and_byte_model():
    c = gi.CONFIGS
    assert (c["cfg1_tiny"].B, c["cfg1_tiny"].C, c["cfg1_tiny"].H, c["cfg1_tiny"].G) == (1, 8, 16, 8)
    assert c["cfg1_tiny"].dir_mask == gi.DIR_TB
    assert (c["cfg2_cls56"].B, c["cfg2_cls56"].C, c["cfg2_cls56"].H, c["cfg2_cls56"].G) == (64, 192, 56, 24)
    assert (c["cfg3_enc378"].B, c["cfg3_enc378"].C, c["cfg3_enc378"].H, c["cfg3_enc378"].G) == (256, 128, 27, 32)
    assert (c["cfg4_2k"].B, c["cfg4_2k"].C, c["cfg4_2k"].H, c["cfg4_2k"].G) == (4, 256, 128, 64)
    assert (c["cfg5_1k"].B, c["cfg5_1k"].C, c["cfg5_1k"].H, c["cfg5_1k"].G) == (32, 128, 73, 32)
    # SURVEY.md 8(d) table
    assert c["cfg1_tiny"].fwd_bytes(4) == 57344
    assert round(c["cfg2_cls56"].fwd_bytes(4) / 1e6, 1) == 1772.6
    assert round(c["cfg4_2k"].fwd_bytes(2) / 1e6, 1) == 436.2
    assert round(c["cfg5_1k"].fwd_bytes(2) / 1e6, 1) == 567.5
    assert round(c["cfg5_1k"].bwd_bytes(2) / 1e6, 1) == 1093.8


def test_taps_are_row_stochastic_and_masked():
    cfg = gi.small_config("t", 2, 4, 5, 7, 2)
    t = gi.make_inputs(cfg, "f32")
    w3 = t["w3"]
    assert w3.shape == (4, 2, 2, 3, 5, 7)
    assert torch.all(w3 >= 0)
    torch.testing.assert_close(w3.sum(dim=3), torch.ones(4, 2, 2, 5, 7), atol=1e-6, rtol=0)
    for q in (0, 1):
        assert torch.all(w3[q, :, :, 0, :, 0] == 0) and torch.all(w3[q, :, :, 2, :, -1] == 0)
    for q in (2, 3):
        assert torch.all(w3[q, :, :, 0, 0, :] == 0) and torch.all(w3[q, :, :, 2, -1, :] == 0)


def test_deterministic_and_sliceable():
    cfg = gi.small_config("t", 4, 4, 6, 5, 2, seed=3, backward=True)
    a = gi.make_inputs(cfg, "bf16", with_h0=True)
    b = gi.make_inputs(cfg, "bf16", with_h0=True)
    s = gi.make_inputs(cfg, "bf16", batch_slice=(1, 3), with_h0=True)
    for k in a:
        assert torch.equal(a[k], b[k])
        full = a[k][1:3] if k in ("x", "dy") else a[k][:, 1:3]
        assert torch.equal(full, s[k]), k
    c = gi.make_inputs(gi.small_config("t", 4, 4, 6, 5, 2, seed=4, backward=True), "bf16")
    assert not torch.equal(a["x"], c["x"])


def test_distributions():
    cfg = gi.small_config("t", 8, 16, 32, 32, 4, seed=9)
    t = gi.make_inputs(cfg, "f32")
    x = t["x"].double().numpy()
    assert abs(x.mean()) < 0.01 and abs(x.std() - 1.0) < 0.01
    lam = t["lam"].double().numpy()
    assert 0.0 < lam.min() and lam.max() < 1.0 and abs(lam.mean() - 0.5) < 0.01
    # the four direction slabs are distinct draws
    assert not np.allclose(t["u"][0].numpy(), t["u"][1].numpy())
    u1 = gi.make_inputs(gi.CONFIGS["cfg1_tiny"], "f32")["lam"].numpy()
    assert 0.0 < u1.min() and u1.max() < 1.0

"""The seeded input generators (paper_2505_22313_b200/synth.py): determinism, ranges, structure."""
import numpy as np
import torch

from paper_2505_22313_b200 import synth


def test_hash_is_deterministic_and_chunk_independent():
    idx = torch.arange(0, 1000, dtype=torch.int64)
    a = synth.hash_u01(5, 0, idx)
    b = torch.cat([synth.hash_u01(5, 0, idx[:333]), synth.hash_u01(5, 0, idx[333:])])
    assert torch.equal(a, b)
    assert not torch.equal(a, synth.hash_u01(5, 1, idx))
    assert not torch.equal(a, synth.hash_u01(6, 0, idx))
    assert float(a.min()) >= 0.0 and float(a.max()) < 1.0
    big = synth.hash_u01(5, 0, idx + (1 << 33))          # 64-bit indices are mixed in
    assert not torch.equal(a, big)
    u = synth.hash_u01(1, 0, torch.arange(0, 1 << 16, dtype=torch.int64)).numpy()
    assert abs(u.mean() - 0.5) < 0.01 and abs(u.var() - 1 / 12) < 0.005


def test_config_table_matches_baseline_json():
    c = synth.CONFIGS
    assert (c["C1"].ny, c["C1"].nx, c["C1"].pitch, c["C1"].z) == (1024, 1024, 1e-6, 1e-3)
    assert c["C2"].lambdas == (450e-9, 550e-9, 650e-9) and c["C2"].ny == 8192
    assert c["C3"].sigma_px == 3.0 and c["C3"].nx == 16384
    assert c["C4"].ny * c["C4"].nx == 1 << 32 and c["C4"].write_intensity
    assert (c["C5"].ny, c["C5"].nx) == (98304, 65536)


def test_recipes_on_small_grids():
    for name, cfg in synth.CONFIGS.items():
        s = cfg.scaled(96, 128)
        h = synth.make_height(s)
        T = synth.make_target(s)
        assert h.shape == (96, 128) and h.dtype == torch.float32 and h.is_contiguous()
        assert float(h.min()) >= 0.0 and float(h.max()) <= s.h_max * (1 + 1e-6), name
        assert float(T.min()) >= 0.0 and float(T.max()) <= 2.0 + 1e-6
        assert torch.equal(h, synth.make_height(s))
    g = synth.make_height(synth.CONFIGS["C3"].scaled(64, 64)).numpy().astype(np.float64)
    lv = g / (1.1e-6 / 255)
    assert np.abs(lv - np.round(lv)).max() < 1e-3 and len(np.unique(np.round(lv))) > 100


def test_tile_plane():
    a = torch.arange(6, dtype=torch.float32).view(2, 3)
    t = synth.tile_plane(a, 2, 2)
    assert t.shape == (4, 6) and torch.equal(t[2:, 3:], a)

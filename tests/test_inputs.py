"""The seeded input recipes: shapes, determinism, structure."""
import numpy as np

from tnlm_inputs import CONFIGS, make_stack, dynamic_range, z_slab


def test_config_table_matches_baseline_json():
    c = CONFIGS
    assert c["config1"].shape == (10, 16, 32, 32) and c["config1"].n_offsets == 27
    assert c["config2"].shape == (10, 64, 128, 128) and c["config2"].n_offsets == 125
    assert c["config3"].shape == (10, 128, 256, 256) and c["config3"].n_iter == 10
    assert c["config4"].shape == (10, 100, 512, 512) and c["config4"].search_radius == 3
    assert c["config5"].shape == (20, 128, 256, 256)
    assert c["config3"].updates_per_sweep == 2 * 10 * 128 * 256 * 256 * 125
    assert c["config1"].updates_per_sweep == 8847360


def test_config1_deterministic_and_structured():
    c = CONFIGS["config1"]
    g1, g2 = make_stack(c), make_stack(c)
    assert g1.dtype == np.float32 and g1.flags.c_contiguous and np.array_equal(g1, g2)
    clean = make_stack(c, clean=True)
    assert set(np.unique(clean)) == {np.float32(0.2), np.float32(1.0), np.float32(1.5)}
    # the sphere's z-centre follows 3 sin(2 pi p / 10)
    zc = [np.argwhere(clean[p] == 1.5)[:, 0].mean() for p in range(10)]
    want = [7.5 + 3 * np.sin(2 * np.pi * p / 10) for p in range(10)]
    assert np.abs(np.array(zc) - np.array(want)).max() < 0.6
    noise = g1 - clean
    assert abs(noise.std() - 0.05) < 0.002 and 1.0 < dynamic_range(g1) < 2.2
    # one standard_normal for the stack == phase-by-phase draws
    rng = np.random.default_rng(c.seed)
    ref = (clean.astype(np.float64) + 0.05 * rng.standard_normal(c.shape)).astype(np.float32)
    assert np.abs(ref - g1).max() < 2e-7      # clean was rounded to fp32 here, not in make_stack


def test_thorax_small_has_moving_tumour_and_phase_varying_streaks():
    c = CONFIGS["config2"].scaled(nz=16, ny=32, nx=32, tumour_radius=2, si_amplitude=3)
    g, clean = make_stack(c), make_stack(c, clean=True)
    assert g.shape == (10, 16, 32, 32)
    vals = np.unique(clean)
    assert {np.float32(0.0), np.float32(0.2), np.float32(0.02), np.float32(1.0), np.float32(0.25)} >= set(vals)
    assert not np.array_equal(clean[0], clean[5])                 # tumour moved
    streak0 = (g[0] - clean[0]).mean(axis=0)
    streak3 = (g[3] - clean[3]).mean(axis=0)
    assert np.abs(streak0).max() > 0.02                           # streaks present, constant in z
    assert np.corrcoef(streak0.ravel(), streak3.ravel())[0, 1] < 0.5   # and differ between phases


def test_z_slab_partition():
    for n, w in [(128, 8), (100, 8), (16, 3), (5, 8)]:
        parts = [z_slab(n, r, w) for r in range(w)]
        assert parts[0][0] == 0 and parts[-1][1] == n
        assert all(parts[i][1] == parts[i + 1][0] for i in range(w - 1))
        sizes = [b - a for a, b in parts]
        assert max(sizes) - min(sizes) <= 1

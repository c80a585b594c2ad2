"""The frozen oracle output under tests/golden/ (written by make_golden.py from the oracle only)."""
import os

import numpy as np

from tnlm_inputs import make_stack

HERE = os.path.dirname(os.path.abspath(__file__))


def load_golden():
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    tab = np.loadtxt(os.path.join(HERE, "golden", "tiny_enhance.txt"))
    cfg = mod.CFG
    g = tab[:, 1].astype(np.float32).reshape(cfg.shape)
    f = tab[:, 2].astype(np.float32).reshape(cfg.shape)
    return cfg, g, f


def test_golden_inputs_are_the_seeded_generator():
    cfg, g, _ = load_golden()
    assert np.array_equal(g, make_stack(cfg))


def test_oracle_reproduces_golden(oracle):
    cfg, g, f = load_golden()
    out = oracle.enhance(g, cfg.patch_radius, cfg.search_radius, np.float32(cfg.h), np.float32(cfg.mu), 2)
    assert np.array_equal(out, f)

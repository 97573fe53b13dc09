"""The input recipe's hard-visibility balance (CPU only): the generator presets carry the visibility bias that
tests/golden/make_vis_bias.py derived from the oracle, and with it the oracle's hard visibility [z_v > 0] is neither
all-occluded nor all-visible at primary points and at secondary hits (the paper's renderer uses
hard visibility, so a config whose rays are all occluded would compare black frames)."""
import os
import sys

import numpy as np
import pytest

import gen

GOLD = os.path.join(os.path.dirname(__file__), "golden")
sys.path.insert(0, GOLD)


def _golden():
    rows = {}
    for line in open(os.path.join(GOLD, "vis_bias.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, b, fp, fs = line.split()
        rows[name] = (float(b), float(fp), float(fs))
    return rows


def test_presets_carry_the_golden_vis_bias():
    g = _golden()
    for name in ("C0", "C1", "C2", "C3", "C4"):
        assert gen.make_config(name).vis_bias == g[name][0]
    assert gen.make_config("C3a").vis_bias == g["C3"][0]           # same seed, same model
    cfg = gen.make_config("C2")
    w = gen.split_mlp(cfg, "irt", gen.make_mlp(cfg, "irt"))
    assert w[2][1][0] == np.float32(cfg.vis_bias) and w[2][1][1] == np.float32(cfg.depth_bias)


@pytest.mark.parametrize("name,over", [("C0", dict(S_i=4, S_2=3, flags=7)), ("C1", {}), ("C2", {}), ("C3", {}),
                                       ("C4", dict(log2_T=16)), ("C4", dict(log2_T=22))])
def test_hard_visibility_is_balanced(name, over):
    from make_vis_bias import logits
    cfg = gen.make_config(name, **over)
    zp, zs = logits(name, cfg.vis_bias, npix=96, **over)
    fp = (zp > 0).mean()
    assert 0.3 <= fp <= 0.7, fp
    if zs is not None:
        fs = (zs > 0).mean()
        assert 0.3 <= fs <= 0.7, fs

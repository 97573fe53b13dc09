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


def test_bench_gather_counts_match_a_count_over_the_oracle_indices():
    """bench.py's L1 roofline of the encode (roofline.l1_gather) prices `sectors` and `loads` per point.  For the levels that are
    not cell-major the device row of a hashed level IS the specified index, so the sectors a point touches can be counted from
    the oracle's corner indices: distinct (index // rows per sector) among a level's 8 corners, averaged over random points."""
    import importlib.util
    from oracle.oracle import Oracle
    spec = importlib.util.spec_from_file_location("bench", os.path.join(os.path.dirname(GOLD), "..", "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    cfg = gen.make_config("C4")                                        # fp16 rows: 8 per 32-byte sector
    m = gen.make_model(cfg)
    o = Oracle.from_gen(cfg, m)
    x = np.random.default_rng(5).random((20000, 3), dtype=np.float32)
    _, idx, _ = o.encode(x)
    hashed = [l for l in range(cfg.L) if (int(m["res"][l]) + 1) ** 3 > cfg.T]
    for rows_per_sector in (8, 4):
        counted = np.mean([[len(set((idx[i, l] // rows_per_sector).tolist())) for l in hashed] for i in range(0, 20000, 10)])
        model_sectors, model_loads = bench.gather_counts(1, 0, rows_per_sector)
        assert model_loads == (6 if rows_per_sector == 8 else 8)      # fp16 rows: a two-row load per x-pair + the neighbour for odd cx
        assert abs(counted - model_sectors) < 0.05 * model_sectors, (rows_per_sector, counted, model_sectors)
    # cell-major levels: one entry = 8 rows = exactly one sector of fp16 rows, two of fp32 rows
    assert bench.gather_counts(16, 16, 8) == (16, 16) and bench.gather_counts(16, 16, 4) == (32, 32)
    assert bench.gather_counts(16, 6, 8) == (6 + 10 * 4.5, 6 + 60) and bench.gather_counts(16, 5, 4) == (10 + 11 * 5.0, 10 + 88)

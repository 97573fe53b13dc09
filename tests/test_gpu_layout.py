"""The device layout of the tables (cell-major copies of the coarsest levels, hashrender_table_layout) and the gather probe.
The values a cell-major level returns are checked by every encode / trace / frame parity test (the layout is the default); this
file checks that those tests really run through BOTH kinds of cell-major level -- dense ones and hashed ones -- and that the
budget rule of hashrender_create holds."""
import numpy as np
import pytest

import gen
from hr_testutil import make_renderer, to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available()
    return torch


def _expected_cell_major(cfg, res, l2_bytes):
    esz = 8 if cfg.table_dtype == "f32" else 4
    table = cfg.L * cfg.T * esz
    budget = l2_bytes // 4 if table <= l2_bytes else 4 * table      # (the free-memory cap of hashrender_create is far away on a test box)
    n, cum = 0, 0
    for N in res:
        b = int(N) ** 3 * 8 * esz
        if cum + b > budget:
            break
        cum += b
        n += 1
    return n, cum


@pytest.mark.parametrize("name,over", [("C0", {}), ("C3", {"N": 640000}), ("C4", {"log2_T": 16}), ("C4", {"log2_T": 22})])
def test_cell_major_levels_follow_the_budget_and_cover_hashed_levels(torch, name, over):
    cfg = gen.make_config(name, **over)
    model = gen.make_model(cfg)
    r = make_renderer(cfg, model)
    nblock, dev_bytes = r.table_layout()
    l2 = torch.cuda.get_device_properties(0).L2_cache_size
    res = [int(v) for v in model["res"]]
    want, cum = _expected_cell_major(cfg, res, l2)
    assert nblock == want and 1 <= nblock <= cfg.L
    assert dev_bytes >= cum
    hashed = [l for l in range(nblock) if (res[l] + 1) ** 3 > cfg.T]
    dense = [l for l in range(nblock) if (res[l] + 1) ** 3 <= cfg.T]
    if name in ("C0", "C4"):
        assert hashed and dense, "the parity tests on this config must cover dense AND hashed cell-major levels"
    # the cell-major copy returns exactly the rows the specified index names: features at random points against
    # interpolating the caller's table at the indices hashrender_encode reports
    rng = np.random.default_rng(7)
    x = rng.random((4096, 3), dtype=np.float32)
    x[:8] = [[0, 0, 0], [1, 1, 1], [1, 0, 0], [0, 1, 0], [0, 0, 1], [1, 1, 0], [0.5, 1, 1], [1, 0.25, 1]]
    feat = torch.empty((4096, 2 * cfg.L), device="cuda")
    idx = torch.empty((4096, cfg.L, 8), device="cuda", dtype=torch.int32)
    w = torch.empty((4096, cfg.L, 3), device="cuda")
    r.encode(to_dev(x), feat, idx=idx, w=w)
    torch.cuda.synchronize()
    idx_h, w_h, f_h = idx.cpu().numpy().astype(np.int64), w.cpu().numpy(), feat.cpu().numpy()
    tab = model["tables"].astype(np.float32)
    if cfg.table_dtype == "f16":
        tab = tab.astype(np.float16).astype(np.float32)
    for l in range(nblock):
        rows = tab[l][idx_h[:, l, :]]                                 # [n, 8, 2]
        wx, wy, wz = w_h[:, l, 0], w_h[:, l, 1], w_h[:, l, 2]
        f = np.zeros((4096, 2), np.float32)
        for k in range(8):
            wt = ((wx if k & 1 else np.float32(1) - wx) * (wy if k & 2 else np.float32(1) - wy)).astype(np.float32)
            wt = (wt * (wz if k & 4 else np.float32(1) - wz)).astype(np.float32)
            f = (f.astype(np.float64) + wt[:, None].astype(np.float64) * rows[:, k, :].astype(np.float64))   # fma: one rounding
            f = f.astype(np.float32)
        # (the fp64 emulation of fmaf can differ from it by a double rounding: one ulp of the feature; a wrong row is O(table scale))
        np.testing.assert_allclose(f, f_h[:, 2 * l:2 * l + 2], rtol=0, atol=3e-7 * float(np.abs(tab[l]).max()), err_msg=f"level {l}")
    r.destroy()


def test_probe_gather_reports_a_sane_rate(torch):
    from paper_2409_10327_b200.binding import HashRenderError, probe_gather
    miss, per_s = probe_gather(32 << 20, 4, 1, 160 << 10)              # L2-resident table, L1 misses
    pair, _ = probe_gather(32 << 20, 4, 2, 160 << 10)
    hit, _ = probe_gather(16 << 10, 4, 1, 160 << 10)                   # L1-resident table
    print(f"probe: {miss:.3f} loads/cycle/SM on misses ({per_s / 1e9:.0f} G loads/s), {pair:.3f} with two loads per sector, {hit:.3f} on L1 hits")
    assert 0.5 < miss < 1.3 and miss < pair < 2.0 * miss + 0.1 and hit > 2.0 * miss
    with pytest.raises(HashRenderError):
        probe_gather(3000, 4, 1, 0)                                    # not a power of two
    with pytest.raises(HashRenderError):
        probe_gather(1 << 20, 16, 3, 0)                                # unsupported shape


@pytest.mark.parametrize("over", [dict(L=3, log2_T=5, base_res=1, max_res=6),            # res 1, 2, 6: a one-cell level, dense and hashed mixed
                                  dict(L=4, log2_T=3, base_res=2, max_res=40),           # T = 8 rows: every level hashed, heavy collisions
                                  dict(L=16, log2_T=10, base_res=16, max_res=2048, table_dtype="f16", mlp_dtype="f16")])
def test_degenerate_grids_encode_bit_exact(torch, over):
    """Tiny tables and coarse grids: all (or the first six) levels end up cell-major, most of them hashed with many cells
    sharing a row.  Indices and fractional positions bit-exact against the oracle, features to rounding."""
    from hr_testutil import check_close
    from oracle.oracle import Oracle
    cfg = gen.make_config("C0", table_scale=0.5, **over)
    m = gen.make_model(cfg)
    o = Oracle.from_gen(cfg, m)
    rng = np.random.default_rng(11)
    n = 3000
    x = rng.random((n, 3), dtype=np.float32)
    x[:6] = [[0, 0, 0], [1, 1, 1], [1, 0, 0.5], [0.5, 0.5, 0.5], [0.999999, 1e-7, 1], [-0.5, 2.0, 0.25]]     # clamped (Q6)
    feat_o, idx_o, w_o = o.encode(x)
    r = make_renderer(cfg, m)
    nblock, _ = r.table_layout()
    assert nblock == (cfg.L if cfg.L <= 4 else 6)                    # the 16-level grid: levels 0-5 fit the budget, T = 1024 rows hash the rest
    feat = torch.empty((n, cfg.D), device="cuda"); idx = torch.empty((n, cfg.L, 8), device="cuda", dtype=torch.int32)
    w = torch.empty((n, cfg.L, 3), device="cuda")
    r.encode(to_dev(x), feat, idx, w)
    torch.cuda.synchronize()
    assert np.array_equal(idx.cpu().numpy().view(np.uint32), idx_o)
    assert np.array_equal(w.cpu().numpy(), w_o)
    check_close(feat.cpu().numpy(), feat_o, 2e-6, what=f"encode {over}")
    r.destroy()

"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on identical seeded inputs.

Bars (BASELINE.json north_star; Q32/Q33): hash indices / corner selection / fractional weights
bit-exact; floating point within 1e-4 relative (fp32) or 3e-3 (fp16 tables/weights), relative to
max(|o|, mean|o|); hard visibility may flip only where |z_v| < delta (flipbound rule).
"""
import numpy as np
import pytest

import gen
from hr_testutil import check_close, gpu_render, make_renderer, oracle_render, to_dev

pytestmark = pytest.mark.gpu

TOL32, TOL16 = 1e-4, 3e-3
# |z_v| band in which a hard-visibility flip is legitimate (Q33): <= 3x the largest |z_v(gpu) - z_v(oracle)|
# the stage-wise tests below measure on the production arithmetic (test_decode_trace_shade_stagewise prints and bounds it).
DELTA32, DELTA16 = 5e-6, 5e-4
# share of the reference radiance that the hard-mode flip allowance may amount to (mean flipbound / mean |o|): the allowance
# must stay an exception.  fp16: a sample may flip inside |z_v| < 5e-4 (measured error of the fp16 arithmetic: 1.0e-4 stage-wise,
# 1.3e-4 at the render kernel's own visibility bits) while the logits of these synthetic models spread over only +-0.1.
FLIPSHARE32, FLIPSHARE16 = 2e-3, 0.05


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available()
    return torch


def _oracle(cfg, model, **kw):
    from oracle.oracle import Oracle
    return Oracle.from_gen(cfg, model, **kw)


def _edge_points(rng, n):
    x = rng.random((n, 3)).astype(np.float32)
    x[:8] = [[0, 0, 0], [1, 1, 1], [0.5, 0.25, 0.125], [1, 0, 0.5], [3 / 16, 5 / 16, 1.0], [1e-8, 1 - 1e-7, 0.999999],
             [-0.5, 2.0, 0.3], [0.0625, 0.9375, 0.5]]
    return x


# ---------------------------------------------------------------------------------------------- encode
@pytest.mark.parametrize("name,n", [("C0", 4096), ("C1", 3001), ("C3", 1537)])
def test_encode_bit_exact_indices_and_features(torch, name, n):
    cfg = gen.make_config(name)
    m = gen.make_model(cfg)
    o = _oracle(cfg, m)
    rng = np.random.default_rng(100)
    x = _edge_points(rng, n)
    if name == "C0":
        x[8:] = gen.make_points(cfg)[0][8:n]
    feat_o, idx_o, w_o = o.encode(x)
    r = make_renderer(cfg, m)
    feat = torch.empty((n, cfg.D), device="cuda"); idx = torch.empty((n, cfg.L, 8), device="cuda", dtype=torch.int32)
    w = torch.empty((n, cfg.L, 3), device="cuda")
    r.encode(to_dev(x), feat, idx, w)
    torch.cuda.synchronize()
    assert np.array_equal(idx.cpu().numpy().view(np.uint32), idx_o), "hash / dense indices must be bit-exact"
    assert np.array_equal(w.cpu().numpy(), w_o), "fractional positions must be bit-exact"
    check_close(feat.cpu().numpy(), feat_o, 2e-6, what=f"encode {name}")
    # vertex reproduction on the GPU too: x on a level-0 vertex returns the table row exactly
    v = np.array([[3 / 16, 5 / 16, 9 / 16]], np.float32)
    f1 = torch.empty((1, cfg.D), device="cuda")
    r.encode(to_dev(v), f1)
    row = 3 + 5 * 17 + 9 * 17 * 17
    assert np.array_equal(f1.cpu().numpy()[0, :2], m["tables"][0, row])


def test_encode_empty_and_errors(torch):
    from paper_2409_10327_b200 import HashRenderError
    cfg = gen.make_config("C0")
    m = gen.make_model(cfg)
    r = make_renderer(cfg, m)
    feat = torch.empty((4, cfg.D), device="cuda")
    r.encode(to_dev(np.zeros((0, 3), np.float32)), feat)            # N == 0: no-op
    with pytest.raises(HashRenderError) as e:
        r.encode(None, feat, N=4)
    assert e.value.code == 1
    with pytest.raises(HashRenderError):
        r.encode(to_dev(np.zeros((4, 3), np.float32)), feat, N=cfg.N * 1000)     # N > max_points
    with pytest.raises(HashRenderError) as e:
        make_renderer(cfg, m, F=4, tables=np.zeros((cfg.L, cfg.T, 4), np.float32),
                      brdf_w=np.zeros(64 * 32 + 64 + 64 * 64 + 64 + 7 * 64 + 7, np.float32),
                      irt_w=np.zeros(64 * 35 + 64 + 64 * 64 + 64 + 2 * 64 + 2, np.float32))
    assert e.value.code == 4


# ---------------------------------------------------------------------------------------------- decode / trace / shade
@pytest.mark.parametrize("name", ["C0", "C1", "C2", "C3"])
def test_decode_trace_shade_stagewise(torch, name):
    """Stage-wise parity on ORACLE-supplied inputs (the strict test, SURVEY 8(c) conditioning note).  hashrender_trace runs the
    tensor-core arithmetic render_frame runs for this model (fp32 models: hi/lo split precision, `tcgen05-f16x3`), with the
    oracle's features and with the encode fused; the largest |z_v(gpu) - z_v(oracle)| is printed and must stay below a third
    of the hard-visibility flip band."""
    cfg = gen.make_config(name)
    m = gen.make_model(cfg)
    n = 777
    pix = np.arange(0, cfg.N, cfg.N // n)[:n]
    fr = gen.make_frame(cfg, m["env"], pix)
    tol = TOL16 if cfg.mlp_dtype == "f16" else TOL32
    o = _oracle(cfg, m)
    feat_o, _, _ = o.encode(fr["x"])
    brdf_o = o.decode(feat_o)
    vis_o, zv_o, t_o, xs_o = o.trace(fr["x"], feat_o, fr["dir_d"])
    r = make_renderer(cfg, m)
    featd = to_dev(feat_o.astype(np.float32))
    S = cfg.S_d
    # decode
    brdf = torch.empty((n, 7), device="cuda")
    r.decode(featd, brdf)
    check_close(brdf.cpu().numpy(), brdf_o, tol, what="decode")
    # trace on oracle features, then with the encode fused
    from paper_2409_10327_b200 import DirSet
    ds = DirSet(to_dev(fr["dir_d"]), to_dev(fr["pdf_d"]))
    delta = DELTA16 if cfg.mlp_dtype == "f16" else DELTA32
    for fused in (False, True):
        vis = torch.empty((n, S), device="cuda"); zv = torch.empty((n, S), device="cuda"); t = torch.empty((n, S), device="cuda")
        xs = torch.empty((n, S, 3), device="cuda")
        r.trace(to_dev(fr["x"]), None if fused else featd, ds, vis, zv, t, xs)
        torch.cuda.synchronize()
        assert r.last_path() == ("tcgen05-f16" if cfg.mlp_dtype == "f16" else "tcgen05-f16x3"), r.last_path()
        check_close(vis.cpu().numpy(), vis_o, tol, what="trace vis")
        check_close(t.cpu().numpy(), t_o, tol, what="trace t")
        check_close(zv.cpu().numpy(), zv_o, tol, extra=tol * 0.05, what="trace zv")
        check_close(xs.cpu().numpy(), xs_o, tol, what="trace x'")
        dzv = float(np.abs(zv.cpu().numpy() - zv_o).max())
        dt = float(np.abs(t.cpu().numpy() - t_o).max())
        print(f"[stagewise {name} fused={fused}] path={r.last_path()} max|dz_v|={dzv:.3e} max|dt|={dt:.3e} (delta={delta:g})")
        assert 3.0 * dzv <= delta, f"flip band {delta} must be >= 3x the measured z_v error {dzv:.3e}"
    # hard mode: bits agree wherever |z_v| >= delta
    oh = _oracle(cfg, m, vis_mode=1)
    vh_o, zvh_o, _, _ = oh.trace(fr["x"], feat_o, fr["dir_d"])
    rh = make_renderer(cfg, m, vis_mode=1)
    vis = torch.empty((n, S), device="cuda"); t = torch.empty((n, S), device="cuda")
    rh.trace(to_dev(fr["x"]), featd, ds, vis, None, t)
    vh = vis.cpu().numpy()
    assert set(np.unique(vh)) <= {0.0, 1.0}
    sure = np.abs(zvh_o) >= delta
    assert np.array_equal(vh[sure], vh_o[sure])
    assert sure.mean() > 0.9
    assert 0.2 <= vh_o.mean() <= 0.8, "hard visibility must be balanced (gen vis_bias)"
    # shade: direct only, then Eq. 2 on one set with a synthetic L'_o
    rng = np.random.default_rng(5)
    Lind = rng.random((n, S, 3)).astype(np.float32)
    for terms, li in ((1, None), (3, Lind), (2, Lind)):
        rgb_o = o.shade(brdf_o, fr["wo"], fr["dir_d"], fr["pdf_d"], vis_o, Lind=li, terms=terms)
        rgb = torch.empty((n, 3), device="cuda")
        r.shade(to_dev(brdf_o.astype(np.float32)), to_dev(fr["wo"]), ds, to_dev(vis_o.astype(np.float32)),
                None if li is None else to_dev(li), terms, rgb)
        check_close(rgb.cpu().numpy(), rgb_o, TOL32, what=f"shade terms={terms}")


def test_trace_shared_set_and_ragged(torch):
    cfg = gen.make_config("C0")
    m = gen.make_model(cfg)
    o = _oracle(cfg, m)
    from paper_2409_10327_b200 import DirSet
    for n in (1, 31, 257, 1000):
        fr = gen.make_frame(cfg, m["env"], np.arange(n))
        feat_o, _, _ = o.encode(fr["x"])
        vis_o, zv_o, t_o, xs_o = o.trace(fr["x"], feat_o, fr["dir_t"], shared=True)
        r = make_renderer(cfg, m)
        S = cfg.S_2
        vis = torch.empty((n, S), device="cuda"); t = torch.empty((n, S), device="cuda"); xs = torch.empty((n, S, 3), device="cuda")
        r.trace(to_dev(fr["x"]), None, DirSet(to_dev(fr["dir_t"]), to_dev(fr["pdf_t"])), vis, None, t, xs)
        check_close(vis.cpu().numpy(), vis_o, TOL32, what="trace shared vis")
        check_close(xs.cpu().numpy(), xs_o, TOL32, what="trace shared x'")


# ---------------------------------------------------------------------------------------------- whole frames
def _frame_case(torch, name, pix, vis_mode, flags=None, over=None, tol=None, delta=None, brdf=None, mask=None):
    cfg = gen.make_config(name, **(over or {}))
    m = gen.make_model(cfg)
    fr = gen.make_frame(cfg, m["env"], pix)
    f16 = cfg.mlp_dtype == "f16"
    tol = tol or (TOL16 if f16 else TOL32)
    delta = delta if delta is not None else (DELTA16 if f16 else DELTA32)
    o = _oracle(cfg, m, vis_mode=vis_mode)
    ref = oracle_render(o, cfg, fr, flags=flags, delta=delta if vis_mode else 0.0, brdf=brdf, mask=mask)
    r = make_renderer(cfg, m, vis_mode=vis_mode)
    got = gpu_render(r, cfg, fr, flags=flags, brdf=brdf, mask=mask)
    worst = check_close(got, ref["rgb"], tol, extra=ref["flipbound"] if vis_mode else None, what=f"{name} vis_mode={vis_mode}")
    _nontrivial(name, cfg, m, fr, ref, vis_mode, mask, worst)
    return cfg, ref, got, worst, r


def _nontrivial(name, cfg, m, fr, ref, vis_mode, mask=None, worst=float("nan")):
    """The reference must be a real image, hard visibility must be balanced, and the flip allowance an exception."""
    live = np.ones(len(fr["x"]), bool) if mask is None else np.asarray(mask, bool)
    mean_o = float(np.abs(ref["rgb"][live]).mean())
    assert mean_o > 0.05, f"{name}: reference image is (nearly) black: mean|o| = {mean_o:.4g}"
    msg = f"[frame {name} vis_mode={vis_mode}] pixels={len(fr['x'])} mean|o|={mean_o:.4f} worst err/allowed={worst:.3f}"
    if vis_mode:
        o = _oracle(cfg, m, vis_mode=1)
        feat, _, _ = o.encode(fr["x"])
        vfrac = float(o.trace(fr["x"], feat, fr["dir_d"])[0].mean())
        assert 0.2 <= vfrac <= 0.8, f"{name}: hard-visibility visible fraction {vfrac:.3f} outside [0.2, 0.8]"
        fb = ref["flipbound"][live]
        share_el = float((fb > 0).mean())
        share_mag = float(fb.mean() / mean_o)
        lim = FLIPSHARE16 if cfg.mlp_dtype == "f16" else FLIPSHARE32
        assert share_mag <= lim, f"{name}: flip allowance is {share_mag:.3g} of the mean radiance (limit {lim})"
        msg += f" visible={vfrac:.3f} elements with a flip allowance={share_el:.3f} mean flipbound/mean|o|={share_mag:.2e}"
    print(msg)


@pytest.mark.parametrize("vis_mode", [0, 1])
def test_frame_C0_full(torch, vis_mode):
    cfg, ref, got, worst, _ = _frame_case(torch, "C0", None, vis_mode)
    assert np.abs(ref["rgb"]).max() > 0.1
    if vis_mode:          # the flip allowance must stay a rare exception, not the rule
        assert (ref["flipbound"].max(axis=1) > 0).mean() < 0.05


@pytest.mark.parametrize("vis_mode", [0, 1])
def test_frame_C1_subset(torch, vis_mode):
    pix = np.concatenate([np.arange(0, 640000, 313), [0, 799, 639200, 639999]])
    _frame_case(torch, "C1", pix, vis_mode)


@pytest.mark.parametrize("vis_mode", [0, 1])
def test_frame_C2_subset(torch, vis_mode):
    """One-bounce indirect, fp32: 1e-4 (soft); hard adds the flip allowance."""
    pix = np.concatenate([np.arange(0, 640000, 1259), [0, 799, 639200, 639999]])
    cfg, ref, got, worst, _ = _frame_case(torch, "C2", pix, vis_mode)
    assert ref["n_sec"] == len(pix) * 64


@pytest.mark.parametrize("name", ["C3", "C3a"])
@pytest.mark.parametrize("vis_mode", [0, 1])
def test_frame_C3_fp16_subset(torch, name, vis_mode):
    pix = np.concatenate([np.arange(0, 640000, 1259), [0, 799, 639200, 639999]])
    _frame_case(torch, name, pix, vis_mode)


@pytest.mark.parametrize("table_scale,tolv", [(0.1, TOL32), (1.0, 4e-4)])
def test_frame_variants_small(torch, table_scale, tolv):
    """External BRDF (Q30), mask (Q27), Lambert model, flag subsets, per-secondary-point tertiary sets (the TSHARED = false,
    G = 2 kernels), ragged N.  On a 0.1-scale table (the scale of BASELINE configs 1-3) every variant holds north_star's 1e-4.
    The second run keeps C0's own U(-1,1) table WITH an indirect bounce, an off-spec combination: the fp32 error of t (~4e-6)
    moves x' and is amplified by N_max * |grad tab| ~ 256 * 2 into a ~1e-3 feature error at the finest level (SURVEY 8(c)
    conditioning note), so it is an extra at 4e-4, not the bar."""
    rng = np.random.default_rng(9)
    n = 333
    pix = np.arange(n)
    over = dict(S_i=4, S_2=3, flags=7, table_scale=table_scale)
    cfg = gen.make_config("C0", **over)
    brdf = np.concatenate([gen._normalize(rng.standard_normal((n, 3))), rng.random((n, 3)), 0.09 + 0.91 * rng.random((n, 1))], 1).astype(np.float32)
    mask = (rng.random(n) > 0.3).astype(np.uint8)
    _frame_case(torch, "C0", pix, 0, over=over, brdf=brdf, mask=mask, tol=tolv)
    for flags in (1, 3):
        _frame_case(torch, "C0", pix, 0, flags=flags, over=over)
    for flags in (4, 6, 5):
        _frame_case(torch, "C0", pix, 0, flags=flags, over=over, tol=tolv)
    # Lambert
    m = gen.make_model(cfg); fr = gen.make_frame(cfg, m["env"], pix)
    o = _oracle(cfg, m, brdf_model=0)
    ref = oracle_render(o, cfg, fr, flags=7)
    got = gpu_render(make_renderer(cfg, m, brdf_model=0), cfg, fr, flags=7)
    check_close(got, ref["rgb"], tolv, what="lambert")
    # per-secondary-point tertiary sets (point_stride != 0, the paper's literal reading of PAPER.md:344)
    dt = gen._normalize(rng.standard_normal((n * 4, 3, 3))).astype(np.float32)
    dt = gen._normalize(dt.astype(np.float64)).astype(np.float32)
    pt = np.full((n * 4, 3), 1 / (4 * np.pi), np.float32)
    fr2 = dict(fr); fr2["dir_t"], fr2["pdf_t"] = dt, pt
    o = _oracle(cfg, m)
    ref = oracle_render(o, cfg, fr2, flags=7)
    r = make_renderer(cfg, m)
    got = gpu_render(r, cfg, fr2, flags=7)
    assert r.last_path() == "tcgen05-f16x3"
    check_close(got, ref["rgb"], tolv, what="per-point tertiary")
    # the same per-point sets with an fp16 model (the G = 2 instantiation of the fp16 kernel)
    cfgh = gen.make_config("C0", **over, table_dtype="f16", mlp_dtype="f16")
    mh = gen.make_model(cfgh)
    ref = oracle_render(_oracle(cfgh, mh), cfgh, fr2, flags=7)
    rh = make_renderer(cfgh, mh)
    got = gpu_render(rh, cfgh, fr2, flags=7)
    assert rh.last_path() == "tcgen05-f16"
    check_close(got, ref["rgb"], TOL16 if table_scale < 1 else 4 * TOL16, what="per-point tertiary fp16")


@pytest.mark.parametrize("L,S_2", [(8, 8), (14, 8), (5, 16)])
def test_prefetched_encode_with_fewer_than_16_levels(torch, L, S_2):
    """fp32 model, indirect bounce, SHARED tertiary set with S_2 >= 8: the split-precision kernel encodes the next group of
    secondary points while it runs the tertiary queries of the current one (two levels per query).  Levels l >= L do not
    exist -- their table slice would lie past the allocation -- so they must be skipped and read as zero features.  L = 14 is
    the paper's own grid, S_2 = 8 its tertiary count."""
    over = dict(S_i=8, S_2=S_2, flags=7, L=L, table_scale=0.1, max_res=256 if L <= 8 else 1024, log2_T=14 if L <= 8 else 17)
    n = 700                                               # 5600 secondary items: many 128-item groups follow one another
    cfg, ref, got, worst, r = _frame_case(torch, "C0", np.arange(n), 0, over=over)
    assert r.last_path() == "tcgen05-f16x3" and ref["n_sec"] == n * 8
    # the table is the last allocation the handle made that a stray gather could run past: render again right after creating and
    # destroying a neighbour handle, and with HR_DENSE
    from paper_2409_10327_b200 import HR_DENSE
    m = gen.make_model(cfg); fr = gen.make_frame(cfg, m["env"], np.arange(n))
    got2 = gpu_render(r, cfg, fr, flags=7 | HR_DENSE)
    np.testing.assert_allclose(got2, got, rtol=5e-6, atol=1e-7)


def test_frame_closed_form_on_gpu(torch):
    """The a*L closed form (Eq. 1) evaluated by the CUDA path itself: Lambert, v == 1, constant env,
    cosine pdf => every pixel equals albedo * L."""
    cfg = gen.make_config("C0")
    m = gen.make_model(cfg)
    m = {**m, "env": np.full((16, 32, 3), 1.75, np.float32)}
    fr = gen.make_frame(cfg, m["env"], np.arange(500))
    rng = np.random.default_rng(2)
    a = rng.random((500, 3)).astype(np.float32)
    brdf = np.concatenate([fr["n_g"], a, np.full((500, 1), 0.5, np.float32)], 1)
    # pdf consistent with the fp32 directions and normals actually passed
    fr["pdf_d"] = (np.einsum("nsk,nk->ns", fr["dir_d"].astype(np.float64), fr["n_g"].astype(np.float64)) / np.pi).astype(np.float32)
    got = gpu_render(make_renderer(cfg, m, brdf_model=0), cfg, fr, flags=1, brdf=brdf)
    np.testing.assert_allclose(got, a * 1.75, rtol=2e-5)


def test_render_frame_host_matches_device(torch):
    cfg = gen.make_config("C0", S_i=4, S_2=3, flags=7)
    m = gen.make_model(cfg)
    fr = gen.make_frame(cfg, m["env"], np.arange(1000))
    r = make_renderer(cfg, m)
    a = gpu_render(r, cfg, fr)
    b = gpu_render(r, cfg, fr, host=True)
    # same kernel, same inputs; the indirect term is summed with shared-memory float atomics, so the order (and the
    # last bit) may differ from run to run
    np.testing.assert_allclose(a, b, rtol=2e-6, atol=1e-7)
    assert r.launch_count() >= 2


@pytest.mark.parametrize("name", ["C2", "C3"])
def test_compaction_equals_dense(torch, name):
    """only rays with a non-zero Eq. 2 weight are traced further.  The compacted evaluation (default) and the
    dense one (HR_DENSE) must give the same frame (up to the summation order of the shared-memory atomics), and the
    ray accounting must add up."""
    from paper_2409_10327_b200 import HR_DENSE
    cfg = gen.make_config(name)
    m = gen.make_model(cfg)
    pix = np.arange(0, cfg.N, 487)
    fr = gen.make_frame(cfg, m["env"], pix)
    r = make_renderer(cfg, m, vis_mode=1)
    r.stats(reset=True)
    a = gpu_render(r, cfg, fr, flags=cfg.flags | HR_DENSE)
    traced_d, eval_d = r.stats(reset=True)
    b = gpu_render(r, cfg, fr, flags=cfg.flags)
    traced_c, eval_c = r.stats(reset=True)
    assert traced_d == traced_c == len(pix) * cfg.S_i
    assert eval_d == traced_d and 0 < eval_c < traced_c
    np.testing.assert_allclose(a, b, rtol=5e-6, atol=1e-7)
    # soft visibility: (1 - v) never vanishes, only back-facing / zero-pdf rays drop out
    r0 = make_renderer(cfg, m, vis_mode=0)
    a0 = gpu_render(r0, cfg, fr, flags=cfg.flags | HR_DENSE)
    b0 = gpu_render(r0, cfg, fr, flags=cfg.flags)
    np.testing.assert_allclose(a0, b0, rtol=5e-6, atol=1e-7)


def test_render_frame_host_chunked_pipeline(torch):
    """render_frame_host cuts a large frame into row chunks whose H2D copies overlap the previous chunk's render; the result
    must equal the one-launch device path (per-point direct / secondary sets, shared tertiary set, mask)."""
    cfg = gen.make_config("C2", S_d=3, S_i=2, S_2=2)
    m = gen.make_model(cfg)
    fr = gen.make_frame(cfg, m["env"])
    mask = (np.arange(cfg.N) % 7 != 0).astype(np.uint8)
    r = make_renderer(cfg, m)
    a = gpu_render(r, cfg, fr, mask=mask)
    b = gpu_render(r, cfg, fr, mask=mask, host=True)
    assert r.launch_count() >= 1 + 4                                  # 640 000 pixels -> 4 chunks on a 148-SM part
    np.testing.assert_allclose(a, b, rtol=2e-6, atol=1e-7)
    b2 = gpu_render(r, cfg, fr, mask=mask, host=True)                 # staging buffers are reused safely
    np.testing.assert_allclose(a, b2, rtol=2e-6, atol=1e-7)


def test_render_frame_host_chunks_per_point_tertiary_and_padded_rows(torch):
    """The multi-chunk host path with everything that moves per chunk: per-point direct / secondary sets whose rows are PADDED
    (point_stride > 3 S, so the last row is shorter than the stride), per-SECONDARY-point tertiary sets (row i S_i + j), a mask."""
    from paper_2409_10327_b200 import DirSet
    cfg = gen.make_config("C2", N=400_000, S_d=3, S_i=2, S_2=2)
    m = gen.make_model(cfg)
    fr = gen.make_frame(cfg, m["env"])
    N = cfg.N
    rng = np.random.default_rng(12)

    def padded(d, p, pad):                                 # [N,S,3] -> rows of S + pad directions; the last point's row is cut short
        S = d.shape[1]
        dd = np.full((N, S + pad, 3), np.nan, np.float32); dd[:, :S] = d
        pp = np.full((N, S + pad), np.nan, np.float32); pp[:, :S] = p
        return dd.reshape(-1)[: (N - 1) * 3 * (S + pad) + 3 * S].copy(), pp.reshape(-1)[: (N - 1) * (S + pad) + S].copy(), S, 3 * (S + pad)

    dd, pd_, Sd, std = padded(fr["dir_d"], fr["pdf_d"], 2)
    sd, ps_, Ss, sts = padded(fr["dir_s"], fr["pdf_s"], 1)
    dt = gen._normalize(rng.standard_normal((N * cfg.S_i, cfg.S_2, 3)))
    dt = gen._normalize(dt.astype(np.float32).astype(np.float64)).astype(np.float32)
    pt = np.full((N * cfg.S_i, cfg.S_2), 1 / (4 * np.pi), np.float32)
    mask = (np.arange(N) % 5 != 0).astype(np.uint8)
    r = make_renderer(cfg, m)
    outs = []
    for host in (False, True):
        up = (lambda a: np.ascontiguousarray(a)) if host else to_dev
        sets = [DirSet(up(dd), up(pd_), S=Sd, point_stride=std), DirSet(up(sd), up(ps_), S=Ss, point_stride=sts), DirSet(up(dt), up(pt))]
        frame = r.make_frame(up(fr["x"]), up(fr["wo"]), *sets, flags=7, mask=up(mask))
        if host:
            rgb = np.empty((N, 3), np.float32)
            l0 = r.launch_count()
            r.render_frame_host(frame, rgb)
            assert r.launch_count() - l0 >= 2, "the frame must have been cut into several chunks"
        else:
            t = torch.empty((N, 3), device="cuda")
            r.render_frame(frame, t)
            rgb = t.cpu().numpy()
        assert np.all(np.isfinite(rgb))
        outs.append(rgb)
    np.testing.assert_allclose(outs[0], outs[1], rtol=2e-6, atol=1e-7)
    assert np.all(outs[0][mask == 0] == 0) and np.abs(outs[0]).mean() > 0.05
    # and against the oracle on a pixel sample (tight rows of the same values)
    pix = np.sort(rng.choice(N, 150, replace=False))
    sub = dict(x=fr["x"][pix], wo=fr["wo"][pix], dir_d=fr["dir_d"][pix], pdf_d=fr["pdf_d"][pix], dir_s=fr["dir_s"][pix], pdf_s=fr["pdf_s"][pix],
               dir_t=dt.reshape(N, cfg.S_i, cfg.S_2, 3)[pix].reshape(-1, cfg.S_2, 3), pdf_t=pt.reshape(N, cfg.S_i, cfg.S_2)[pix].reshape(-1, cfg.S_2))
    ref = oracle_render(_oracle(cfg, m), cfg, sub, flags=7, mask=mask[pix])
    check_close(outs[1][pix], ref["rgb"], TOL32, what="host path, per-point tertiary, padded rows")


def test_fp32_model_outside_the_fp16_range_uses_the_ffma_kernels(torch):
    """The tcgen05 fp32 path carries operands as fp16 hi + lo; a model whose weights / activation bounds do not fit that range must
    fall back to the plain fp32 kernels (hashrender_last_path says which) and still match the oracle."""
    cfg = gen.make_config("C0", S_i=4, S_2=3, flags=7)
    m = gen.make_model(cfg)
    big = {**m, "brdf_w": m["brdf_w"].copy()}
    big["brdf_w"][: 64 * cfg.D] *= 4000.0                      # layer-1 weights of B: hidden activations up to ~1e5
    fr = gen.make_frame(cfg, m["env"], np.arange(300))
    r = make_renderer(cfg, big)
    got = gpu_render(r, cfg, fr)
    assert r.last_path() == "ffma32"
    ref = oracle_render(_oracle(cfg, big), cfg, fr)
    check_close(got, ref["rgb"], 4e-4, what="ffma fallback")
    r2 = make_renderer(cfg, m)
    gpu_render(r2, cfg, fr)
    assert r2.last_path() == "tcgen05-f16x3"


def test_frame_errors(torch):
    from paper_2409_10327_b200 import DirSet, HashRenderError
    cfg = gen.make_config("C0")
    m = gen.make_model(cfg)
    fr = gen.make_frame(cfg, m["env"], np.arange(64))
    from paper_2409_10327_b200 import HashRenderer
    r = HashRenderer.from_gen(cfg, m)                       # no env set
    x, wo = to_dev(fr["x"]), to_dev(fr["wo"])
    d = DirSet(to_dev(fr["dir_d"]), to_dev(fr["pdf_d"]))
    rgb = torch.empty((64, 3), device="cuda")
    with pytest.raises(HashRenderError) as e:
        r.render_frame(r.make_frame(x, wo, d), rgb)
    assert e.value.code == 1 and "env" in str(e.value)
    r.set_env(to_dev(m["env"]))
    with pytest.raises(HashRenderError):
        r.render_frame(r.make_frame(x, wo, d, flags=0), rgb)
    with pytest.raises(HashRenderError):
        r.render_frame(r.make_frame(x, wo, d, flags=7), rgb)            # INDIRECT without secondary set
    r.render_frame(r.make_frame(x, wo, d, N=0), rgb)                    # N == 0 no-op
    r.render_frame(r.make_frame(x, wo, d), rgb)
    torch.cuda.synchronize()


# ---------------------------------------------------------------------------------------------- full size, bench configuration
@pytest.mark.parametrize("name", ["C1", "C2", "C3"])
def test_full_size_sampled_pixels(torch, name):
    """BASELINE full size (800x800, 128 + 64x8 directions) in the launch configurations bench.py times -- both visibility
    modes, the default flags (compacted) and HR_DENSE (bench's headline); the oracle checks a seeded sample of pixels one by
    one (it needs ~6 ms per pixel).  The reference must be a real image in both modes."""
    from paper_2409_10327_b200 import HR_DENSE
    cfg = gen.make_config(name)
    m = gen.make_model(cfg)
    fr = gen.make_frame(cfg, m["env"])
    rng = np.random.default_rng(77)
    pix = np.sort(np.concatenate([rng.choice(cfg.N, 188, replace=False), [0, 799, 639200, 639999]]))
    sub = {k: (v[pix] if k not in ("dir_t", "pdf_t") else v) for k, v in fr.items()}
    f16 = cfg.mlp_dtype == "f16"
    indirect = bool(cfg.flags & gen.HR_INDIRECT)
    for vis_mode in (1, 0):
        r = make_renderer(cfg, m, vis_mode=vis_mode)
        o = _oracle(cfg, m, vis_mode=vis_mode)
        ref = oracle_render(o, cfg, sub, delta=(DELTA16 if f16 else DELTA32) if vis_mode else 0.0)
        for flags in ([cfg.flags, cfg.flags | HR_DENSE] if indirect else [cfg.flags]):
            got = gpu_render(r, cfg, fr, flags=flags)
            assert np.all(np.isfinite(got)) and got.shape == (cfg.N, 3)
            assert r.last_path() == ("tcgen05-f16" if f16 else "tcgen05-f16x3")
            # tolerance scale s (mean |o|) from the sample itself
            worst = check_close(got[pix], ref["rgb"], TOL16 if f16 else TOL32, extra=ref["flipbound"] if vis_mode else None,
                                what=f"{name} full-size sample vis_mode={vis_mode} flags={flags}")
            assert abs(float(got.mean()) / float(got[pix].mean()) - 1) < 0.25      # the whole frame looks like its sample
        _nontrivial(f"{name} full size", cfg, m, sub, ref, vis_mode, worst=worst)
        r.destroy()
    # a generator subset reproduces the same inputs as the full frame (so bench's CPU sample is the same workload)
    fr_sub = gen.make_frame(cfg, m["env"], pix)
    assert np.array_equal(fr_sub["dir_d"], sub["dir_d"]) and np.array_equal(fr_sub["x"], sub["x"])


@pytest.mark.parametrize("name", ["C1", "C3a"])
def test_direct_visibility_bits_of_the_render_kernel(torch, name):
    """Hard visibility as the RENDER kernel decides it, read back bit by bit.  Direct term only, external Lambert BRDF with
    albedo 1 and normal n_g, pdf = (n.w)/pi (so f_r (n.w)/p = 1) and caller-supplied radiance Lin_k = 2^k: the pixel value
    times S is the integer sum_k v_k 2^k, exactly.  Every bit must equal the oracle's [z_v > 0] wherever |z_v| >= delta, and the
    largest |z_v| at which a bit differs is printed: it is the z_v error of the kernel's own direct-query arithmetic (fp16:
    the fp16x2 final-layer epilogue `epi_fast`; fp32 models: split precision), which hashrender_trace does not go through."""
    from paper_2409_10327_b200 import DirSet
    cfg = gen.make_config(name)
    m = gen.make_model(cfg)
    n, S = 6000, 16
    pix = np.sort(np.random.default_rng(31).choice(cfg.N, n, replace=False))
    x, n_g, wo = gen.make_points(cfg, pix)
    d, _ = gen.make_cosine_hemisphere_dirs(cfg, n_g, pix, S, gen._ST_DIR_S)
    cos = np.einsum("nsk,nk->ns", d.astype(np.float64), n_g.astype(np.float64))
    keep = (cos > 1e-3).all(axis=1)                                        # every sample strictly above the horizon
    x, n_g, wo, d, cos = x[keep], n_g[keep], wo[keep], d[keep], cos[keep]
    n = len(x)
    pdf = (cos / np.pi).astype(np.float32)
    Lin = np.zeros((n, S, 3), np.float32); Lin[:, :, 0] = 2.0 ** np.arange(S); Lin[:, :, 1] = 1.0
    brdf = np.concatenate([n_g, np.ones((n, 3), np.float32), np.full((n, 1), 0.5, np.float32)], 1)
    o = _oracle(cfg, m, vis_mode=1)
    feat, _, _ = o.encode(x)
    _, zv_o, _, _ = o.trace(x, feat, d)
    r = make_renderer(cfg, m, vis_mode=1, brdf_model=0)
    rgb = torch.empty((n, 3), device="cuda")
    r.render_frame(r.make_frame(to_dev(x), to_dev(wo), DirSet(to_dev(d), to_dev(pdf), to_dev(Lin)), flags=3, brdf=to_dev(brdf)), rgb)
    got = rgb.cpu().numpy().astype(np.float64)
    code = got[:, 0] * S
    assert np.abs(code - np.round(code)).max() < 0.2, "pixel value is not an integer code"
    bits = (np.round(code).astype(np.int64)[:, None] >> np.arange(S)[None, :]) & 1
    np.testing.assert_allclose(got[:, 1] * S, bits.sum(axis=1), atol=1e-3)      # green counts the visible samples
    ref_bits = (zv_o > 0).astype(np.int64)
    diff = bits != ref_bits
    f16 = cfg.mlp_dtype == "f16"
    delta = DELTA16 if f16 else DELTA32
    worst = float(np.abs(zv_o[diff]).max()) if diff.any() else 0.0
    print(f"[render-kernel visibility bits {name}] path={r.last_path()} queries={bits.size} visible={ref_bits.mean():.3f} "
          f"flipped={int(diff.sum())} ({diff.mean():.2e}) largest |z_v| at a flip={worst:.3e} (delta={delta:g})")
    assert r.last_path() == ("tcgen05-f16" if f16 else "tcgen05-f16x3")
    assert 0.2 <= ref_bits.mean() <= 0.8
    assert worst < delta, "a visibility bit differs outside the flip band"
    assert diff.mean() < (0.03 if f16 else 5e-4), "flip fraction"


@pytest.mark.parametrize("log2_T", [16, 19, 22, 24])
def test_c4_sweep_full_size_sampled_points(torch, log2_T):
    """BASELINE.json configs[4]: encode + IRT over 2^20 uniform random points x 1 direction (fp16, L=16, F=2) at every table
    size of the sweep, through the call bench.py --workload C4 times (hashrender_trace with the encode fused, full N in one
    launch).  The oracle checks a seeded sample of points one by one: indices / fractional positions bit-exact at this T
    (the dense / hashed split of the levels moves with T), v / t / x' within the fp16 tolerance, hard
    visibility equal wherever |z_v| >= delta."""
    from paper_2409_10327_b200 import DirSet
    cfg = gen.make_config("C4", log2_T=log2_T)
    assert cfg.N == 1 << 20 and cfg.S_d == 1
    m = gen.make_model(cfg)
    fr = gen.make_frame(cfg, m["env"])
    N = cfg.N
    rng = np.random.default_rng(44)
    pix = np.sort(np.concatenate([rng.choice(N, 3000, replace=False), np.arange(N - 77, N), [0, 127, 128]]))
    xs_in, ds_in = fr["x"][pix], fr["dir_d"][pix]
    o = _oracle(cfg, m)
    feat_o, idx_o, w_o = o.encode(xs_in)
    vis_o, zv_o, t_o, x2_o = o.trace(xs_in, feat_o, ds_in)
    n_dense = int(sum((int(n) + 1) ** 3 <= cfg.T for n in m["res"]))
    assert n_dense == {16: 3, 19: 5, 22: 8, 24: 9}[log2_T]              # SURVEY Q3's list
    assert idx_o.max() < cfg.T and (log2_T < 22 or idx_o.max() >= (1 << (log2_T - 1)))
    r = make_renderer(cfg, m, max_points=N)
    xd = to_dev(fr["x"]); ds = DirSet(to_dev(fr["dir_d"]), to_dev(fr["pdf_d"]))
    vis = torch.empty((N, 1), device="cuda"); zv = torch.empty((N, 1), device="cuda"); t = torch.empty((N, 1), device="cuda")
    x2 = torch.empty((N, 1, 3), device="cuda")
    r.trace(xd, None, ds, vis, zv, t, x2, N=N)
    torch.cuda.synchronize()
    assert r.last_path() == "tcgen05-f16", r.last_path()                # k_trace_wg, the kernel the sweep times
    pd = to_dev(pix)
    got = [a[pd].cpu().numpy() for a in (vis, zv, t, x2)]
    assert all(np.all(np.isfinite(g)) for g in got)
    assert bool(torch.isfinite(t).all()) and float(t.min()) >= 0.05 and float(t.max()) <= 1.5
    check_close(got[0], vis_o, TOL16, what=f"C4 T=2^{log2_T} vis")
    check_close(got[1], zv_o, TOL16, extra=TOL16 * 0.05, what=f"C4 T=2^{log2_T} zv")
    check_close(got[2], t_o, TOL16, what=f"C4 T=2^{log2_T} t")
    check_close(got[3], x2_o, TOL16, what=f"C4 T=2^{log2_T} x'")
    # the index path at this table size, bit-exact
    n = len(pix)
    feat = torch.empty((n, cfg.D), device="cuda"); idx = torch.empty((n, cfg.L, 8), device="cuda", dtype=torch.int32)
    w = torch.empty((n, cfg.L, 3), device="cuda")
    r.encode(to_dev(xs_in), feat, idx, w)
    torch.cuda.synchronize()
    assert np.array_equal(idx.cpu().numpy().view(np.uint32), idx_o)
    assert np.array_equal(w.cpu().numpy(), w_o)
    check_close(feat.cpu().numpy(), feat_o, 2e-6, what=f"C4 T=2^{log2_T} encode")
    # hard visibility, same launch shape without the optional outputs (what bench.py passes)
    r.destroy()
    rh = make_renderer(cfg, m, vis_mode=1, max_points=N)
    rh.trace(xd, None, ds, vis, None, t, N=N)
    torch.cuda.synchronize()
    vh = vis[pd].cpu().numpy()
    assert set(np.unique(vh)) <= {0.0, 1.0}
    sure = np.abs(zv_o) >= DELTA16
    assert np.array_equal(vh[sure], (zv_o[sure] > 0).astype(np.float32)) and sure.mean() > 0.9
    check_close(t[pd].cpu().numpy(), t_o, TOL16, what=f"C4 T=2^{log2_T} t (hard)")
    rh.destroy()


def test_full_frame_is_reproducible_run_to_run(torch):
    """The same C2 frame rendered repeatedly must agree to the last bits (only the shared-memory atomics of the indirect sum
    reorder).  Regression test for a shared-memory race between warps of a warpgroup (the fp32 model's primary-BRDF scratch
    aliased the float4 copy of P): about one frame in ten had 32 pixels of one warp off by up to 0.5."""
    from paper_2409_10327_b200 import DirSet
    cfg = gen.make_config("C2")
    m = gen.make_model(cfg)
    fr = gen.make_frame(cfg, m["env"])
    x, wo = to_dev(fr["x"]), to_dev(fr["wo"])
    d, s, t = (DirSet(to_dev(fr["dir_" + k]), to_dev(fr["pdf_" + k])) for k in "dst")
    for vis_mode in (1, 0):
        r = make_renderer(cfg, m, vis_mode=vis_mode)
        for flags in (cfg.flags, cfg.flags | gen.HR_DENSE):
            frame = r.make_frame(x, wo, d, s, t, flags=flags)
            ref = torch.empty((cfg.N, 3), device="cuda")
            r.render_frame(frame, ref)
            scale = ref.abs().mean()
            for _ in range(10):
                rgb = torch.full((cfg.N, 3), float("nan"), device="cuda")
                r.render_frame(frame, rgb)
                rel = ((rgb - ref).abs() / torch.maximum(ref.abs(), scale)).max().item()
                assert rel <= 5e-6, f"vis_mode={vis_mode} flags={flags}: run-to-run difference {rel:.3e}"
        r.destroy()

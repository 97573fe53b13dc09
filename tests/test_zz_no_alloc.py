"""hashrender_denoise_static -- the denoiser with its image planes in the library's file-scope device array, for callers that cannot
call cudaMalloc -- against hashrender_denoise (the handle-owned scratch) on the same inputs: two calls in a row, of different
sizes and contents, so stale scratch of the first call would show in the second.  Collected last on purpose (pytest -x)."""
import numpy as np
import pytest

import gen
from hr_testutil import check_close, make_renderer, to_dev

pytestmark = pytest.mark.gpu

TOL = 5e-4          # the SVGF parity tolerance of tests/test_gpu_svgf.py; the two paths run the same kernels, so 0 is expected


def _window(h, w, y0, x0, seed):
    cfg = gen.make_config("C1")
    m = gen.make_model(cfg)
    ys, xs = np.mgrid[y0:y0 + h, x0:x0 + w]
    fr = gen.make_frame(cfg, m["env"], (ys * 800 + xs).ravel())
    rng = np.random.default_rng(seed)
    alb = (0.15 + 0.8 * rng.random((h, w, 3))).astype(np.float32)
    illum = 0.6 + 0.4 * np.sin(np.linspace(0, 6, w))[None, :, None] + 0.25 * rng.standard_normal((h, w, 3))
    rgb = (alb * np.maximum(illum, 0.0)).astype(np.float32)
    mask = (rng.random((h, w)) > 0.1).astype(np.uint8)
    nrm = np.ascontiguousarray(fr["n_g"].reshape(h, w, 3), np.float32)
    pos = np.ascontiguousarray(fr["x"].reshape(h, w, 3), np.float32)
    return cfg, m, [to_dev(a) for a in (rgb, nrm, pos, alb, mask)], rgb


def test_denoise_static_matches_denoise_twice_and_allocates_nothing():
    import torch
    assert torch.cuda.is_available()
    from paper_2409_10327_b200 import HashRenderError
    from paper_2409_10327_b200.binding import DENOISE_STATIC_MAX_PIXELS
    cam = (0.5, 0.5, -1.2)
    cases = [dict(h=200, w=311, y0=300, x0=250, seed=1, kw=dict(iterations=5, sigma_z=1.0, sigma_n=128.0, sigma_l=4.0), masked=True),
             dict(h=97, w=120, y0=100, x0=500, seed=2, kw=dict(iterations=2, sigma_z=2.0, sigma_n=32.0, sigma_l=1.5), masked=False)]
    r = None
    for k, c in enumerate(cases):
        cfg, m, (rgb, nrm, pos, alb, mask), rgb_host = _window(c["h"], c["w"], c["y0"], c["x0"], c["seed"])
        if r is None:
            r = make_renderer(cfg, m)
        extra = dict(albedo=alb, mask=mask if c["masked"] else None, **c["kw"])
        ref = torch.empty((c["h"], c["w"], 3), device="cuda")
        r.denoise(rgb, nrm, pos, cam, ref, **extra)                   # existing path (grows the handle's scratch)
        got = torch.full((c["h"], c["w"], 3), float("nan"), device="cuda")
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        n0 = r.launch_count()
        r.denoise_static(rgb, nrm, pos, cam, got, **extra)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0, "denoise_static changed the device's free memory"
        assert r.launch_count() - n0 == 2 + c["kw"]["iterations"]
        g, o = got.cpu().numpy(), ref.cpu().numpy()
        worst = check_close(g, o, TOL, what=f"denoise_static call {k}")
        assert np.abs(o - rgb_host).max() > 0.05                      # the filter did something
        print(f"denoise_static call {k}: {c['h']}x{c['w']}, worst err/allowed {worst:.3g}, max |diff| {np.abs(g - o).max():.3g}")
    # beyond the limit: refused before any launch, with the limit in the message
    hh, ww = 801, 800
    assert hh * ww > DENOISE_STATIC_MAX_PIXELS
    big = torch.zeros((hh, ww, 3), device="cuda")
    n0 = r.launch_count()
    with pytest.raises(HashRenderError, match=str(DENOISE_STATIC_MAX_PIXELS)):
        r.denoise_static(big, big, big, cam, big)
    assert r.launch_count() == n0
    # exactly the limit is accepted (a constant image is a fixed point of the filter)
    cfg = gen.make_config("C1")
    fr = gen.make_frame(cfg, gen.make_model(cfg)["env"])
    const = torch.full((800, 800, 3), 0.75, device="cuda")
    out = torch.empty((800, 800, 3), device="cuda")
    r.denoise_static(const, to_dev(fr["n_g"].reshape(800, 800, 3)), to_dev(fr["x"].reshape(800, 800, 3)), cam, out)
    torch.cuda.synchronize()
    assert torch.allclose(out, const, rtol=2e-6)
    r.destroy()

"""GPU parity of hashrender_denoise (spatial-only SVGF) against the numpy oracle on a window of the seeded
800x800 G-buffer (real depth / normal discontinuities between the scene's spheres, boxes and walls)."""
import numpy as np
import pytest

import gen
from hr_testutil import check_close, make_renderer, to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available()
    return torch


def _window(h, w, y0=300, x0=250, seed=0):
    cfg = gen.make_config("C1")
    m = gen.make_model(cfg)
    ys, xs = np.mgrid[y0:y0 + h, x0:x0 + w]
    pix = (ys * 800 + xs).ravel()
    fr = gen.make_frame(cfg, m["env"], pix)
    rng = np.random.default_rng(seed)
    pos = fr["x"].reshape(h, w, 3); nrm = fr["n_g"].reshape(h, w, 3)
    alb = (0.15 + 0.8 * rng.random((h, w, 3))).astype(np.float32)
    illum = 0.6 + 0.4 * np.sin(np.linspace(0, 6, w))[None, :, None] + 0.25 * rng.standard_normal((h, w, 3))
    rgb = (alb * np.maximum(illum, 0.0)).astype(np.float32)
    return cfg, m, rgb, alb, np.ascontiguousarray(nrm, np.float32), np.ascontiguousarray(pos, np.float32)


@pytest.mark.parametrize("variant", ["default", "no_albedo_masked", "two_passes"])
def test_denoise_matches_oracle(torch, variant):
    from oracle import svgf
    h, w = 96, 120
    cfg, m, rgb, alb, nrm, pos = _window(h, w)
    cam = (0.5, 0.5, -1.2)
    kw = dict(iterations=5, sigma_z=1.0, sigma_n=128.0, sigma_l=4.0)
    mask = None
    if variant == "no_albedo_masked":
        alb = None
        mask = (np.random.default_rng(3).random((h, w)) > 0.1).astype(np.uint8)
    if variant == "two_passes":
        kw.update(iterations=2, sigma_z=2.0, sigma_n=32.0, sigma_l=1.5)
    ref = svgf.denoise(rgb, nrm, pos, np.array(cam), albedo=alb, mask=mask, **kw)
    r = make_renderer(cfg, m)
    out = torch.empty((h, w, 3), device="cuda")
    r.denoise(to_dev(rgb), to_dev(nrm), to_dev(pos), cam, out, albedo=None if alb is None else to_dev(alb),
              mask=None if mask is None else to_dev(mask), **kw)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    check_close(got, ref, 5e-4, what=f"svgf {variant}")
    assert np.abs(ref - rgb).max() > 0.05                              # the filter did something
    if mask is not None:
        assert np.all(got[mask == 0] == 0)


def test_denoise_errors_and_full_frame(torch):
    from paper_2409_10327_b200 import HashRenderError
    cfg, m, rgb, alb, nrm, pos = _window(8, 8)
    r = make_renderer(cfg, m)
    out = torch.empty((8, 8, 3), device="cuda")
    with pytest.raises(HashRenderError):
        r.denoise(to_dev(rgb), to_dev(nrm), to_dev(pos), (0, 0, 0), out, iterations=0)
    with pytest.raises(HashRenderError):
        r.denoise(to_dev(rgb), None, to_dev(pos), (0, 0, 0), out)
    # constant image on the full 800x800 G-buffer: a fixed point of the filter at any size
    cfg = gen.make_config("C1")
    fr = gen.make_frame(cfg, m["env"])
    const = torch.full((800, 800, 3), 0.75, device="cuda")
    out = torch.empty((800, 800, 3), device="cuda")
    r.denoise(const, to_dev(fr["n_g"].reshape(800, 800, 3)), to_dev(fr["x"].reshape(800, 800, 3)), (0.5, 0.5, -1.2), out)
    torch.cuda.synchronize()
    assert torch.allclose(out, const, rtol=2e-6)

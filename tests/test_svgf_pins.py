"""Pins of the SVGF oracle (oracle/svgf.py) against what the filter's definition fixes -- no GPU.
PAPER.md:122 (spatial-only SVGF on the raw MC result), PAPER.md:346 (finite-difference depth gradient)."""
import numpy as np
import pytest
from scipy import ndimage

from oracle import svgf

H, W = 40, 56
CAM = np.array([0.5, 0.5, -2.0])


def _flat_scene(h=H, w=W, tilt=0.0):
    """A plane facing the camera (optionally tilted in x): positions, normals."""
    ys, xs = np.meshgrid(np.linspace(0, 1, h), np.linspace(0, 1, w), indexing="ij")
    pos = np.stack([xs, ys, tilt * xs], -1)
    nrm = np.zeros((h, w, 3)); nrm[..., 2] = -1.0
    return pos, nrm


def test_constant_image_is_a_fixed_point():
    pos, nrm = _flat_scene(tilt=0.3)
    rgb = np.tile(np.array([0.3, 1.7, 0.05]), (H, W, 1))
    out = svgf.denoise(rgb, nrm, pos, CAM)
    np.testing.assert_allclose(out, rgb, rtol=1e-12)


def test_without_edge_stopping_it_is_the_b3_atrous_convolution():
    """sigma_z, sigma_l -> inf and sigma_n = 0 switch every edge-stopping weight to 1: one iteration with hole size s must equal the
    dilated 5x5 B3-spline convolution (scipy.ndimage, zero padding) renormalised by the convolution of ones."""
    rng = np.random.default_rng(0)
    pos, nrm = _flat_scene()
    col = rng.random((H, W, 3)); var = rng.random((H, W))
    z = np.full((H, W), 3.0); gx = np.zeros((H, W)); gy = np.zeros((H, W))     # constant depth: w_z = 1
    live = np.ones((H, W), bool)
    for step in (1, 2, 4):
        out, vout = svgf.atrous_iteration(col, var, z, gx, gy, nrm, live, step, 1e30, 0.0, 1e30)
        k1 = np.zeros(4 * step + 1); k1[::step] = svgf.B3
        k2 = np.outer(k1, k1)
        ones = ndimage.convolve(np.ones((H, W)), k2, mode="constant")
        for ch in range(3):
            ref = ndimage.convolve(col[..., ch], k2, mode="constant") / ones
            np.testing.assert_allclose(out[..., ch], ref, rtol=1e-10)
        np.testing.assert_allclose(vout, ndimage.convolve(var, k2 * k2, mode="constant") / ones ** 2, rtol=1e-10)


def test_depth_weight_closed_form_on_a_ramp_and_gradient_definition():
    """Linear depth: |z_p - z_q| = |grad z . (p - q)|, so w_z = exp(-1/sigma_z) for every off-centre tap (SVGF eq. 3)."""
    h, w = 12, 16
    pos = np.zeros((h, w, 3)); pos[..., 2] = 0.25 * np.arange(w)[None, :] + 0.5 * np.arange(h)[:, None]
    cam = np.array([0.0, 0.0, -1e9])                   # far camera: z = pos_z + 1e9 up to rounding, linear in the pixel index
    pos64 = pos.copy(); z, gx, gy = svgf.depth_and_gradient(pos64, cam)
    np.testing.assert_allclose(gx, 0.25, atol=1e-5); np.testing.assert_allclose(gy, 0.5, atol=1e-5)
    nrm = np.zeros((h, w, 3)); nrm[..., 2] = -1
    live = np.ones((h, w), bool)
    wgt = svgf._geometry_weight(z, gx, gy, nrm, live, 1, 2, 2.0, 128.0)
    np.testing.assert_allclose(wgt[:-1, :-2], np.exp(-0.5), rtol=1e-4)
    assert np.all(wgt[-1, :] == 0) and np.all(wgt[:, -2:] == 0)       # taps outside the image are skipped
    np.testing.assert_allclose(svgf._geometry_weight(z, gx, gy, nrm, live, 0, 0, 2.0, 128.0), 1.0)
    # backward difference on the last column / row
    z2 = np.arange(5.0)[None, :] ** 2 + np.zeros((3, 1))
    _, gx2, gy2 = svgf.depth_and_gradient(np.dstack([np.zeros((3, 5)), np.zeros((3, 5)), z2]), np.array([0, 0, 0.0]))
    np.testing.assert_allclose(gx2[0], [1, 3, 5, 7, 7]); np.testing.assert_allclose(gy2, 0)


def test_edges_in_depth_and_normal_do_not_bleed():
    pos, nrm = _flat_scene()
    rgb = np.zeros((H, W, 3)); rgb[:, : W // 2] = [1.0, 0.2, 0.1]; rgb[:, W // 2:] = [0.1, 0.3, 2.0]
    pos_d = pos.copy(); pos_d[:, W // 2:, 2] += 5.0                   # depth discontinuity between columns W/2-1 and W/2
    z, gx, gy = svgf.depth_and_gradient(pos_d, CAM)
    live = np.ones((H, W), bool)
    for d in (1, 2, 4, 8):                                            # a tap that crosses the jump has (numerically) zero weight ...
        wgt = svgf._geometry_weight(z, gx, gy, nrm, live, 0, d, 1.0, 128.0)
        cross = wgt[:, W // 2 - d: W // 2 - 1]                        # ... except from the column whose forward difference spans it
        assert cross.size == 0 or cross.max() < 1e-30
        assert wgt[:, : W // 2 - d].min() > 1e-3 and wgt[:, W // 2: W - d].min() > 1e-3   # same-side taps: 27 orders of magnitude above the crossing ones
    assert svgf._geometry_weight(z, gx, gy, nrm, live, 0, 1, 1.0, 128.0)[:, W // 2 - 1].min() > 0.3   # PAPER.md:346's gradient sees the jump
    nrm_n = nrm.copy(); nrm_n[:, W // 2:] = [1.0, 0.0, 0.0]           # orthogonal normals, same depth
    out = svgf.denoise(rgb, nrm_n, pos, CAM, sigma_l=1e30, sigma_z=1e30)
    np.testing.assert_allclose(out, rgb, atol=1e-12)
    out = svgf.denoise(rgb, nrm, pos, CAM, sigma_l=1e30, sigma_z=1e30)   # control: without an edge the colours do mix
    assert np.abs(out - rgb).max() > 0.3


def test_noise_is_reduced_and_the_mean_kept():
    rng = np.random.default_rng(1)
    pos, nrm = _flat_scene(64, 64)
    mu = np.array([0.8, 0.5, 0.3]); s = 0.2
    rgb = mu + s * rng.standard_normal((64, 64, 3))
    var = svgf.estimate_variance(rgb @ svgf.LUMA, *svgf.depth_and_gradient(pos, CAM), nrm, np.ones((64, 64), bool), 1.0, 128.0)
    s_l = s * np.sqrt((svgf.LUMA ** 2).sum())
    assert abs(var[8:-8, 8:-8].mean() / s_l ** 2 - 48 / 49) < 0.1       # 7x7 sample variance of iid noise
    out = svgf.denoise(rgb, nrm, pos, CAM)
    inner = out[16:-16, 16:-16]
    assert np.abs(inner.mean((0, 1)) - mu).max() < 0.02
    assert inner.std((0, 1)).max() < s / 5


def test_albedo_demodulation_keeps_texture_and_mask_does_not_leak():
    rng = np.random.default_rng(2)
    pos, nrm = _flat_scene()
    ys, xs = np.mgrid[0:H, 0:W]
    alb = np.where(((ys // 4 + xs // 4) % 2)[..., None] == 0, [0.9, 0.8, 0.7], [0.1, 0.2, 0.05])
    rgb = alb * np.array([1.5, 1.5, 1.5])                            # constant illumination under a checkerboard albedo
    np.testing.assert_allclose(svgf.denoise(rgb, nrm, pos, CAM, albedo=alb), rgb, rtol=1e-9)
    assert np.abs(svgf.denoise(rgb, nrm, pos, CAM) - rgb).max() > 0.05   # without demodulation the texture blurs
    mask = np.ones((H, W), np.uint8); mask[10:20, 10:30] = 0
    noisy = 0.5 + 0.1 * rng.standard_normal((H, W, 3))
    a = noisy.copy(); a[10:20, 10:30] = 1e6
    b = noisy.copy(); b[10:20, 10:30] = -3.0
    oa, ob = svgf.denoise(a, nrm, pos, CAM, mask=mask), svgf.denoise(b, nrm, pos, CAM, mask=mask)
    np.testing.assert_array_equal(oa, ob)
    assert np.all(oa[10:20, 10:30] == 0)

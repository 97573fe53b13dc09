"""oracle/svgf.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain numpy (float64) statement of the spatial-only SVGF denoiser that follows the hash-grid renderer:
PAPER.md:122 "SVGF [17] ... operates on the raw MC rendering results to greatly reduce pixel color variance.  Since our model is
not targeting video generation, all temporal elements of SVGF are removed"; "The clip-space depth gradient map
required to operate SVGF is approximated by offsetting the predicted depth map (derived from the direct illumination renderer's
primary surface coordinate map) vertically and horizontally and calculating the numerical difference to the original value".

The paper gives no parameter; the filter below is the published spatial part of SVGF (Schied et al. 2017) restated, with the readings
Q39-Q44 of DESIGN.md: albedo demodulation, 7x7 bilateral estimate of the luminance variance (SVGF's fallback without history), five
5x5 a-trous iterations with step 2^i, B3-spline kernel, edge-stopping weights on depth (scaled by the finite-difference gradient),
normal and luminance (scaled by the 3x3-gaussian-filtered variance), variance filtered with squared weights.
Written as per-tap shifted-array sums: one term of the paper's sums per line, no blocking or separable shortcuts.
Only tests/, __graft_entry__ and bench.py's oracle legs import this; it never imports paper_2409_10327_b200.
"""
from __future__ import annotations

import numpy as np

LUMA = np.array([0.2126, 0.7152, 0.0722])
B3 = np.array([1 / 16, 1 / 4, 3 / 8, 1 / 4, 1 / 16])          # a-trous kernel h
G3 = np.array([[1, 2, 1], [2, 4, 2], [1, 2, 1]]) / 16.0       # 3x3 gaussian prefilter of the variance


def _shift(a, dy, dx):
    """a[y + dy, x + dx] with a validity mask (taps outside the image are skipped, Q43)."""
    H, W = a.shape[:2]
    out = np.zeros_like(a)
    ok = np.zeros((H, W), bool)
    y0, y1 = max(0, -dy), min(H, H - dy)
    x0, x1 = max(0, -dx), min(W, W - dx)
    if y0 < y1 and x0 < x1:
        out[y0:y1, x0:x1] = a[y0 + dy:y1 + dy, x0 + dx:x1 + dx]
        ok[y0:y1, x0:x1] = True
    return out, ok


def depth_and_gradient(pos, cam):
    """z = |x - o| (depth from the primary surface coordinate map); forward differences, backward at the last
    row / column (Q40).  Returns z [H,W], dzdx [H,W], dzdy [H,W]."""
    z = np.linalg.norm(np.asarray(pos, np.float64) - np.asarray(cam, np.float64), axis=-1)
    dzdx = np.empty_like(z); dzdy = np.empty_like(z)
    dzdx[:, :-1] = z[:, 1:] - z[:, :-1]; dzdx[:, -1] = z[:, -1] - z[:, -2] if z.shape[1] > 1 else 0.0
    dzdy[:-1, :] = z[1:, :] - z[:-1, :]; dzdy[-1, :] = z[-1, :] - z[-2, :] if z.shape[0] > 1 else 0.0
    return z, dzdx, dzdy


def _geometry_weight(z, dzdx, dzdy, nrm, live, dy, dx, sigma_z, sigma_n):
    """w_z * w_n of tap q = p + (dy, dx) (SVGF eq. 3, 4), zero outside the image or on masked pixels."""
    zq, ok = _shift(z, dy, dx)
    nq, _ = _shift(nrm, dy, dx)
    lq, _ = _shift(live.astype(np.float64), dy, dx)
    wz = np.exp(-np.abs(z - zq) / (sigma_z * np.abs(dzdx * dx + dzdy * dy) + 1e-6))
    wn = np.maximum(0.0, np.sum(nrm * nq, axis=-1)) ** sigma_n
    return wz * wn * ok * (lq > 0) * live


def estimate_variance(lum, z, dzdx, dzdy, nrm, live, sigma_z, sigma_n):
    """Spatial estimate of the luminance variance: bilateral 7x7 first and second moments (Q41)."""
    s0 = np.zeros_like(lum); s1 = np.zeros_like(lum); s2 = np.zeros_like(lum)
    for dy in range(-3, 4):
        for dx in range(-3, 4):
            w = _geometry_weight(z, dzdx, dzdy, nrm, live, dy, dx, sigma_z, sigma_n)
            lq, _ = _shift(lum, dy, dx)
            s0 += w; s1 += w * lq; s2 += w * lq * lq
    s0 = np.maximum(s0, 1e-12)
    m1, m2 = s1 / s0, s2 / s0
    return np.maximum(0.0, m2 - m1 * m1)


def atrous_iteration(col, var, z, dzdx, dzdy, nrm, live, step, sigma_z, sigma_n, sigma_l):
    """One 5x5 a-trous pass with hole size `step` (SVGF eq. 1, 2, 5)."""
    lum = col @ LUMA
    gv = np.zeros_like(var); gw = np.zeros_like(var)
    for dy in (-1, 0, 1):
        for dx in (-1, 0, 1):
            vq, ok = _shift(var, dy, dx)
            gv += G3[dy + 1, dx + 1] * vq * ok; gw += G3[dy + 1, dx + 1] * ok
    sd = np.sqrt(np.maximum(gv / np.maximum(gw, 1e-12), 0.0))
    num = np.zeros_like(col); den = np.zeros_like(var); vnum = np.zeros_like(var)
    for iy in range(5):
        for ix in range(5):
            dy, dx = (iy - 2) * step, (ix - 2) * step
            w = _geometry_weight(z, dzdx, dzdy, nrm, live, dy, dx, sigma_z, sigma_n)
            cq, _ = _shift(col, dy, dx); vq, _ = _shift(var, dy, dx); lq, _ = _shift(lum, dy, dx)
            wl = np.exp(-np.abs(lum - lq) / (sigma_l * sd + 1e-6))
            w = B3[iy] * B3[ix] * w * wl
            num += w[..., None] * cq; den += w; vnum += w * w * vq
    den_s = np.maximum(den, 1e-12)
    out = np.where((den > 0)[..., None], num / den_s[..., None], col)
    vout = np.where(den > 0, vnum / (den_s * den_s), var)
    return out, vout


def denoise(rgb, normal, pos, cam, albedo=None, mask=None, iterations=5, sigma_z=1.0, sigma_n=128.0, sigma_l=4.0):
    """rgb [H,W,3] raw MC radiance -> filtered [H,W,3].  albedo [H,W,3] given => illumination is filtered demodulated (Q39)."""
    rgb = np.asarray(rgb, np.float64); nrm = np.asarray(normal, np.float64)
    H, W = rgb.shape[:2]
    live = np.ones((H, W), bool) if mask is None else np.asarray(mask).astype(bool)
    alb = None if albedo is None else np.maximum(np.asarray(albedo, np.float64), 1e-3)
    col = rgb if alb is None else rgb / alb
    z, dzdx, dzdy = depth_and_gradient(pos, cam)
    var = estimate_variance(col @ LUMA, z, dzdx, dzdy, nrm, live, sigma_z, sigma_n)
    for i in range(iterations):
        col, var = atrous_iteration(col, var, z, dzdx, dzdy, nrm, live, 1 << i, sigma_z, sigma_n, sigma_l)
    out = col if alb is None else col * alb
    return np.where(live[..., None], out, 0.0)

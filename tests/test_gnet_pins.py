"""Pins of the G-network oracle (oracle/gnet_oracle.py) against what the paper and PyTorch's conventions fix (CPU only).
The paper's pipeline is PyTorch, so every op is pinned to the independent torch CPU routine in float64 and
to a closed form / textbook property; the whole network is pinned to the same graph assembled from torch.nn.functional."""
import math

import numpy as np
import pytest

from gen import gnet
from oracle import gnet_oracle as G

torch = pytest.importorskip("torch")
F = torch.nn.functional
T = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64))


def test_conv3x3_is_zero_padded_cross_correlation():
    rng = np.random.default_rng(0)
    x = rng.standard_normal((3, 7, 9)); W = rng.standard_normal((4, 3, 3, 3)); b = rng.standard_normal(4)
    y = G.conv3x3(x, W, b)
    ref = F.conv2d(T(x)[None], T(W), T(b), padding=1)[0].numpy()
    np.testing.assert_allclose(y, ref, atol=1e-12)
    from scipy.signal import correlate2d                      # a second, library-independent statement
    for o in range(4):
        acc = sum(correlate2d(x[c], W[o, c], mode="same", boundary="fill", fillvalue=0.0) for c in range(3)) + b[o]
        np.testing.assert_allclose(y[o], acc, atol=1e-12)
    # a transposed / flipped kernel (true convolution) must NOT pass: the asymmetric kernel tells them apart
    assert np.abs(y - G.conv3x3(x, W[:, :, ::-1, ::-1], b)).max() > 0.1
    # one-hot kernel tap (ky, kx) = (0, 2) reads the pixel up-right
    W1 = np.zeros((1, 1, 3, 3)); W1[0, 0, 0, 2] = 1.0
    y1 = G.conv3x3(x[:1], W1, np.zeros(1))
    assert np.array_equal(y1[0, 1:, :-1], x[0, :-1, 1:]) and np.all(y1[0, 0] == 0) and np.all(y1[0, :, -1] == 0)


def test_conv1x1_is_a_channel_matmul():
    rng = np.random.default_rng(1)
    x = rng.standard_normal((5, 4, 6)); W = rng.standard_normal((3, 5)); b = rng.standard_normal(3)
    ref = F.conv2d(T(x)[None], T(W)[:, :, None, None], T(b))[0].numpy()
    np.testing.assert_allclose(G.conv1x1(x, W, b), ref, atol=1e-12)
    np.testing.assert_allclose(G.conv1x1(x, W, b)[:, 2, 3], W @ x[:, 2, 3] + b, atol=1e-12)


def test_instance_norm_closed_forms():
    rng = np.random.default_rng(2)
    x = rng.standard_normal((6, 11, 13)) * rng.uniform(0.1, 5, (6, 1, 1)) + rng.uniform(-3, 3, (6, 1, 1))
    g = rng.uniform(0.5, 1.5, 6); be = rng.uniform(-1, 1, 6)
    y = G.instance_norm(x, g, be)
    ref = F.instance_norm(T(x)[None], weight=T(g), bias=T(be), eps=1e-5)[0].numpy()
    np.testing.assert_allclose(y, ref, atol=1e-12)
    y0 = G.instance_norm(x, np.ones(6), np.zeros(6))
    np.testing.assert_allclose(y0.mean(axis=(1, 2)), 0, atol=1e-12)                      # zero mean per channel
    v = x.var(axis=(1, 2))                                                              # biased variance
    np.testing.assert_allclose(y0.var(axis=(1, 2)), v / (v + 1e-5), rtol=1e-12)          # unit variance up to eps
    np.testing.assert_allclose(G.instance_norm(np.full((2, 4, 4), 7.0), g[:2], be[:2]), np.broadcast_to(be[:2, None, None], (2, 4, 4)), atol=1e-9)
    # invariance: scaling and shifting a channel does not change its normalised map (up to eps)
    np.testing.assert_allclose(G.instance_norm(3 * x + 2, g, be), y, atol=2e-5)


def test_gelu_closed_forms():
    x = np.linspace(-6, 6, 241)
    ref = np.array([0.5 * v * (1 + math.erf(v / math.sqrt(2))) for v in x])             # x Phi(x), math.erf
    np.testing.assert_allclose(G.gelu(x), ref, atol=1e-15)
    np.testing.assert_allclose(G.gelu(x), F.gelu(T(x)).numpy(), atol=1e-15)              # exact form, not the tanh approximation
    assert G.gelu(np.zeros(1))[0] == 0 and abs(G.gelu(np.ones(1))[0] - 0.8413447460685429) < 1e-15
    np.testing.assert_allclose(G.gelu(x) - G.gelu(-x), x, atol=1e-15)                    # x Phi(x) + x Phi(-x) = x
    assert abs(G.gelu(np.array([10.0]))[0] - 10.0) < 1e-12 and abs(G.gelu(np.array([-10.0]))[0]) < 1e-12
    assert np.abs(G.gelu(x) - 0.5 * x * (1 + np.tanh(math.sqrt(2 / math.pi) * (x + 0.044715 * x ** 3)))).max() > 1e-4


def test_bilinear_upsample_half_pixel_centres():
    rng = np.random.default_rng(3)
    x = rng.standard_normal((2, 5, 7))
    y = G.upsample2(x)
    ref = F.interpolate(T(x)[None], scale_factor=2, mode="bilinear", align_corners=False)[0].numpy()
    np.testing.assert_allclose(y, ref, atol=1e-13)
    assert y.shape == (2, 10, 14)
    np.testing.assert_allclose(G.upsample2(np.full((1, 3, 3), 2.5)), 2.5)                # constants preserved
    # a linear ramp is reproduced exactly away from the clamped border: value at output pixel j is the ramp at (j + 0.5)/2 - 0.5
    ramp = np.broadcast_to(np.arange(8.0)[None, None, :], (1, 4, 8)).copy()
    u = G.upsample2(ramp)
    j = np.arange(16)
    expect = np.clip((j + 0.5) / 2 - 0.5, 0, 7)
    np.testing.assert_allclose(u[0, 3], expect, atol=1e-14)
    # weights 1/4, 3/4 in the interior
    assert abs(y[0, 2, 3] - (0.75 * 0.75 * x[0, 1, 1] + 0.75 * 0.25 * x[0, 1, 2] + 0.25 * 0.75 * x[0, 0, 1] + 0.25 * 0.25 * x[0, 0, 2])) < 1e-14


def _torch_forward(blob, rays, n_res, width, sr_ch):
    net = G.split_blob(blob, width=width, n_res=n_res, sr_ch=sr_ch, in_ch=6)
    cna = lambda x, l, pad: F.gelu(F.instance_norm(F.conv2d(x, T(l[0]), T(l[1]), padding=pad), weight=T(l[2]), bias=T(l[3]), eps=1e-5))
    x = T(rays).permute(2, 0, 1)[None]
    x = cna(x, net["stem"], 0)
    for i in range(0, n_res, 2):
        x = x + cna(cna(x, net[f"res{i}"], 0), net[f"res{i + 1}"], 0)
    out = None
    up = lambda t: F.interpolate(t, scale_factor=2, mode="bilinear", align_corners=False)
    for s in range(len(sr_ch)):
        x = cna(cna(up(x), net[f"sr{s}a"], 1), net[f"sr{s}b"], 1)
        m = F.conv2d(x, T(net[f"sr{s}map"][0]), T(net[f"sr{s}map"][1]))
        out = m if out is None else up(out) + m
    return out[0].permute(1, 2, 0).reshape(-1, 11).numpy()


@pytest.mark.parametrize("n_res,width,sr_ch,hw", [(4, 32, (16, 8), (5, 6)), (28, 256, (128, 64, 32), (3, 4))])
def test_whole_network_against_torch_functional(n_res, width, sr_ch, hw):
    """The same graph assembled from torch.nn.functional in float64 (readings Q45-Q51)."""
    kw = dict(width=width, n_res=n_res, sr_ch=sr_ch)
    blob = gnet.make_gnet(11, dtype="f32", **kw)
    rays = gnet.make_rays(11, *hw)
    r = G.forward(blob, rays, **kw)
    ref = _torch_forward(blob, rays, n_res, width, sr_ch)
    np.testing.assert_allclose(r["raw"], ref, atol=1e-9)
    N = hw[0] * hw[1] * 4 ** len(sr_ch)
    assert r["raw"].shape == (N, 11) and r["x"].shape == (N, 3) and r["brdf"].shape == (N, 7)
    np.testing.assert_allclose(np.linalg.norm(r["brdf"][:, :3], axis=1), 1, atol=1e-12)          # output maps
    assert np.all((r["brdf"][:, 3:6] > 0) & (r["brdf"][:, 3:6] < 1)) and np.all((r["brdf"][:, 6] >= 0.09) & (r["brdf"][:, 6] <= 1))
    assert np.all((r["x"] > 0) & (r["x"] < 1)) and set(np.unique(r["mask"])) <= {0, 1}
    assert np.array_equal(r["mask"], (r["raw"][:, 10] > 0))


def test_structure_special_cases():
    """Zeroed residual branches leave the stem's output unchanged; the output skip adds the upsampled maps of the previous block."""
    kw = dict(width=16, n_res=4, sr_ch=(8, 4))
    blob = gnet.make_gnet(3, dtype="f32", **kw)
    rays = gnet.make_rays(3, 4, 4)
    net = G.split_blob(blob, in_ch=6, **kw)
    # (i) brute force of one output pixel of the first SR block's first conv, written as explicit loops
    x = np.moveaxis(rays.astype(np.float64), -1, 0)
    x = G.cna1(x, net["stem"])
    for i in (0, 2):
        x = x + G.cna1(G.cna1(x, net[f"res{i}"]), net[f"res{i + 1}"])
    u = G.upsample2(x)
    W, b = net["sr0a"][0], net["sr0a"][1]
    acc = b[3]
    for c in range(16):
        for ky in range(3):
            for kx in range(3):
                yy, xx = 5 + ky - 1, 0 + kx - 1
                if 0 <= yy < 8 and 0 <= xx < 8:
                    acc += W[3, c, ky, kx] * u[c, yy, xx]
    assert abs(G.conv3x3(u, W, b)[3, 5, 0] - acc) < 1e-12
    # (ii) instance-norm gamma = beta = 0 on the second layer of every residual block => the branch is GELU(0) = 0 => identity
    off = 0
    z = blob.copy()
    for name, co, ci, k, norm in G.layer_shapes(in_ch=6, **kw):
        n = co * ci * k * k + co
        if name in ("res1", "res3"):
            z[off + n: off + n + 2 * co] = 0
        off += n + (2 * co if norm else 0)
    r0 = G.forward(z, rays, **kw)
    z2 = z.copy()
    # with identity residual blocks the result does not depend on the (now dead) first layers of the blocks
    off = 0
    for name, co, ci, k, norm in G.layer_shapes(in_ch=6, **kw):
        n = co * ci * k * k + co
        if name in ("res0", "res2"):
            z2[off: off + n] *= -3.0
        off += n + (2 * co if norm else 0)
    np.testing.assert_allclose(G.forward(z2, rays, **kw)["raw"], r0["raw"], atol=1e-12)
    # (iii) output skip: zero the last block's map layer => the output is the bilinear upsample of the first block's maps
    z3 = blob.copy()
    off = 0
    for name, co, ci, k, norm in G.layer_shapes(in_ch=6, **kw):
        n = co * ci * k * k + co
        if name == "sr1map":
            z3[off: off + n] = 0
        off += n + (2 * co if norm else 0)
    full = G.forward(z3, rays, **kw)["raw"].reshape(16, 16, 11)
    x = np.moveaxis(rays.astype(np.float64), -1, 0)
    x = G.cna1(x, net["stem"])
    for i in (0, 2):
        x = x + G.cna1(G.cna1(x, net[f"res{i}"]), net[f"res{i + 1}"])
    f0 = G.cna3(G.cna3(G.upsample2(x), net["sr0a"]), net["sr0b"])
    m0 = G.conv1x1(f0, net["sr0map"][0].reshape(11, -1), net["sr0map"][1])
    np.testing.assert_allclose(full, np.moveaxis(G.upsample2(m0), 0, -1), atol=1e-12)

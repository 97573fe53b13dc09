"""oracle/gnet_oracle.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain float64 numpy statement of the forward pass of the paper's CNN direct-illumination renderer G
(arXiv 2409.10327; PAPER.md = /root/reference/PAPER.md): the step that hands the hash-grid renderer its inputs --
"full-resolution maps of material, normal, and primary surface coordinates".  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline legs may import it; it shares nothing with paper_2409_10327_b200/.

Architecture as the paper states it, with the DESIGN.md readings (Q45-Q51) where it is silent:
  * input gamma = [o, d_down]: camera position broadcast + ray direction per pixel of the downsampled array, 6 ch;
  * "an initial 1x1 conv-norm-act layer" 6 -> 256; norm = instance normalisation with affine
    parameters, act = GELU;
  * "a deep residual MLP": 28 identical 1x1 conv-norm-act layers at 256 channels, read as 14 residual
    blocks of two layers, x <- x + L2(L1(x)) (Q47: the paper follows MobileR2L's stacked ResMLP and says no more);
  * three super-resolution blocks (PAPER.md:68b): bilinear x2 upsample, two 3x3 conv-norm-act layers, then 1x1 "output
    mapping" convolutions; channels 128, 64, 32;
  * output skip (PAPER.md:68a, 96 "output skip structure from StyleGAN2"): "Each output from an SR block is bilinearly
    upsampled and added to the output from the next SR block";
  * 11 output channels [n(3), a(3), r(1), x(3), mask(1)] with the maps of PAPER.md:114 (n/||n||,
    sigma(a), 0.09 + 0.91 sigma(r)), x = sigma(raw) so that it lies in the unit cube the hash grid takes (Q50), mask = [raw > 0].
Conventions are PyTorch's (the paper's framework): cross-correlation with zero padding 1 for 3x3, instance
norm over H x W per channel with biased variance and eps = 1e-5, exact (erf) GELU, bilinear with align_corners = False.

Pins (tests/test_gnet_pins.py): every op against the independent torch CPU routine in float64 and against closed forms
(scipy correlate2d, zero-mean / unit-variance, GELU identities, linear-ramp reproduction), and the whole network against
the same graph assembled from torch.nn.functional.  "Agreement with the authors' trained G" is PARITY UNPINNED (no weights).
"""
from __future__ import annotations

import math

import numpy as np

OUT_CH = 11          # n3 a3 r1 x3 mask1
EPS = 1e-5


# ------------------------------------------------------------------------------------------------------ ops
def conv1x1(x, W, b):
    """x [Cin,H,W], W [Cout,Cin], b [Cout] -> [Cout,H,W]   (a 1x1 convolution is a matmul over channels)."""
    C, H, Wd = x.shape
    return (W @ x.reshape(C, H * Wd) + b[:, None]).reshape(-1, H, Wd)


def conv3x3(x, W, b):
    """x [Cin,H,W], W [Cout,Cin,3,3], zero padding 1, cross-correlation (PyTorch conv2d):
    y[o,i,j] = b[o] + sum_{c,ky,kx} W[o,c,ky,kx] x[c, i+ky-1, j+kx-1]."""
    C, H, Wd = x.shape
    xp = np.zeros((C, H + 2, Wd + 2), dtype=np.float64)
    xp[:, 1:-1, 1:-1] = x
    y = np.zeros((W.shape[0], H * Wd), dtype=np.float64)
    for ky in range(3):
        for kx in range(3):
            y += W[:, :, ky, kx] @ xp[:, ky:ky + H, kx:kx + Wd].reshape(C, H * Wd)
    return (y + b[:, None]).reshape(-1, H, Wd)


def instance_norm(x, gamma, beta):
    """Per channel over H x W: (x - mean) / sqrt(var + eps) * gamma + beta, biased variance ("[19] with affine parameters")."""
    m = x.mean(axis=(1, 2), keepdims=True)
    v = ((x - m) ** 2).mean(axis=(1, 2), keepdims=True)
    return (x - m) / np.sqrt(v + EPS) * gamma[:, None, None] + beta[:, None, None]


def gelu(x):
    """GELU(x) = x Phi(x) = x/2 (1 + erf(x / sqrt 2))  ("[9]"); erf is scipy's (a library primitive)."""
    from scipy.special import erf
    return 0.5 * x * (1.0 + erf(x / math.sqrt(2.0)))


def upsample2(x):
    """Bilinear x2, align_corners = False: output pixel i samples the input at (i + 0.5)/2 - 0.5, clamped to the border."""
    C, H, Wd = x.shape

    def taps(n):
        src = (np.arange(2 * n) + 0.5) / 2.0 - 0.5
        src = np.maximum(src, 0.0)
        i0 = np.floor(src).astype(np.int64)
        i1 = np.minimum(i0 + 1, n - 1)
        return i0, i1, src - i0
    y0, y1, fy = taps(H)
    x0, x1, fx = taps(Wd)
    top = x[:, y0][:, :, x0] * (1 - fx) + x[:, y0][:, :, x1] * fx
    bot = x[:, y1][:, :, x0] * (1 - fx) + x[:, y1][:, :, x1] * fx
    return top * (1 - fy)[None, :, None] + bot * fy[None, :, None]


def cna1(x, layer):
    W, b, g, be = layer
    return gelu(instance_norm(conv1x1(x, W.reshape(W.shape[0], W.shape[1]), b), g, be))


def cna3(x, layer):
    W, b, g, be = layer
    return gelu(instance_norm(conv3x3(x, W, b), g, be))


def sigmoid(z):
    return 1.0 / (1.0 + np.exp(-z))


# ------------------------------------------------------------------------------------------------------ network
def layer_shapes(width=256, n_res=28, sr_ch=(128, 64, 32), in_ch=6):
    """[(name, Cout, Cin, k, has_norm)] in blob order."""
    out = [("stem", width, in_ch, 1, True)]
    out += [(f"res{i}", width, width, 1, True) for i in range(n_res)]
    c = width
    for s, ch in enumerate(sr_ch):
        out += [(f"sr{s}a", ch, c, 3, True), (f"sr{s}b", ch, ch, 3, True), (f"sr{s}map", OUT_CH, ch, 1, False)]
        c = ch
    return out


def split_blob(blob, **kw):
    """Flat fp32 blob -> {name: (W[Cout,Cin,k,k], b[Cout], gamma[Cout], beta[Cout])} as float64 (gamma/beta absent for map layers)."""
    blob = np.asarray(blob, dtype=np.float64)
    out, off = {}, 0
    for name, co, ci, k, norm in layer_shapes(**kw):
        n = co * ci * k * k
        W = blob[off:off + n].reshape(co, ci, k, k); off += n
        b = blob[off:off + co]; off += co
        if norm:
            g = blob[off:off + co]; off += co
            be = blob[off:off + co]; off += co
            out[name] = (W, b, g, be)
        else:
            out[name] = (W, b)
    assert off == blob.size, (off, blob.size)
    return out


def forward(blob, rays, rough_min=0.09, n_res=28, width=256, sr_ch=(128, 64, 32), return_raw=False):
    """rays [h, w, 6] (gamma = [o, d_down]) -> dict(x [N,3], brdf [N,7] = n a r, mask [N], raw [N,11]),
    N = (8h)(8w) pixels in row-major image order -- the arrays hr_frame takes."""
    net = split_blob(blob, width=width, n_res=n_res, sr_ch=sr_ch, in_ch=rays.shape[-1])
    x = np.ascontiguousarray(np.moveaxis(np.asarray(rays, dtype=np.float64), -1, 0))        # [6,h,w]
    x = cna1(x, net["stem"])
    for i in range(0, n_res, 2):                        # residual block of two conv-norm-act layers (Q47)
        x = x + cna1(cna1(x, net[f"res{i}"]), net[f"res{i + 1}"])
    out = None
    for s in range(len(sr_ch)):
        f = cna3(cna3(upsample2(x), net[f"sr{s}a"]), net[f"sr{s}b"])
        Wm, bm = net[f"sr{s}map"]
        m = conv1x1(f, Wm.reshape(OUT_CH, -1), bm)
        out = m if out is None else upsample2(out) + m   # output skip (PAPER.md:68a)
        x = f
    raw = np.moveaxis(out, 0, -1).reshape(-1, OUT_CH)    # [N,11]
    n = raw[:, 0:3]
    nn = np.maximum(np.linalg.norm(n, axis=1, keepdims=True), 1e-12)
    brdf = np.concatenate([n / nn, sigmoid(raw[:, 3:6]), rough_min + (1.0 - rough_min) * sigmoid(raw[:, 6:7])], axis=1)
    res = dict(x=sigmoid(raw[:, 7:10]), brdf=brdf, mask=(raw[:, 10] > 0.0).astype(np.uint8), raw=raw)
    return res

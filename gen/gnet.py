"""Seeded synthetic inputs of the CNN direct renderer G: random-init weights of the stated
architecture and the ray map gamma = [o, d_down] of a camera pose.  No method arithmetic lives here (only draws and the
pinhole geometry of the input rays); serves the oracle and the CUDA path alike, imports neither.

Stands in for the trained G of the paper (no weights exist here): conv weights and biases U(+-1/sqrt(fan_in)) (PyTorch's
default initialisation of the paper's framework), instance-norm gamma U(0.5, 1.5), beta U(+-0.2)."""
from __future__ import annotations

import math

import numpy as np

from . import _rng

_ST_GNET, _ST_GPOSE = 32, 33
OUT_CH = 11


def layer_shapes(width=256, n_res=28, sr_ch=(128, 64, 32), in_ch=6):
    out = [(width, in_ch, 1, True)] + [(width, width, 1, True)] * n_res
    c = width
    for ch in sr_ch:
        out += [(ch, c, 3, True), (ch, ch, 3, True), (OUT_CH, ch, 1, False)]
        c = ch
    return out


def make_gnet(seed: int, dtype: str = "f16", **kw) -> np.ndarray:
    """Flat fp32 blob, per layer W[Cout][Cin][k][k], b[Cout] and, for conv-norm-act layers, gamma[Cout], beta[Cout].
    dtype "f16": the conv WEIGHTS are rounded once (RNE) to fp16-representable values (the tensor-core operand type);
    biases and affine parameters stay fp32."""
    g = _rng(seed, _ST_GNET)
    parts = []
    for co, ci, k, norm in layer_shapes(**kw):
        a = 1.0 / math.sqrt(ci * k * k)
        W = ((g.random((co, ci, k, k)) * 2 - 1) * a).astype(np.float32)
        if dtype == "f16":
            W = W.astype(np.float16).astype(np.float32)
        parts += [W.ravel(), ((g.random(co) * 2 - 1) * a).astype(np.float32)]
        if norm:
            parts += [(0.5 + g.random(co)).astype(np.float32), ((g.random(co) * 2 - 1) * 0.2).astype(np.float32)]
    return np.concatenate(parts)


def make_rays(seed: int, h: int, w: int) -> np.ndarray:
    """gamma [h, w, 6] = [o, d_down]: a camera on the upper hemisphere about the scene centre
    looking at it; d_down = unit directions through the centres of an h x w pixel array."""
    g = _rng(seed, _ST_GPOSE)
    th = math.acos(g.uniform(0.2, 0.95)); ph = g.uniform(0, 2 * math.pi)
    c = np.array([0.5, 0.5, 0.5])
    o = c + 1.8 * np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)])
    fwd = (c - o) / np.linalg.norm(c - o)
    right = np.cross(fwd, [0.0, 0.0, 1.0]); right /= np.linalg.norm(right)
    up = np.cross(right, fwd)
    half = math.tan(math.radians(20.0))
    u = ((np.arange(w) + 0.5) / w * 2 - 1) * half
    v = (1 - (np.arange(h) + 0.5) / h * 2) * half * h / w
    d = fwd[None, None, :] + u[None, :, None] * right[None, None, :] + v[:, None, None] * up[None, None, :]
    d /= np.linalg.norm(d, axis=-1, keepdims=True)
    rays = np.concatenate([np.broadcast_to(o, d.shape), d], axis=-1)
    return np.ascontiguousarray(rays, dtype=np.float32)

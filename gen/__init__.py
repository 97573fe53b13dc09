"""Seeded synthetic input generators for the hash-grid renderer.

This module serves BOTH the CPU oracle and the CUDA path with bit-identical inputs and holds none of
the method's arithmetic: it only draws random tables / weights / scenes / direction sets.  It never
imports `oracle/` or `paper_2409_10327_b200/`.

The inputs stand in for the paper's workloads (800x800 frames of TensoIR-/InvRender-synthetic scenes,
HDR equirect env maps, spp 16-64, 8 tertiary rays: PAPER.md:120, 122, 344), none of which exist here.
Configs C0..C4 follow BASELINE.json `configs` (zero-indexed) as read in SURVEY.md section 8(d).

All randomness comes from numpy's counter-based Philox generator keyed by (seed, stream id), so every
blob is a pure function of (config, seed) and independent of the order blobs are requested in.
"""
from __future__ import annotations

import dataclasses
import math
from dataclasses import dataclass

import numpy as np

HR_DIRECT, HR_SHADOW, HR_INDIRECT, HR_DENSE = 1, 2, 4, 8

# stream ids (one independent Philox sub-stream per blob)
_ST_TABLE, _ST_BRDF_W, _ST_IRT_W, _ST_ENV, _ST_POINTS, _ST_SCENE, _ST_DIR_D, _ST_DIR_S, _ST_DIR_T = range(9)


def _rng(seed: int, stream: int, sub: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[(seed << 8) | stream, sub]))


@dataclass(frozen=True)
class Config:
    name: str
    seed: int
    N: int                      # primary points
    S_d: int                    # direct directions / point
    S_i: int                    # secondary directions / point (0 = none)
    S_2: int                    # tertiary directions / secondary point (shared set)
    L: int
    F: int
    log2_T: int
    base_res: int
    max_res: int
    table_scale: float          # tables ~ U(-scale, scale)
    table_dtype: str            # "f32" | "f16"
    mlp_dtype: str              # "f32" | "f16"
    env_hw: tuple               # (He, We); (0, 0) = none
    points: str                 # "sphere" | "scene" | "uniform"
    width: int = 0              # image width for "scene"
    flags: int = HR_DIRECT | HR_SHADOW
    hidden: int = 64
    near_t: float = 0.05
    far_t: float = 1.5
    rough_min: float = 0.09
    fresnel_f0: float = 0.04
    depth_bias: float = -1.5    # keeps x' inside the cube
    vis_bias: float = 0.0       # I's visibility bias b_v: centres z_v so hard visibility is neither all 0 nor all 1
                                # (presets: tests/golden/vis_bias.txt, written by tests/golden/make_vis_bias.py from the oracle)
    tol: float = 1e-4

    @property
    def T(self) -> int:
        return 1 << self.log2_T

    @property
    def D(self) -> int:
        return self.L * self.F

    @property
    def queries(self) -> int:
        """IRT (point, direction) evaluations per frame (SURVEY 8(d) metric unit)."""
        q = self.N * self.S_d
        if self.flags & HR_INDIRECT:
            q += self.N * self.S_i * (1 + self.S_2)
        return q


def make_config(name: str, **over) -> Config:
    """Named presets C0..C4 (BASELINE.json configs[0..4]); C3a = C1 in fp16; `over` overrides fields."""
    c0 = dict(seed=0, N=4096, S_d=8, S_i=0, S_2=8, L=8, F=2, log2_T=14, base_res=16, max_res=256,
              table_scale=1.0, table_dtype="f32", mlp_dtype="f32", env_hw=(16, 32), points="sphere", vis_bias=0.0986328125)
    c1 = dict(seed=1, N=640_000, S_d=128, S_i=0, S_2=8, L=16, F=2, log2_T=19, base_res=16, max_res=2048,
              table_scale=0.1, table_dtype="f32", mlp_dtype="f32", env_hw=(32, 64), points="scene", width=800, vis_bias=0.001953125)
    presets = {
        "C0": c0,
        "C1": c1,
        "C2": {**c1, "seed": 2, "S_i": 64, "flags": HR_DIRECT | HR_SHADOW | HR_INDIRECT, "vis_bias": -0.041015625},
        "C3": {**c1, "seed": 3, "S_i": 64, "flags": HR_DIRECT | HR_SHADOW | HR_INDIRECT,
               "table_dtype": "f16", "mlp_dtype": "f16", "tol": 3e-3, "vis_bias": 0.1259765625},
        "C3a": {**c1, "seed": 3, "table_dtype": "f16", "mlp_dtype": "f16", "tol": 3e-3, "vis_bias": 0.1259765625},
        "C4": dict(seed=4, N=1 << 20, S_d=1, S_i=0, S_2=0, L=16, F=2, log2_T=19, base_res=16, max_res=2048,
                   table_scale=0.1, table_dtype="f16", mlp_dtype="f16", env_hw=(0, 0), points="uniform",
                   tol=3e-3, vis_bias=-0.0166015625),
    }
    d = dict(presets[name])
    d.update(over)
    return Config(name=name, **d)


def with_points(cfg: Config, N: int) -> Config:
    return dataclasses.replace(cfg, N=int(N))


# --------------------------------------------------------------------------------------------------
# grid, tables, weights, env
# --------------------------------------------------------------------------------------------------
def resolutions(L: int, base_res: int, max_res: int) -> np.ndarray:
    """Geometric level resolutions N_l = floor(base * b^l), b = exp(ln(max/base)/(L-1)).

    The integers are computed ONCE here and handed to both sides as `res[L]`; a 1e-6 guard keeps the
    last level from flooring to max-1 through round-off.
    """
    if L == 1:
        return np.array([base_res], dtype=np.uint32)
    b = math.exp(math.log(max_res / base_res) / (L - 1))
    return np.array([int(math.floor(base_res * b ** l + 1e-6)) for l in range(L)], dtype=np.uint32)


def _round_dtype(a: np.ndarray, dtype: str) -> np.ndarray:
    """fp16 configs: round ONCE (RNE) here, return fp32 holding fp16-representable values."""
    a = a.astype(np.float32)
    if dtype == "f16":
        a = a.astype(np.float16).astype(np.float32)
    return a


def make_tables(cfg: Config) -> np.ndarray:
    """Hash tables [L][T][F] ~ U(-scale, scale); fp32 array (fp16-representable for f16 configs)."""
    out = np.empty((cfg.L, cfg.T, cfg.F), dtype=np.float32)
    for l in range(cfg.L):
        g = _rng(cfg.seed, _ST_TABLE, l)
        out[l] = (g.random((cfg.T, cfg.F), dtype=np.float32) * 2.0 - 1.0) * np.float32(cfg.table_scale)
    return _round_dtype(out, cfg.table_dtype)


def mlp_shapes(cfg: Config, which: str):
    d_in = cfg.D if which == "brdf" else cfg.D + 3
    d_out = 7 if which == "brdf" else 2
    return [(cfg.hidden, d_in), (cfg.hidden, cfg.hidden), (d_out, cfg.hidden)]


def make_mlp(cfg: Config, which: str) -> np.ndarray:
    """Weight blob: per layer W[out][in] (row-major) then b[out]; Xavier-uniform W, U(+-0.05) b."""
    g = _rng(cfg.seed, _ST_BRDF_W if which == "brdf" else _ST_IRT_W)
    parts = []
    shapes = mlp_shapes(cfg, which)
    for li, (o, i) in enumerate(shapes):
        a = math.sqrt(6.0 / (i + o))
        W = (g.random((o, i)) * 2.0 - 1.0) * a
        b = (g.random(o) * 2.0 - 1.0) * 0.05
        if which == "irt" and li == len(shapes) - 1:
            b[0] = cfg.vis_bias
            b[1] = cfg.depth_bias
        parts += [W.ravel(), b]
    return _round_dtype(np.concatenate(parts), cfg.mlp_dtype)


def split_mlp(cfg: Config, which: str, blob: np.ndarray):
    """Blob -> [(W[out,in], b[out])] views (layout helper, no arithmetic)."""
    out, off = [], 0
    for (o, i) in mlp_shapes(cfg, which):
        W = blob[off:off + o * i].reshape(o, i); off += o * i
        b = blob[off:off + o]; off += o
        out.append((W, b))
    assert off == blob.size
    return out


def make_env(cfg: Config) -> np.ndarray:
    He, We = cfg.env_hw
    if He == 0:
        return np.zeros((0, 0, 3), dtype=np.float32)
    g = _rng(cfg.seed, _ST_ENV)
    return np.exp(g.standard_normal((He, We, 3))).astype(np.float32)


# --------------------------------------------------------------------------------------------------
# points
# --------------------------------------------------------------------------------------------------
def _normalize(v):
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def _points_sphere(cfg: Config):
    g = _rng(cfg.seed, _ST_POINTS)
    n = _normalize(g.standard_normal((cfg.N, 3)))
    x = 0.5 + 0.5 * n                       # unit-DIAMETER sphere inscribed in [0,1]^3
    cam = np.array([0.5, -2.0, 0.5])
    wo = _normalize(cam - x)
    return x, n, wo


def _scene_shapes(seed: int):
    g = _rng(seed, _ST_SCENE)
    shapes = []
    for k in range(8):
        c = g.uniform(0.2, 0.8, 3)
        if k % 2 == 0:
            shapes.append(("sphere", c, g.uniform(0.08, 0.18)))
        else:
            shapes.append(("box", c, g.uniform(0.06, 0.15, 3)))
    return shapes


def _points_scene(cfg: Config, pix: np.ndarray):
    """Analytic ray cast of 8 random spheres/boxes inside an open-front unit-cube room; every pixel hits.

    `pix` = flat pixel indices (row-major over a width x width image, image-coherent order).
    """
    W = cfg.width
    py, px = np.divmod(pix.astype(np.int64), W)
    cam = np.array([0.5, -1.0, 0.5])
    # image plane = the open front face y=0 of the room, pixel centres
    tx = (px + 0.5) / W
    tz = 1.0 - (py + 0.5) / W
    target = np.stack([tx, np.zeros_like(tx), tz], axis=-1)
    d = _normalize(target - cam)
    o = np.broadcast_to(cam, d.shape)
    M = d.shape[0]
    tbest = np.full(M, np.inf)
    nbest = np.zeros((M, 3))
    # room: 5 inner faces (front y=0 is open)
    for axis, val, sign in [(1, 1.0, -1.0), (0, 0.0, 1.0), (0, 1.0, -1.0), (2, 0.0, 1.0), (2, 1.0, -1.0)]:
        with np.errstate(divide="ignore", invalid="ignore"):
            t = (val - o[:, axis]) / d[:, axis]
        p = o + t[:, None] * d
        ok = (t > 1e-9) & np.all((p > -1e-9) & (p < 1 + 1e-9), axis=1) & (t < tbest)
        tbest = np.where(ok, t, tbest)
        nn = np.zeros(3); nn[axis] = sign
        nbest[ok] = nn
    for kind, c, s in _scene_shapes(cfg.seed):
        if kind == "sphere":
            oc = o - c
            b = np.sum(oc * d, axis=1)
            cc = np.sum(oc * oc, axis=1) - s * s
            disc = b * b - cc
            t = -b - np.sqrt(np.maximum(disc, 0.0))
            ok = (disc > 0) & (t > 1e-9) & (t < tbest)
            tbest = np.where(ok, t, tbest)
            p = o + t[:, None] * d
            nbest[ok] = ((p - c) / s)[ok]
        else:
            with np.errstate(divide="ignore", invalid="ignore"):
                t0 = (c - s - o) / d
                t1 = (c + s - o) / d
            tn = np.minimum(t0, t1); tf = np.maximum(t0, t1)
            tnear = tn.max(axis=1); tfar = tf.min(axis=1)
            ok = (tnear < tfar) & (tnear > 1e-9) & (tnear < tbest)
            tbest = np.where(ok, tnear, tbest)
            ax = tn.argmax(axis=1)
            nn = np.zeros((M, 3))
            nn[np.arange(M), ax] = -np.sign(d[np.arange(M), ax])
            nbest[ok] = nn[ok]
    assert np.all(np.isfinite(tbest)), "every camera ray must hit the room or a shape"
    x = np.clip(o + tbest[:, None] * d, 0.0, 1.0)
    return x, _normalize(nbest), -d


def make_points(cfg: Config, pix: np.ndarray | None = None):
    """-> x[N,3], n_g[N,3] (geometric normal, used only to orient direction sets), wo[N,3]; fp32.

    `pix` selects a subset (pixel indices for "scene", row indices otherwise) WITHOUT changing the values
    of the selected points, so a sampled oracle run sees exactly the full frame's inputs.
    """
    if cfg.points == "scene":
        if pix is None:
            pix = np.arange(cfg.N)
        x, n, wo = _points_scene(cfg, np.asarray(pix))
    else:
        if cfg.points == "sphere":
            x, n, wo = _points_sphere(cfg)
        else:
            g = _rng(cfg.seed, _ST_POINTS)
            x = g.random((cfg.N, 3))
            n = _normalize(g.standard_normal((cfg.N, 3)))
            wo = n.copy()
        if pix is not None:
            x, n, wo = x[pix], n[pix], wo[pix]
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return f32(x), f32(n), f32(_normalize(wo.astype(np.float32).astype(np.float64)))


# --------------------------------------------------------------------------------------------------
# direction sets (inputs to the hot path: SURVEY A11/A12 are generator-side)
# --------------------------------------------------------------------------------------------------
def _frame(n):
    """Orthonormal tangent frame per normal (Frisvad-style branch on n_z sign, double precision)."""
    s = np.where(n[:, 2] >= 0, 1.0, -1.0)
    a = -1.0 / (s + n[:, 2])
    b = n[:, 0] * n[:, 1] * a
    t = np.stack([1.0 + s * n[:, 0] ** 2 * a, s * b, -s * n[:, 0]], axis=-1)
    bt = np.stack([b, s + n[:, 1] ** 2 * a, -n[:, 1]], axis=-1)
    return t, bt


def _point_keyed_uniform(seed: int, stream: int, ids: np.ndarray, S: int, chunk: int = 4096):
    """u[len(ids), S, 2] in [0,1): point `i` always draws the same numbers whichever subset it is in.

    Points are grouped in blocks of `chunk` consecutive ids; each block is its own Philox sub-stream.
    """
    ids = np.asarray(ids, dtype=np.int64)
    out = np.empty((ids.size, S, 2), dtype=np.float64)
    blocks = ids // chunk
    for b in np.unique(blocks):
        sel = np.nonzero(blocks == b)[0]
        u = _rng(seed, stream, int(b)).random((chunk, S, 2))
        out[sel] = u[ids[sel] - b * chunk]
    return out


def make_cosine_hemisphere_dirs(cfg: Config, n_g: np.ndarray, ids: np.ndarray, S: int, stream: int):
    """Stratified (sx x sy) cosine-weighted hemisphere about n_g; pdf = cos(theta)/pi.  -> dir[M,S,3], pdf[M,S]."""
    sx = 1 << ((S.bit_length() - 1 + 1) // 2)
    sy = S // sx
    assert sx * sy == S, "S must be a power of two"
    u = _point_keyed_uniform(cfg.seed, stream, ids, S)
    k = np.arange(S)
    u1 = ((k % sx)[None, :] + u[:, :, 0]) / sx
    u2 = ((k // sx)[None, :] + u[:, :, 1]) / sy
    r = np.sqrt(u1); phi = 2 * np.pi * u2
    lx, ly = r * np.cos(phi), r * np.sin(phi)
    lz = np.sqrt(np.maximum(1.0 - u1, 1e-12))
    t, bt = _frame(n_g.astype(np.float64))
    d = lx[..., None] * t[:, None, :] + ly[..., None] * bt[:, None, :] + lz[..., None] * n_g[:, None, :].astype(np.float64)
    d = _normalize(d).astype(np.float32)
    d = _normalize(d.astype(np.float64)).astype(np.float32)
    pdf = (lz / np.pi).astype(np.float32)
    return np.ascontiguousarray(d), np.ascontiguousarray(pdf)


def make_env_importance_dirs(cfg: Config, env: np.ndarray, ids: np.ndarray, S: int):
    """Light-importance directions: texel prob ~ luminance*sin(theta), jittered inside the texel.

    Equirect convention: z-up, theta from +z, phi = atan2(y, x), u = (phi/2pi + 1/2) We.
    pdf(omega) = P_texel / (dtheta * dphi * sin(theta)).  -> dir[M,S,3], pdf[M,S]
    """
    He, We, _ = env.shape
    lum = env.astype(np.float64) @ np.array([0.2126, 0.7152, 0.0722])
    th_c = (np.arange(He) + 0.5) / He * np.pi
    w = lum * np.sin(th_c)[:, None]
    P = (w / w.sum()).ravel()
    cdf = np.cumsum(P); cdf[-1] = 1.0
    M = len(ids)
    g = _point_keyed_uniform(cfg.seed, _ST_DIR_D, ids, 2 * S).reshape(M, S, 4)
    us = (np.arange(S)[None, :] + g[:, :, 0]) / S            # stratified over the texel CDF
    tex = np.minimum(np.searchsorted(cdf, us, side="right"), He * We - 1)
    ty, tx = np.divmod(tex, We)
    theta = (ty + g[:, :, 1]) / He * np.pi
    phi = ((tx + g[:, :, 2]) / We - 0.5) * 2 * np.pi
    st = np.sin(theta)
    d = np.stack([st * np.cos(phi), st * np.sin(phi), np.cos(theta)], axis=-1)
    d = _normalize(d).astype(np.float32)
    d = _normalize(d.astype(np.float64)).astype(np.float32)
    pdf = P[tex] / ((np.pi / He) * (2 * np.pi / We) * np.maximum(st, 1e-9))
    return np.ascontiguousarray(d), np.ascontiguousarray(pdf.astype(np.float32))


def make_sphere_dirs_shared(cfg: Config, S: int):
    """One SHARED stratified whole-sphere set (point_stride = 0), pdf = 1/(4 pi)."""
    if S == 0:
        return np.zeros((0, 3), np.float32), np.zeros((0,), np.float32)
    g = _rng(cfg.seed, _ST_DIR_T)
    sx = 1 << ((S.bit_length() - 1 + 1) // 2)
    sy = S // sx
    u = g.random((S, 2))
    k = np.arange(S)
    phi = 2 * np.pi * ((k % sx) + u[:, 0]) / sx
    cz = 1.0 - 2.0 * ((k // sx) + u[:, 1]) / sy
    sz = np.sqrt(np.maximum(1 - cz * cz, 0))
    d = np.stack([sz * np.cos(phi), sz * np.sin(phi), cz], axis=-1)
    d = _normalize(_normalize(d).astype(np.float32).astype(np.float64)).astype(np.float32)
    return np.ascontiguousarray(d), np.full((S,), 1.0 / (4 * np.pi), dtype=np.float32)


def make_uniform_sphere_dirs(cfg: Config, ids: np.ndarray, S: int):
    u = _point_keyed_uniform(cfg.seed, _ST_DIR_D, ids, S)
    cz = 1 - 2 * u[:, :, 0]; phi = 2 * np.pi * u[:, :, 1]
    sz = np.sqrt(np.maximum(1 - cz * cz, 0))
    d = np.stack([sz * np.cos(phi), sz * np.sin(phi), cz], axis=-1)
    d = _normalize(_normalize(d).astype(np.float32).astype(np.float64)).astype(np.float32)
    return np.ascontiguousarray(d), np.full(d.shape[:2], 1.0 / (4 * np.pi), dtype=np.float32)


# --------------------------------------------------------------------------------------------------
# whole workloads
# --------------------------------------------------------------------------------------------------
def make_model(cfg: Config) -> dict:
    """Frame-independent blobs: res, tables, weights, env."""
    return dict(res=resolutions(cfg.L, cfg.base_res, cfg.max_res), tables=make_tables(cfg),
                brdf_w=make_mlp(cfg, "brdf"), irt_w=make_mlp(cfg, "irt"), env=make_env(cfg))


def _make_frame_chunk(cfg: Config, env: np.ndarray, ids: np.ndarray, subset: bool) -> dict:
    x, n_g, wo = make_points(cfg, ids if (subset or cfg.points == "scene") else None)
    fr = dict(x=x, n_g=n_g, wo=wo)
    if cfg.points == "scene":
        fr["dir_d"], fr["pdf_d"] = make_env_importance_dirs(cfg, env, ids, cfg.S_d)
    elif cfg.points == "sphere":
        fr["dir_d"], fr["pdf_d"] = make_cosine_hemisphere_dirs(cfg, n_g, ids, cfg.S_d, _ST_DIR_D)
    else:
        fr["dir_d"], fr["pdf_d"] = make_uniform_sphere_dirs(cfg, ids, cfg.S_d)
    if cfg.S_i:
        fr["dir_s"], fr["pdf_s"] = make_cosine_hemisphere_dirs(cfg, n_g, ids, cfg.S_i, _ST_DIR_S)
    return fr


def make_frame(cfg: Config, env: np.ndarray, pix: np.ndarray | None = None, chunk: int = 32768) -> dict:
    """Per-frame inputs for the points `pix` (default: all N): x, n_g, wo, direction sets + pdfs.

    A point's inputs depend only on (config, seed, point id), never on which subset it is generated in.
    """
    ids = np.arange(cfg.N) if pix is None else np.asarray(pix, dtype=np.int64)
    if cfg.points == "scene" or pix is not None:
        parts = [_make_frame_chunk(cfg, env, ids[i:i + chunk], True) for i in range(0, len(ids), chunk)]
        fr = {k: np.concatenate([p[k] for p in parts]) for k in parts[0]} if parts else {}
    else:
        fr = _make_frame_chunk(cfg, env, ids, False)
    fr["ids"] = ids
    fr["dir_t"], fr["pdf_t"] = make_sphere_dirs_shared(cfg, cfg.S_2)
    return fr

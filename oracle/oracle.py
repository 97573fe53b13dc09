"""ctypes front-end of the CPU oracle (oracle/hashrender_oracle.cpp) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It never imports paper_2409_10327_b200 (the CUDA path) and shares nothing with it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hashrender_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """g++ -O2, no fast-math, no FMA contraction (keeps the fp32 index path one IEEE multiply)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off",
                               "-fno-fast-math", "-o", _LIB, _SRC])
    return _LIB


class OrConfig(C.Structure):
    _fields_ = [("L", C.c_uint32), ("F", C.c_uint32), ("log2_T", C.c_uint32), ("res", C.POINTER(C.c_uint32)),
                ("hidden", C.c_uint32), ("near_t", C.c_float), ("far_t", C.c_float), ("rough_min", C.c_float),
                ("fresnel_f0", C.c_float), ("vis_mode", C.c_uint32), ("brdf_model", C.c_uint32),
                ("albedo_scale", C.c_float * 3), ("He", C.c_uint32), ("We", C.c_uint32)]


class OrDirset(C.Structure):
    _fields_ = [("dir", C.c_void_p), ("pdf", C.c_void_p), ("Lin", C.c_void_p), ("S", C.c_uint32),
                ("point_stride", C.c_uint64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.or_hash_index.restype = C.c_uint32
        _lib.or_hash_index.argtypes = [C.c_uint32] * 4
        _lib.or_grid_index.restype = C.c_uint32
        _lib.or_grid_index.argtypes = [C.c_uint32] * 5
        _lib.or_level_is_dense.restype = C.c_int
        _lib.or_level_is_dense.argtypes = [C.c_uint32] * 2
    return _lib


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


class Oracle:
    """Holds one model (grid + weights + env) and evaluates the path on it, in double precision."""

    def __init__(self, *, L, F, log2_T, res, tables, brdf_w, irt_w, env=None, hidden=64, near_t=0.05, far_t=1.5,
                 rough_min=0.09, fresnel_f0=0.04, vis_mode=0, brdf_model=1, albedo_scale=(1.0, 1.0, 1.0)):
        self.res = np.ascontiguousarray(res, dtype=np.uint32)
        self.tables = _f32(tables)
        assert self.tables.size == L * (1 << log2_T) * F
        self.brdf_w, self.irt_w = _f32(brdf_w), _f32(irt_w)
        self.env = _f32(env) if env is not None and np.size(env) else np.zeros((1, 1, 3), np.float32)
        self.L, self.F, self.D = L, F, L * F
        self.cfg = OrConfig(L=L, F=F, log2_T=log2_T, res=self.res.ctypes.data_as(C.POINTER(C.c_uint32)), hidden=hidden,
                            near_t=near_t, far_t=far_t, rough_min=rough_min, fresnel_f0=fresnel_f0, vis_mode=vis_mode,
                            brdf_model=brdf_model, albedo_scale=(C.c_float * 3)(*albedo_scale),
                            He=self.env.shape[0], We=self.env.shape[1])
        self.hidden = hidden

    @classmethod
    def from_gen(cls, cfg, model, **over):
        kw = dict(L=cfg.L, F=cfg.F, log2_T=cfg.log2_T, res=model["res"], tables=model["tables"], brdf_w=model["brdf_w"],
                  irt_w=model["irt_w"], env=model["env"], hidden=cfg.hidden, near_t=cfg.near_t, far_t=cfg.far_t,
                  rough_min=cfg.rough_min, fresnel_f0=cfg.fresnel_f0)
        kw.update(over)
        return cls(**kw)

    def set_modes(self, vis_mode=None, brdf_model=None):
        if vis_mode is not None:
            self.cfg.vis_mode = vis_mode
        if brdf_model is not None:
            self.cfg.brdf_model = brdf_model

    # -- helpers ---------------------------------------------------------------------------------
    @staticmethod
    def dirset(dir, pdf, Lin=None, shared=None):
        """dir [N,S,3] (or [S,3] shared), pdf [N,S] (or [S]).  Returns (OrDirset, keepalive)."""
        dir = _f32(dir); pdf = _f32(pdf)
        if shared is None:
            shared = dir.ndim == 2
        S = dir.shape[-2]
        Lin = None if Lin is None else _f32(Lin)
        ds = OrDirset(dir=dir.ctypes.data, pdf=pdf.ctypes.data, Lin=None if Lin is None else Lin.ctypes.data,
                      S=S, point_stride=0 if shared else 3 * S)
        return ds, (dir, pdf, Lin)

    # -- stages -----------------------------------------------------------------------------------
    def encode(self, x, want_idx=True):
        x = _f32(x); N = x.shape[0]
        feat = np.empty((N, self.D), np.float64)
        idx = np.empty((N, self.L, 8), np.uint32) if want_idx else None
        w = np.empty((N, self.L, 3), np.float32) if want_idx else None
        lib().or_encode(C.byref(self.cfg), _p(self.tables), _p(x), C.c_uint64(N), _p(feat), _p(idx), _p(w))
        return feat, idx, w

    def mlp3(self, blob, d_in, d_out, inp):
        inp = _f64(inp); N = inp.shape[0]
        out = np.empty((N, d_out), np.float64)
        lib().or_mlp3(_p(_f32(blob)), C.c_uint32(d_in), C.c_uint32(self.hidden), C.c_uint32(d_out), _p(inp), C.c_uint64(N), _p(out))
        return out

    def decode(self, feat):
        feat = _f64(feat); N = feat.shape[0]
        brdf = np.empty((N, 7), np.float64)
        lib().or_decode(C.byref(self.cfg), _p(self.brdf_w), _p(feat), C.c_uint64(N), _p(brdf))
        return brdf

    def trace(self, x, feat, dir, shared=None):
        x = _f32(x); feat = _f64(feat); N = x.shape[0]
        ds, keep = self.dirset(dir, np.ones(np.shape(dir)[:-1], np.float32), shared=shared)
        S = ds.S
        vis = np.empty((N, S)); zv = np.empty((N, S)); t = np.empty((N, S))
        xsec = np.empty((N, S, 3), np.float32)
        lib().or_trace(C.byref(self.cfg), _p(self.irt_w), _p(x), _p(feat), C.c_uint64(N), C.byref(ds), _p(vis), _p(zv), _p(t), _p(xsec))
        return vis, zv, t, xsec

    def env_lookup(self, dirs):
        dirs = _f64(dirs).reshape(-1, 3)
        rgb = np.empty_like(dirs)
        lib().or_env_lookup(C.byref(self.cfg), _p(self.env), _p(dirs), C.c_uint64(dirs.shape[0]), _p(rgb))
        return rgb

    def brdf_eval(self, brdf7, wi, wo):
        fr = np.empty(3)
        lib().or_brdf_eval(C.byref(self.cfg), _p(_f64(brdf7)), _p(_f64(wi)), _p(_f64(wo)), _p(fr))
        return fr

    def shade(self, brdf, wo, dir, pdf, vis, Lind=None, Lin=None, terms=3, shared=None):
        brdf = _f64(brdf); wo = _f32(wo); N = brdf.shape[0]
        ds, keep = self.dirset(dir, pdf, Lin, shared=shared)
        vis = _f64(vis); Lind = None if Lind is None else _f64(Lind)
        rgb = np.empty((N, 3))
        lib().or_shade(C.byref(self.cfg), _p(self.env), _p(brdf), _p(wo), C.c_uint64(N), C.byref(ds), _p(vis), _p(Lind),
                       C.c_uint32(terms), _p(rgb))
        return rgb

    def render_frame(self, x, wo, direct, secondary=None, tertiary=None, flags=3, brdf=None, mask=None, delta=0.0):
        """direct/secondary/tertiary: (dir, pdf[, Lin]) tuples or None.  -> dict(rgb, flipbound, n_sec, n_sec_clamped)."""
        x = _f32(x); wo = _f32(wo); N = x.shape[0]
        keep = []

        def mk(t):
            if t is None:
                return None
            ds, k = self.dirset(*t)
            keep.append(k)
            return ds
        d, s, tt = mk(direct), mk(secondary), mk(tertiary)
        brdf = None if brdf is None else _f32(brdf)
        mask = None if mask is None else np.ascontiguousarray(mask, dtype=np.uint8)
        rgb = np.empty((N, 3)); fb = np.empty((N, 3)); stats = np.zeros(2, np.uint64)
        ref = lambda z: None if z is None else C.byref(z)
        lib().or_render_frame(C.byref(self.cfg), _p(self.tables), _p(self.brdf_w), _p(self.irt_w), _p(self.env),
                              C.c_uint64(N), _p(x), _p(brdf), _p(wo), _p(mask), ref(d), ref(s), ref(tt),
                              C.c_uint32(flags), C.c_double(delta), _p(rgb), _p(fb), _p(stats))
        return dict(rgb=rgb, flipbound=fb, n_sec=int(stats[0]), n_sec_clamped=int(stats[1]))

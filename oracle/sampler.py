"""ctypes front-end of the CPU sampler oracle (oracle/sampler_oracle.cpp) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__ and bench.py's oracle legs import this; it never imports paper_2409_10327_b200."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sampler_oracle.cpp")
_LIB = os.path.join(_HERE, "libsampler_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math", "-o", _LIB, _SRC])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.ors_rng_bits.restype = C.c_uint32
        _lib.ors_rng_bits.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32]
        _lib.ors_rng_uniform.restype = C.c_float
        _lib.ors_rng_uniform.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32]
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def rng_bits(seed, row, sample, dim):
    return int(lib().ors_rng_bits(seed, row, sample, dim))


def rng_uniform(seed, row, sample, dim):
    return float(lib().ors_rng_uniform(seed, row, sample, dim))


def light_tables(env):
    env = _f32(env); He, We = env.shape[:2]
    pmf = np.empty((He, We), np.float64); cdf = np.empty(He * We, np.float32)
    lib().ors_light_tables(_p(env), C.c_uint32(He), C.c_uint32(We), _p(pmf), _p(cdf))
    return pmf, cdf


def light_pdf(env, dirs):
    env = _f32(env); He, We = env.shape[:2]
    d = _f64(dirs).reshape(-1, 3); out = np.empty(len(d), np.float64)
    lib().ors_light_pdf(_p(env), C.c_uint32(He), C.c_uint32(We), _p(d), C.c_uint64(len(d)), _p(out))
    return out.reshape(np.shape(dirs)[:-1])


def ggx_pdf(n, rough, wo, wi):
    n, wo, wi = (_f64(np.broadcast_to(a, np.shape(wi))).reshape(-1, 3) for a in (n, wo, wi))
    r = _f64(np.broadcast_to(rough, (len(wi),))); out = np.empty(len(wi), np.float64)
    lib().ors_ggx_pdf(_p(n), _p(r), _p(wo), _p(wi), C.c_uint64(len(wi)), _p(out))
    return out


def ggx_sample(n, rough, wo, u):
    u = _f64(u).reshape(-1, 2); M = len(u)
    n, wo = (_f64(np.broadcast_to(a, (M, 3))) for a in (n, wo))
    r = _f64(np.broadcast_to(rough, (M,))); out = np.empty((M, 3), np.float64)
    lib().ors_ggx_sample(_p(n), _p(r), _p(wo), _p(u), C.c_uint64(M), _p(out))
    return out


def sample_mis(env, brdf, wo, spp, seed):
    """-> dir [N, 2 spp, 3], pdf [N, 2 spp] (balance heuristic), texel [N, spp]; slot 2s = light ray, 2s+1 = GGX ray."""
    env = _f32(env); He, We = env.shape[:2]
    brdf, wo = _f32(brdf), _f32(wo); N = len(brdf)
    d = np.empty((N, 2 * spp, 3), np.float64); p = np.empty((N, 2 * spp), np.float64); t = np.empty((N, spp), np.uint32)
    lib().ors_sample_mis(_p(env), C.c_uint32(He), C.c_uint32(We), _p(brdf), _p(wo), C.c_uint64(N), C.c_uint32(spp), C.c_uint64(seed),
                         _p(d), _p(p), _p(t))
    return d, p, t


def sample_stratified(normal, rows, Sa, Sb, seed):
    """-> dir [rows, Sa*Sb, 3], pdf [rows, Sa*Sb]; normal None = whole sphere, else cosine hemisphere about normal[row]."""
    nrm = None if normal is None else _f32(normal)
    d = np.empty((rows, Sa * Sb, 3), np.float64); p = np.empty((rows, Sa * Sb), np.float64)
    lib().ors_sample_stratified(None if nrm is None else _p(nrm), C.c_uint64(rows), C.c_uint32(Sa), C.c_uint32(Sb), C.c_uint64(seed), _p(d), _p(p))
    return d, p

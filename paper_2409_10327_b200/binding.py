"""ctypes binding of include/hashrender.h.  Same names as the C ABI; marshals torch CUDA tensors (device
pointers) and numpy arrays (host pointers) into plain pointers + sizes.  No arithmetic happens here, and there
is NO fallback: if the CUDA library cannot be loaded every call raises."""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

HR_DIRECT, HR_SHADOW, HR_INDIRECT, HR_DENSE = 1, 2, 4, 8
HR_TERM_DIRECT, HR_TERM_INDIRECT = 1, 2
_STATUS = {1: "HR_ERR_INVALID_ARG", 2: "HR_ERR_CUDA", 3: "HR_ERR_OOM", 4: "HR_ERR_UNSUPPORTED"}
DENOISE_STATIC_MAX_PIXELS = 640000      # HASHRENDER_DENOISE_STATIC_MAX_PIXELS of include/hashrender.h
_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libhashrender.so")

EXPORTS = ["hashrender_create", "hashrender_destroy", "hashrender_set_env", "hashrender_encode", "hashrender_decode",
           "hashrender_trace", "hashrender_shade", "hashrender_render_frame", "hashrender_render_frame_host",
           "hashrender_sample_mis", "hashrender_sample_stratified", "hashrender_denoise", "hashrender_denoise_static", "hashrender_table_layout", "hashrender_probe_gather", "hashrender_stats", "hashrender_launch_count", "hashrender_last_path", "hashrender_last_error",
           "hashrender_gbuffer_create", "hashrender_gbuffer_destroy", "hashrender_gbuffer_forward", "hashrender_gbuffer_launch_count",
           "hashrender_gbuffer_flops", "hashrender_gbuffer_last_error"]


class HashRenderError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{_STATUS.get(code, code)}: {msg}")
        self.code = code


class hr_config(C.Structure):
    _fields_ = [("L", C.c_uint32), ("F", C.c_uint32), ("log2_T", C.c_uint32), ("res", C.POINTER(C.c_uint32)),
                ("table_dtype", C.c_uint32), ("mlp_dtype", C.c_uint32), ("hidden", C.c_uint32), ("brdf_out", C.c_uint32),
                ("irt_out", C.c_uint32), ("near_t", C.c_float), ("far_t", C.c_float), ("rough_min", C.c_float),
                ("fresnel_f0", C.c_float), ("vis_mode", C.c_uint32), ("brdf_model", C.c_uint32),
                ("albedo_scale", C.c_float * 3), ("max_points", C.c_uint64)]


class hr_dirset(C.Structure):
    _fields_ = [("dir", C.c_void_p), ("pdf", C.c_void_p), ("Lin", C.c_void_p), ("S", C.c_uint32), ("point_stride", C.c_uint64)]


class hr_denoise(C.Structure):
    _fields_ = [("H", C.c_uint32), ("W", C.c_uint32), ("rgb", C.c_void_p), ("albedo", C.c_void_p), ("normal", C.c_void_p),
                ("pos", C.c_void_p), ("cam", C.c_float * 3), ("mask", C.c_void_p), ("iterations", C.c_uint32),
                ("sigma_z", C.c_float), ("sigma_n", C.c_float), ("sigma_l", C.c_float)]


class hr_gnet_config(C.Structure):
    _fields_ = [("h", C.c_uint32), ("w", C.c_uint32), ("width", C.c_uint32), ("n_res", C.c_uint32), ("sr_ch", C.c_uint32 * 3),
                ("rough_min", C.c_float)]


class hr_frame(C.Structure):
    _fields_ = [("N", C.c_uint64), ("x", C.c_void_p), ("brdf", C.c_void_p), ("wo", C.c_void_p), ("mask", C.c_void_p),
                ("direct", hr_dirset), ("secondary", hr_dirset), ("tertiary", hr_dirset), ("flags", C.c_uint32)]


_lib = None


def load_library(path: str | None = None):
    """Loads libhashrender.so (must have been built: `python -m paper_2409_10327_b200.build`).  Fails loudly."""
    global _lib
    if _lib is None:
        p = path or _LIB_PATH
        if not os.path.exists(p):
            raise ImportError(f"{p} not found: build it with `python -m paper_2409_10327_b200.build` "
                              "(there is no CPU fallback)")
        lib = C.CDLL(p)
        vp, u64, u32 = C.c_void_p, C.c_uint64, C.c_uint32
        lib.hashrender_create.argtypes = [C.POINTER(hr_config), vp, vp, vp, C.POINTER(vp)]
        lib.hashrender_destroy.argtypes = [vp]
        lib.hashrender_set_env.argtypes = [vp, vp, u32, u32, vp]
        lib.hashrender_encode.argtypes = [vp, vp, u64, vp, vp, vp, vp]
        lib.hashrender_decode.argtypes = [vp, vp, u64, vp, vp]
        lib.hashrender_trace.argtypes = [vp, vp, vp, u64, C.POINTER(hr_dirset), vp, vp, vp, vp, vp]
        lib.hashrender_shade.argtypes = [vp, vp, vp, u64, C.POINTER(hr_dirset), vp, vp, u32, vp, vp]
        lib.hashrender_render_frame.argtypes = [vp, C.POINTER(hr_frame), vp, vp]
        lib.hashrender_render_frame_host.argtypes = [vp, C.POINTER(hr_frame), vp, vp, C.POINTER(u64), C.POINTER(u64)]
        lib.hashrender_sample_mis.argtypes = [vp, vp, vp, u64, u32, u64, vp, vp, vp]
        lib.hashrender_sample_stratified.argtypes = [vp, vp, u64, u32, u32, u64, vp, vp, vp]
        lib.hashrender_denoise.argtypes = [vp, C.POINTER(hr_denoise), vp, vp]
        lib.hashrender_denoise_static.argtypes = [vp, C.POINTER(hr_denoise), vp, vp]
        lib.hashrender_stats.argtypes = [vp, C.POINTER(u64), C.POINTER(u64), C.c_int]
        lib.hashrender_table_layout.argtypes = [vp, C.POINTER(C.c_uint32), C.POINTER(u64)]
        lib.hashrender_probe_gather.argtypes = [u64, C.c_uint32, C.c_uint32, C.c_uint32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        lib.hashrender_launch_count.argtypes = [vp]
        lib.hashrender_launch_count.restype = u64
        lib.hashrender_last_path.argtypes = [vp]
        lib.hashrender_last_path.restype = C.c_char_p
        lib.hashrender_last_error.argtypes = [vp]
        lib.hashrender_last_error.restype = C.c_char_p
        lib.hashrender_gbuffer_create.argtypes = [C.POINTER(hr_gnet_config), vp, u64, C.POINTER(vp)]
        lib.hashrender_gbuffer_destroy.argtypes = [vp]
        lib.hashrender_gbuffer_forward.argtypes = [vp, vp, vp, vp, vp, vp, vp]
        lib.hashrender_gbuffer_launch_count.argtypes = [vp]
        lib.hashrender_gbuffer_launch_count.restype = u64
        lib.hashrender_gbuffer_flops.argtypes = [vp]
        lib.hashrender_gbuffer_flops.restype = C.c_double
        lib.hashrender_gbuffer_last_error.argtypes = [vp]
        lib.hashrender_gbuffer_last_error.restype = C.c_char_p
        special = ("hashrender_launch_count", "hashrender_last_path", "hashrender_last_error", "hashrender_gbuffer_launch_count",
                   "hashrender_gbuffer_flops", "hashrender_gbuffer_last_error")
        for name in EXPORTS:
            if name not in special:
                getattr(lib, name).restype = C.c_int
        _lib = lib
    return _lib


def _ptr(a):
    """torch tensor (any device) or numpy array -> raw pointer; None -> NULL.  Must be contiguous."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return C.c_void_p(a.ctypes.data)
    assert a.is_contiguous()
    return C.c_void_p(a.data_ptr())


_DT = {"f32": ("float32", 4), "u8": ("uint8", 1), "u32": ("uint32", 4), "i32": ("int32", 4)}


def _arg(a, what, dt="f32", where="device", align=4):
    """Marshals one array argument after checking what the C side cannot: element type, placement (the device entry points
    take device pointers, render_frame_host takes host pointers) and alignment.  A wrong dtype or a host array passed to a
    device call would otherwise be misread silently.  None -> NULL."""
    if a is None:
        return None
    names = [_DT[d][0] for d in (dt if isinstance(dt, tuple) else (dt,))]
    if isinstance(a, np.ndarray):
        kind, on_dev = a.dtype.name, False
    else:
        kind, on_dev = str(a.dtype).replace("torch.", ""), bool(a.is_cuda)
    if kind not in names:
        raise TypeError(f"{what}: expected {' / '.join(names)}, got {kind}")
    if where == "device" and not on_dev:
        raise TypeError(f"{what}: expected a CUDA tensor (device pointer), got a host array")
    if where == "host" and on_dev:
        raise TypeError(f"{what}: expected a host array, got a CUDA tensor")
    p = _ptr(a)
    if p.value is not None and p.value % align:
        raise ValueError(f"{what}: pointer must be {align}-byte aligned")
    return p


@dataclass
class DirSet:
    """dir [N,S,3] (or [S,3] = one shared set), pdf [N,S] (or [S]), optional Lin like dir."""
    dir: object
    pdf: object
    Lin: object = None
    S: int | None = None                 # directions used per point when the rows are padded (default: dir.shape[-2])
    point_stride: int | None = None      # floats of `dir` between points (default 3 * dir.shape[-2]; 0 = one shared set)

    def c(self, where="device") -> hr_dirset:
        for nm in ("dir", "pdf", "Lin"):
            _arg(getattr(self, nm), f"DirSet.{nm}", "f32", where)
        shared = self.dir.ndim == 2
        S = self.dir.shape[-2] if self.S is None else self.S
        stride = (0 if shared else 3 * self.dir.shape[-2]) if self.point_stride is None else self.point_stride
        return hr_dirset(dir=_ptr(self.dir), pdf=_ptr(self.pdf), Lin=_ptr(self.Lin), S=S, point_stride=stride)


class HashRenderer:
    """Owns one hashrender_t handle.  Methods mirror the C ABI one to one."""

    def __init__(self, *, L, F, log2_T, res, tables, brdf_w, irt_w, table_dtype="f32", mlp_dtype="f32", hidden=64,
                 near_t=0.05, far_t=1.5, rough_min=0.09, fresnel_f0=0.04, vis_mode=0, brdf_model=1,
                 albedo_scale=(1.0, 1.0, 1.0), max_points=1 << 20):
        self._lib = load_library()
        self._res = np.ascontiguousarray(res, dtype=np.uint32)
        tables = np.ascontiguousarray(tables, dtype=np.float32)
        brdf_w = np.ascontiguousarray(brdf_w, dtype=np.float32)
        irt_w = np.ascontiguousarray(irt_w, dtype=np.float32)
        assert tables.size == L * (1 << log2_T) * F
        assert brdf_w.size == hidden * (L * F) + hidden + hidden * hidden + hidden + 7 * hidden + 7
        assert irt_w.size == hidden * (L * F + 3) + hidden + hidden * hidden + hidden + 2 * hidden + 2
        self.L, self.F, self.D = L, F, L * F
        self.cfg = hr_config(L=L, F=F, log2_T=log2_T, res=self._res.ctypes.data_as(C.POINTER(C.c_uint32)),
                             table_dtype={"f32": 0, "f16": 1}[table_dtype], mlp_dtype={"f32": 0, "f16": 1}[mlp_dtype],
                             hidden=hidden, brdf_out=7, irt_out=2, near_t=near_t, far_t=far_t, rough_min=rough_min,
                             fresnel_f0=fresnel_f0, vis_mode=vis_mode, brdf_model=brdf_model,
                             albedo_scale=(C.c_float * 3)(*albedo_scale), max_points=max_points)
        self._h = C.c_void_p()
        rc = self._lib.hashrender_create(C.byref(self.cfg), _ptr(tables), _ptr(brdf_w), _ptr(irt_w), C.byref(self._h))
        if rc != 0:
            msg = self._lib.hashrender_last_error(self._h).decode() if self._h else "create failed"
            if self._h:
                self._lib.hashrender_destroy(self._h)
                self._h = C.c_void_p()
            raise HashRenderError(rc, msg)

    @classmethod
    def from_gen(cls, cfg, model, **over):
        kw = dict(L=cfg.L, F=cfg.F, log2_T=cfg.log2_T, res=model["res"], tables=model["tables"], brdf_w=model["brdf_w"],
                  irt_w=model["irt_w"], table_dtype=cfg.table_dtype, mlp_dtype=cfg.mlp_dtype, hidden=cfg.hidden,
                  near_t=cfg.near_t, far_t=cfg.far_t, rough_min=cfg.rough_min, fresnel_f0=cfg.fresnel_f0,
                  max_points=max(cfg.N, 1 << 16))
        kw.update(over)
        return cls(**kw)

    def _check(self, rc):
        if rc != 0:
            raise HashRenderError(rc, self._lib.hashrender_last_error(self._h).decode())

    def destroy(self):
        if getattr(self, "_h", None):
            self._lib.hashrender_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # ---- C ABI mirrors (device pointers; stream = int cudaStream_t handle or None) -----------------------
    def set_env(self, env, stream=None):
        self._check(self._lib.hashrender_set_env(self._h, _arg(env, "env"), env.shape[0], env.shape[1], stream))

    def encode(self, x, feat, idx=None, w=None, stream=None, N=None):
        n = N if N is not None else x.shape[0]
        self._check(self._lib.hashrender_encode(self._h, _arg(x, "x"), n, _arg(feat, "feat"), _arg(idx, "idx", ("u32", "i32")), _arg(w, "w"), stream))

    def decode(self, feat, brdf, stream=None):
        self._check(self._lib.hashrender_decode(self._h, _arg(feat, "feat"), feat.shape[0], _arg(brdf, "brdf"), stream))

    def trace(self, x, feat, ds: DirSet, vis, zv, t, xsec=None, stream=None, N=None):
        n = N if N is not None else (x.shape[0] if x is not None else feat.shape[0])
        d = ds.c()
        self._check(self._lib.hashrender_trace(self._h, _arg(x, "x"), _arg(feat, "feat", align=8), n, C.byref(d), _arg(vis, "vis"), _arg(zv, "zv"),
                                               _arg(t, "t"), _arg(xsec, "xsec"), stream))

    def shade(self, brdf, wo, ds: DirSet, vis, Lind, terms, rgb, stream=None):
        d = ds.c()
        self._check(self._lib.hashrender_shade(self._h, _arg(brdf, "brdf"), _arg(wo, "wo"), brdf.shape[0], C.byref(d), _arg(vis, "vis"),
                                               _arg(Lind, "Lind"), terms, _arg(rgb, "rgb"), stream))

    def make_frame(self, x, wo, direct: DirSet | None, secondary: DirSet | None = None, tertiary: DirSet | None = None,
                   flags=HR_DIRECT | HR_SHADOW, brdf=None, mask=None, N=None) -> hr_frame:
        z = hr_dirset()
        where = "host" if isinstance(x, np.ndarray) or not getattr(x, "is_cuda", False) else "device"    # all arrays of a frame live together
        fr = hr_frame(N=x.shape[0] if N is None else N, x=_arg(x, "x", "f32", where), brdf=_arg(brdf, "brdf", "f32", where),
                      wo=_arg(wo, "wo", "f32", where), mask=_arg(mask, "mask", "u8", where, 1),
                      direct=direct.c(where) if direct else z, secondary=secondary.c(where) if secondary else z,
                      tertiary=tertiary.c(where) if tertiary else z, flags=flags)
        fr._where = where
        fr._keep = (x, wo, direct, secondary, tertiary, brdf, mask)
        return fr

    def render_frame(self, frame: hr_frame, rgb, stream=None):
        if getattr(frame, "_where", "device") != "device":
            raise TypeError("render_frame takes a frame of device arrays (use render_frame_host for host arrays)")
        self._check(self._lib.hashrender_render_frame(self._h, C.byref(frame), _arg(rgb, "rgb"), stream))

    def render_frame_host(self, frame: hr_frame, rgb, stream=None):
        up, down = C.c_uint64(), C.c_uint64()
        if getattr(frame, "_where", "host") != "host":
            raise TypeError("render_frame_host takes a frame of host arrays")
        self._check(self._lib.hashrender_render_frame_host(self._h, C.byref(frame), _arg(rgb, "rgb", "f32", "host"), stream, C.byref(up), C.byref(down)))
        return up.value, down.value

    def sample_mis(self, brdf, wo, spp, seed, dir, pdf, stream=None):
        # k_sample_mis stores the (light, GGX) pdf pair of a sample as one float2
        self._check(self._lib.hashrender_sample_mis(self._h, _arg(brdf, "brdf"), _arg(wo, "wo"), brdf.shape[0], spp, seed, _arg(dir, "dir"),
                                                    _arg(pdf, "pdf", align=8), stream))

    def sample_stratified(self, normal, rows, Sa, Sb, seed, dir, pdf, stream=None):
        self._check(self._lib.hashrender_sample_stratified(self._h, _arg(normal, "normal"), rows, Sa, Sb, seed, _arg(dir, "dir"), _arg(pdf, "pdf"), stream))

    def denoise(self, rgb, normal, pos, cam, out, albedo=None, mask=None, iterations=5, sigma_z=1.0, sigma_n=128.0, sigma_l=4.0,
                stream=None, static_scratch=False):
        """rgb / normal / pos / out: [H, W, 3] device tensors; cam: 3 floats.  static_scratch: hashrender_denoise_static (no
        allocation; the planes live in the library's fixed device array, at most DENOISE_STATIC_MAX_PIXELS pixels)."""
        d = hr_denoise(H=rgb.shape[0], W=rgb.shape[1], rgb=_arg(rgb, "rgb"), albedo=_arg(albedo, "albedo"), normal=_arg(normal, "normal"),
                       pos=_arg(pos, "pos"), cam=(C.c_float * 3)(*[float(v) for v in cam]), mask=_arg(mask, "mask", "u8", align=1),
                       iterations=iterations, sigma_z=sigma_z, sigma_n=sigma_n, sigma_l=sigma_l)
        fn = self._lib.hashrender_denoise_static if static_scratch else self._lib.hashrender_denoise
        self._check(fn(self._h, C.byref(d), _arg(out, "out"), stream))

    def denoise_static(self, rgb, normal, pos, cam, out, **kw):
        self.denoise(rgb, normal, pos, cam, out, static_scratch=True, **kw)

    def stats(self, reset=False):
        """(secondary rays traced, secondary rays whose L'_o was evaluated) since the last reset."""
        a, b = C.c_uint64(), C.c_uint64()
        self._check(self._lib.hashrender_stats(self._h, C.byref(a), C.byref(b), 1 if reset else 0))
        return a.value, b.value

    def table_layout(self):
        """(number of cell-major levels, bytes of the device copy of the tables)."""
        a, b = C.c_uint32(), C.c_uint64()
        self._check(self._lib.hashrender_table_layout(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def launch_count(self) -> int:
        return int(self._lib.hashrender_launch_count(self._h))

    def last_path(self) -> str:
        return self._lib.hashrender_last_path(self._h).decode()


def probe_gather(table_bytes, width=4, group=1, smem_bytes=0):
    """hashrender_probe_gather on the current device: (loads per cycle and SM, loads per second)."""
    lib = load_library()
    a, b = C.c_double(), C.c_double()
    rc = lib.hashrender_probe_gather(table_bytes, width, group, smem_bytes, C.byref(a), C.byref(b))
    if rc != 0:
        raise HashRenderError(rc, "hashrender_probe_gather")
    return a.value, b.value


class GBufferNet:
    """Owns one hr_gnet_t handle: the CNN direct renderer G (hashrender_gbuffer_*).  forward() fills the arrays hr_frame takes."""

    def __init__(self, weights, h, w, width=256, n_res=28, sr_ch=(128, 64, 32), rough_min=0.09):
        self._lib = load_library()
        weights = np.ascontiguousarray(weights, dtype=np.float32)
        self.cfg = hr_gnet_config(h=h, w=w, width=width, n_res=n_res, sr_ch=(C.c_uint32 * 3)(*sr_ch), rough_min=rough_min)
        self.h, self.w, self.N = h, w, 64 * h * w
        self._h = C.c_void_p()
        rc = self._lib.hashrender_gbuffer_create(C.byref(self.cfg), _ptr(weights), weights.size, C.byref(self._h))
        if rc != 0:
            msg = self._lib.hashrender_gbuffer_last_error(self._h).decode() if self._h else "create failed"
            if self._h:
                self._lib.hashrender_gbuffer_destroy(self._h)
                self._h = C.c_void_p()
            raise HashRenderError(rc, msg)

    def forward(self, rays, x=None, brdf=None, mask=None, raw=None, stream=None):
        rc = self._lib.hashrender_gbuffer_forward(self._h, _arg(rays, "rays"), _arg(x, "x"), _arg(brdf, "brdf"), _arg(mask, "mask", "u8", align=1),
                                                  _arg(raw, "raw"), stream)
        if rc != 0:
            raise HashRenderError(rc, self._lib.hashrender_gbuffer_last_error(self._h).decode())

    def launch_count(self) -> int:
        return int(self._lib.hashrender_gbuffer_launch_count(self._h))

    def flops(self) -> float:
        return float(self._lib.hashrender_gbuffer_flops(self._h))

    def destroy(self):
        if getattr(self, "_h", None):
            self._lib.hashrender_gbuffer_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

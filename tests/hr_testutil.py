"""Shared helpers for the GPU parity tests: upload generator blobs, call the C ABI, compare with the oracle."""
import numpy as np


def torch_dev():
    import torch
    return torch, torch.device("cuda:0")


def to_dev(a):
    torch, dev = torch_dev()
    return torch.from_numpy(np.ascontiguousarray(a)).to(dev)


def make_renderer(cfg, model, **over):
    from paper_2409_10327_b200 import HashRenderer
    r = HashRenderer.from_gen(cfg, model, **over)
    if model["env"].size:
        r.set_env(to_dev(model["env"]))
    return r


def gpu_render(r, cfg, fr, flags=None, brdf=None, mask=None, host=False):
    """Runs hashrender_render_frame on the generator frame `fr`; returns rgb [N,3] float32 (numpy)."""
    import torch
    from paper_2409_10327_b200 import DirSet
    flags = cfg.flags if flags is None else flags
    up = (lambda a: np.ascontiguousarray(a)) if host else to_dev
    x, wo = up(fr["x"]), up(fr["wo"])
    d = DirSet(up(fr["dir_d"]), up(fr["pdf_d"]))
    s = DirSet(up(fr["dir_s"]), up(fr["pdf_s"])) if "dir_s" in fr and (flags & 4) else None
    t = DirSet(up(fr["dir_t"]), up(fr["pdf_t"])) if (flags & 4) else None
    b = None if brdf is None else up(np.asarray(brdf, np.float32))
    m = None if mask is None else up(np.asarray(mask, np.uint8))
    frame = r.make_frame(x, wo, d, s, t, flags=flags, brdf=b, mask=m)
    N = fr["x"].shape[0]
    if host:
        rgb = np.empty((N, 3), np.float32)
        r.render_frame_host(frame, rgb)
        return rgb
    rgb = torch.full((N, 3), float("nan"), device="cuda:0", dtype=torch.float32)
    r.render_frame(frame, rgb)
    torch.cuda.synchronize()
    return rgb.cpu().numpy()


def oracle_render(o, cfg, fr, flags=None, delta=0.0, brdf=None, mask=None):
    flags = cfg.flags if flags is None else flags
    sec = (fr["dir_s"], fr["pdf_s"]) if "dir_s" in fr and (flags & 4) else None
    ter = (fr["dir_t"], fr["pdf_t"]) if (flags & 4) else None
    return o.render_frame(fr["x"], fr["wo"], (fr["dir_d"], fr["pdf_d"]), sec, ter, flags=flags, delta=delta, brdf=brdf, mask=mask)


def check_close(got, ref, tol, extra=None, what=""):
    """DESIGN.md Q32: pass iff |g - o| <= tol * max(|o|, s) (+ extra), s = mean |o| of the array.  Returns the
    worst ratio err / allowed, for reporting."""
    got = np.asarray(got, np.float64); ref = np.asarray(ref, np.float64)
    assert got.shape == ref.shape, (got.shape, ref.shape)
    assert np.all(np.isfinite(got)), f"{what}: non-finite GPU output"
    s = np.mean(np.abs(ref)) if ref.size else 0.0
    allowed = tol * np.maximum(np.abs(ref), s)
    if extra is not None:
        allowed = allowed + np.asarray(extra, np.float64)
    err = np.abs(got - ref)
    bad = err > allowed
    worst = float((err / np.maximum(allowed, 1e-300)).max()) if ref.size else 0.0
    assert not bad.any(), (f"{what}: {bad.sum()} / {bad.size} elements outside tol={tol}; worst err/allowed = {worst:.3g}; "
                           f"max abs err {err.max():.3g}, max|ref| {np.abs(ref).max():.3g}")
    return worst

"""The library only enqueues work on the caller's stream (include/hashrender.h, conventions), so its calls can be captured into CUDA
graphs as they stand.  Captured and replayed here: one frame of hashrender_render_frame (memset of the tile counter + the fused
kernel), the 77 launches of the G forward, and hashrender_denoise_static; each replay must reproduce the eager result (bit for bit where the
kernels are deterministic; the frame kernel and G's norm statistics add floats with atomics, so theirs agree to rounding)."""
import numpy as np
import pytest

import gen
from hr_testutil import make_renderer, to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available()
    return torch


def _capture(torch, fn):
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        fn(side.cuda_stream)
    return g


def test_render_frame_replays_from_a_cuda_graph(torch):
    from paper_2409_10327_b200 import DirSet
    cfg = gen.make_config("C3", N=640000)
    model = gen.make_model(cfg)
    pix = np.arange(0, cfg.N, 997)
    fr = gen.make_frame(cfg, model["env"], pix)
    r = make_renderer(cfg, model)
    frame = r.make_frame(to_dev(fr["x"]), to_dev(fr["wo"]), DirSet(to_dev(fr["dir_d"]), to_dev(fr["pdf_d"])),
                         DirSet(to_dev(fr["dir_s"]), to_dev(fr["pdf_s"])), DirSet(to_dev(fr["dir_t"]), to_dev(fr["pdf_t"])), flags=cfg.flags)
    n = len(pix)
    eager = torch.full((n, 3), float("nan"), device="cuda")
    r.render_frame(frame, eager)                                       # also warms up (lazy module load must not happen under capture)
    torch.cuda.synchronize()
    out = torch.full((n, 3), float("nan"), device="cuda")
    g = _capture(torch, lambda st: r.render_frame(frame, out, st))
    for _ in range(2):
        out.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        assert torch.allclose(out, eager, rtol=1e-4, atol=1e-6), float((out - eager).abs().max())
    assert float(eager.abs().mean()) > 0.01
    del g
    r.destroy()


def test_gbuffer_forward_and_static_denoise_replay_from_cuda_graphs(torch):
    from gen import gnet
    from paper_2409_10327_b200 import GBufferNet
    blob, rays = gnet.make_gnet(5), to_dev(gnet.make_rays(5, 10, 12))
    net = GBufferNet(blob, 10, 12)
    eager = torch.empty((net.N, 11), device="cuda")
    net.forward(rays, raw=eager)
    torch.cuda.synchronize()
    raw = torch.zeros((net.N, 11), device="cuda")
    g = _capture(torch, lambda st: net.forward(rays, raw=raw, stream=st))
    for _ in range(2):
        raw.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.allclose(raw, eager, rtol=1e-3, atol=1e-5), float((raw - eager).abs().max())
    del g
    net.destroy()
    # hashrender_denoise_static exists for exactly this caller: no allocation, so it can sit inside a capture
    cfg = gen.make_config("C1")
    model = gen.make_model(cfg)
    h, w = 64, 80
    ys, xs = np.mgrid[200:200 + h, 300:300 + w]
    fr = gen.make_frame(cfg, model["env"], (ys * 800 + xs).ravel())
    rng = np.random.default_rng(2)
    rgb = to_dev((0.5 + 0.3 * rng.standard_normal((h, w, 3))).astype(np.float32))
    nrm, pos = to_dev(fr["n_g"].reshape(h, w, 3)), to_dev(fr["x"].reshape(h, w, 3))
    r = make_renderer(cfg, model)
    ref = torch.empty((h, w, 3), device="cuda")
    r.denoise_static(rgb, nrm, pos, (0.5, 0.5, -1.2), ref)
    torch.cuda.synchronize()
    out = torch.zeros((h, w, 3), device="cuda")
    g = _capture(torch, lambda st: r.denoise_static(rgb, nrm, pos, (0.5, 0.5, -1.2), out, stream=st))
    out.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out, ref)
    del g
    r.destroy()

"""GPU parity of the CNN direct renderer G (hashrender_gbuffer_*: tcgen05 implicit-GEMM convolutions fed by TMA) against the
float64 oracle (oracle/gnet_oracle.py) on the same seeded weights and rays.

Tolerance (Q51): north_star's bar for fp16 operands, 3e-3 relative to max(|o|, mean |o|), on the raw outputs and on the
mapped arrays alike.  The operands of every MMA are fp16 (weights fp16-representable, activations as fp16 hi + lo pairs), the
accumulation is the tensor core's fp32, everything between two convolutions is fp32.  The random-weight network amplifies a
perturbation of its activations about a hundredfold over its 34 layers (measured on the oracle with rounded conv inputs: plain
fp16 activations give 8e-2, 28x over the bar), so what remains is the tensor core's fp32 accumulation over K up to 4608
amplified by the network: measured worst 1.6e-3.  The mask is an integer decided by a float: it must agree wherever |raw| >= 1e-2."""
import numpy as np
import pytest

from gen import gnet
from hr_testutil import check_close, to_dev

pytestmark = pytest.mark.gpu
TOL = 3e-3


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available()
    return torch


def _run(torch, blob, rays, **kw):
    from paper_2409_10327_b200 import GBufferNet
    h, w = rays.shape[:2]
    net = GBufferNet(blob, h, w, **kw)
    N = net.N
    x = torch.full((N, 3), float("nan"), device="cuda"); brdf = torch.full((N, 7), float("nan"), device="cuda")
    mask = torch.full((N,), 7, device="cuda", dtype=torch.uint8); raw = torch.full((N, 11), float("nan"), device="cuda")
    net.forward(to_dev(rays), x, brdf, mask, raw)
    torch.cuda.synchronize()
    out = dict(x=x.cpu().numpy(), brdf=brdf.cpu().numpy(), mask=mask.cpu().numpy(), raw=raw.cpu().numpy())
    return net, out


def _compare(got, ref, what):
    w = check_close(got["raw"], ref["raw"], TOL, what=f"{what} raw")
    check_close(got["x"], ref["x"], TOL, what=f"{what} x")
    check_close(got["brdf"][:, 3:], ref["brdf"][:, 3:], TOL, what=f"{what} a, r")
    # n = o/||o|| amplifies the error of o by 1/||o||
    nn = np.linalg.norm(ref["raw"][:, :3], axis=1, keepdims=True)
    check_close(got["brdf"][:, :3], ref["brdf"][:, :3], TOL, extra=TOL * np.abs(ref["raw"]).mean() / np.maximum(nn, 1e-9) * np.ones((1, 3)), what=f"{what} n")
    sure = np.abs(ref["raw"][:, 10]) >= 1e-2
    assert np.array_equal(got["mask"][sure], ref["mask"][sure]) and set(np.unique(got["mask"])) <= {0, 1}
    return w


@pytest.mark.parametrize("hw,kw", [((12, 16), {}), ((9, 5), {}), ((7, 10), dict(width=128, n_res=6, sr_ch=(64, 64, 32))),
                                   ((4, 4), dict(width=64, n_res=2, sr_ch=(32, 32, 32)))])
def test_gbuffer_matches_oracle_small(torch, hw, kw):
    """The paper's channel configuration on small ray arrays whose tiles are ragged in every direction (9 x 5 -> 72 x 40 pixels:
    neither multiple of the 16 x 8 output patch at the first block nor of 128 pixels), and two narrower networks."""
    from oracle import gnet_oracle as G
    blob = gnet.make_gnet(21, **kw)
    rays = gnet.make_rays(21, *hw)
    ref = G.forward(blob, rays, **kw)
    net, got = _run(torch, blob, rays, **kw)
    worst = _compare(got, ref, f"G {hw} {kw}")
    print(f"[gbuffer {hw} {kw}] pixels={net.N} launches={net.launch_count()} worst err/allowed={worst:.3f} (tol {TOL})")
    assert np.abs(ref["raw"]).mean() > 0.1 and 0.05 < ref["mask"].mean() < 0.95
    # a second forward on the same handle gives the same result (statistics buffers are re-zeroed; only the order of the
    # floating-point atomics of the instance-norm sums may differ)
    import torch as T
    raw2 = T.empty((net.N, 11), device="cuda")
    net.forward(to_dev(rays), raw=raw2)
    assert float((raw2.cpu() - T.from_numpy(got["raw"])).abs().max()) < 2e-4
    net.destroy()


def test_gbuffer_full_size_matches_oracle(torch):
    """The paper's shape: 100 x 100 rays -> 800 x 800 maps, every pixel compared with the oracle."""
    from oracle import gnet_oracle as G
    blob = gnet.make_gnet(22)
    rays = gnet.make_rays(22, 100, 100)
    ref = G.forward(blob, rays)
    net, got = _run(torch, blob, rays)
    assert net.N == 640000
    worst = _compare(got, ref, "G 100x100")
    print(f"[gbuffer full size] launches={net.launch_count()} flops={net.flops():.4g} worst err/allowed={worst:.3f} (tol {TOL})")
    net.destroy()


def test_gbuffer_feeds_the_hash_renderer(torch):
    """G's outputs are the arrays hr_frame takes: x, brdf, mask go straight into hashrender_render_frame, and the
    frame equals the oracle renderer on the oracle G's maps."""
    import gen
    from hr_testutil import make_renderer
    from oracle import gnet_oracle as G
    from oracle.oracle import Oracle
    from paper_2409_10327_b200 import DirSet, GBufferNet
    blob = gnet.make_gnet(23)
    rays = gnet.make_rays(23, 6, 8)
    ref = G.forward(blob, rays)
    net = GBufferNet(blob, 6, 8)
    N = net.N
    x = torch.empty((N, 3), device="cuda"); brdf = torch.empty((N, 7), device="cuda"); mask = torch.empty((N,), device="cuda", dtype=torch.uint8)
    net.forward(to_dev(rays), x, brdf, mask)
    cfg = gen.make_config("C1", N=N, S_d=16)
    m = gen.make_model(cfg)
    fr = gen.make_frame(cfg, m["env"], np.arange(N))
    r = make_renderer(cfg, m)
    wo = to_dev(fr["wo"])
    rgb = torch.empty((N, 3), device="cuda")
    r.render_frame(r.make_frame(x, wo, DirSet(to_dev(fr["dir_d"]), to_dev(fr["pdf_d"])), flags=3, brdf=brdf, mask=mask), rgb)
    o = Oracle.from_gen(cfg, m)
    sure = np.abs(ref["raw"][:, 10]) >= 1e-2
    want = o.render_frame(ref["x"].astype(np.float32), fr["wo"], (fr["dir_d"], fr["pdf_d"]), flags=3, brdf=ref["brdf"].astype(np.float32), mask=ref["mask"])
    got = rgb.cpu().numpy()
    # x moves by the G error (up to 3e-3 of sigma's range) and the hash grid amplifies that (SURVEY 8(c) conditioning note): loose bar,
    # the strict checks are the two parities this composes (G above, the renderer in test_gpu_parity.py)
    check_close(got[sure], want["rgb"][sure], 5e-2, what="G -> render_frame")
    assert np.abs(want["rgb"]).mean() > 0.01


def test_gbuffer_errors(torch):
    from paper_2409_10327_b200 import GBufferNet, HashRenderError
    blob = gnet.make_gnet(1)
    with pytest.raises(HashRenderError) as e:
        GBufferNet(blob[:-1], 4, 4)
    assert e.value.code == 1
    with pytest.raises(HashRenderError) as e:
        GBufferNet(blob, 4, 4, width=100)
    assert e.value.code == 4
    bad = gnet.make_gnet(1, dtype="f32")
    with pytest.raises(HashRenderError) as e:
        GBufferNet(bad, 4, 4)                         # weights that are not fp16-representable are refused, not rounded silently
    assert e.value.code == 1
    net = GBufferNet(blob, 4, 4)
    with pytest.raises(HashRenderError):
        net.forward(None, raw=torch.empty((net.N, 11), device="cuda"))

"""Pins of the CPU sampler oracle (oracle/sampler_oracle.cpp) against what the mathematics fixes -- no GPU.

PAPER.md:122 (MIS of a light-importance ray and a GGX-VNDF ray, balance heuristic), PAPER.md:344 / 338 (stratified rays).
A wrong pdf, a transposed frame, a dropped sin(theta) or a mis-scaled stratum fails one of these."""
import numpy as np
import pytest

from oracle import sampler as S

PI = np.pi


def _env(seed=0, hw=(16, 32)):
    return np.exp(np.random.default_rng(seed).standard_normal((*hw, 3))).astype(np.float32)


def _sphere_quadrature(nt=720, nph=1440):
    """Midpoint rule in (theta, phi): directions [nt*nph, 3] and solid-angle weights."""
    th = (np.arange(nt) + 0.5) * PI / nt
    ph = (np.arange(nph) + 0.5) * 2 * PI / nph - PI
    T, P = np.meshgrid(th, ph, indexing="ij")
    d = np.stack([np.sin(T) * np.cos(P), np.sin(T) * np.sin(P), np.cos(T)], -1).reshape(-1, 3)
    w = (np.sin(T) * (PI / nt) * (2 * PI / nph)).reshape(-1)
    return d, w


# ---------------------------------------------------------------------------------------------- generator (Q35)
def test_rng_is_a_pure_counter_function_with_24_bit_uniforms():
    a = S.rng_bits(5, 17, 3, 2)
    assert a == S.rng_bits(5, 17, 3, 2)
    assert len({S.rng_bits(5, 17, 3, 2), S.rng_bits(6, 17, 3, 2), S.rng_bits(5, 18, 3, 2), S.rng_bits(5, 17, 4, 2), S.rng_bits(5, 17, 3, 1),
                S.rng_bits(5 + (1 << 32), 17, 3, 2), S.rng_bits(5, 17 + (1 << 32), 3, 2)}) == 7
    u = S.rng_uniform(5, 17, 3, 2)
    assert 0.0 <= u < 1.0 and u == (a >> 8) / 2.0 ** 24


def test_rng_uniformity_and_independence():
    n = 40000
    u = np.array([[S.rng_uniform(11, r, 0, d) for d in range(3)] for r in range(n)])
    v = np.array([S.rng_uniform(11, 0, s, 0) for s in range(n)])
    for x in (u[:, 0], u[:, 1], u[:, 2], v):
        assert abs(x.mean() - 0.5) < 4 * np.sqrt(1 / 12 / n)
        assert abs(x.var() - 1 / 12) < 0.002
        chi2 = ((np.histogram(x, 64, (0, 1))[0] - n / 64) ** 2 / (n / 64)).sum()
        assert chi2 < 120                                              # 63 dof: mean 63, sd 11
    c = np.corrcoef(u.T)
    assert np.abs(c - np.eye(3)).max() < 0.02                          # dimensions of one sample are uncorrelated
    assert abs(np.corrcoef(u[:-1, 0], u[1:, 0])[0, 1]) < 0.02          # consecutive rows are uncorrelated
    h2 = np.histogram2d(u[:, 0], u[:, 1], 8, [[0, 1], [0, 1]])[0]
    assert ((h2 - n / 64) ** 2 / (n / 64)).sum() < 120


# ---------------------------------------------------------------------------------------------- light sampling (Q37)
def test_light_pmf_and_cdf():
    env = _env(1)
    pmf, cdf = S.light_tables(env)
    assert abs(pmf.sum() - 1) < 1e-12 and cdf[-1] == 1.0 and np.all(np.diff(cdf) >= 0)
    Y = env.astype(np.float64) @ [0.2126, 0.7152, 0.0722]
    w = Y * np.sin((np.arange(16) + 0.5) * PI / 16)[:, None]
    np.testing.assert_allclose(pmf, w / w.sum(), rtol=1e-12)
    np.testing.assert_allclose(cdf, np.cumsum(pmf.ravel()), atol=1e-6)


def test_light_pdf_integrates_to_one_and_follows_radiance():
    env = _env(2)
    d, w = _sphere_quadrature(480, 960)
    p = S.light_pdf(env, d)
    assert abs((p * w).sum() - 1) < 2e-3
    # inside one texel the density is pmf / (dtheta dphi sin theta): constant * 1/sin(theta)
    th = np.array([0.40, 0.41]) * PI
    dd = np.stack([np.sin(th) * np.cos(0.3), np.sin(th) * np.sin(0.3), np.cos(th)], -1)     # both in row 6 of 16
    q = S.light_pdf(env, dd)
    np.testing.assert_allclose(q[0] * np.sin(th[0]), q[1] * np.sin(th[1]), rtol=1e-12)


def test_light_rays_land_in_their_texel_and_match_the_pmf():
    env = np.full((8, 16, 3), 1e-6, np.float32)
    env[2, 5] = 7.0                                                    # (almost) one-hot map: every light ray goes to texel (2, 5)
    brdf = np.tile(np.array([[0, 0, 1, .5, .5, .5, .5]], np.float32), (64, 1))
    wo = np.tile(np.array([[0, 0, 1]], np.float32), (64, 1))
    d, p, t = S.sample_mis(env, brdf, wo, 4, 3)
    assert np.all(t == 2 * 16 + 5)
    L = d[:, 0::2]
    th = np.arccos(L[..., 2]); ph = np.arctan2(L[..., 1], L[..., 0])
    assert np.all((th >= 2 * PI / 8) & (th <= 3 * PI / 8))
    assert np.all((ph >= 2 * PI * 5 / 16 - PI) & (ph <= 2 * PI * 6 / 16 - PI))
    # stratified CDF inversion: texel frequencies follow the pmf (one sample per 1/spp stratum of the CDF)
    env = _env(3, (8, 16)); pmf, cdf = S.light_tables(env)
    spp = 256
    _, _, t = S.sample_mis(env, brdf, wo, spp, 9)
    cnt = np.bincount(t.ravel(), minlength=128).reshape(8, 16) / t.size
    assert np.abs(cnt - pmf).max() < 1.5 / spp
    for s in range(spp):                                               # sample s sits in stratum s of the CDF
        k = t[0, s]
        lo = cdf[k - 1] if k else 0.0
        assert lo <= (s + 1) / spp + 1e-6 and cdf[k] >= s / spp - 1e-6


# ---------------------------------------------------------------------------------------------- GGX VNDF (Q38)
@pytest.mark.parametrize("rough,vz", [(0.3, 0.9), (0.6, 0.3), (1.0, 0.7), (0.2, 0.05)])
def test_vndf_pdf_integrates_to_one(rough, vz):
    n = np.array([0.36, -0.48, 0.8])
    t = np.cross(n, [0, 0, 1.0]); t /= np.linalg.norm(t)
    wo = vz * n + np.sqrt(1 - vz * vz) * t
    d, w = _sphere_quadrature(1440, 1440)
    p = S.ggx_pdf(n, rough, wo, d)
    assert abs((p * w).sum() - 1) < 5e-3


def test_vndf_samples_follow_their_pdf_and_are_reflections():
    n = np.array([0.0, 0.6, 0.8]); wo = np.array([0.6, 0.0, 0.8]); rough = 0.5
    m = 400
    g = (np.arange(m) + 0.5) / m
    u = np.stack(np.meshgrid(g, g, indexing="ij"), -1).reshape(-1, 2)
    L = S.ggx_sample(n, rough, wo, u)
    np.testing.assert_allclose(np.linalg.norm(L, axis=1), 1, atol=1e-12)
    # empirical density over a coarse (theta, phi) grid about n vs the analytic pdf integrated over the same cells
    d, w = _sphere_quadrature(360, 720)
    p = S.ggx_pdf(n, rough, wo, d)
    def cell(x):
        th = np.arccos(np.clip(x[:, 2], -1, 1)); ph = np.arctan2(x[:, 1], x[:, 0])
        return (np.minimum((th / PI * 12).astype(int), 11)) * 12 + np.minimum(((ph + PI) / (2 * PI) * 12).astype(int), 11)
    emp = np.bincount(cell(L), minlength=144) / len(L)
    ana = np.bincount(cell(d), weights=p * w, minlength=144)
    assert np.abs(emp - ana).max() < 4e-3 and abs(ana.sum() - 1) < 5e-3
    # every sample is the reflection of wo about a half vector in the upper hemisphere, with positive pdf
    H = L + wo; H /= np.linalg.norm(H, axis=1, keepdims=True)
    assert np.all(H @ n > -1e-12) and np.all(S.ggx_pdf(n, rough, wo, L) > 0)
    # alpha -> small: samples collapse onto the mirror direction
    Lm = S.ggx_sample(n, 0.09, wo, u[::97])
    mirror = 2 * (wo @ n) * n - wo
    assert np.median(Lm @ mirror) > 0.9998 and np.quantile(Lm @ mirror, 0.05) > 0.997    # GGX tails are long, the bulk is tight


def _dvis_textbook(n, alpha, v, h):
    """Distribution of visible normals as Heitz (2014, 2018) defines it, written out in world space with numpy:
    D_vis(h) = G1(v) max(0, v.h) D(h) / (v.n),  D(h) = a^2 / (pi ((n.h)^2 (a^2 - 1) + 1)^2),
    G1(v) = 2 (n.v) / ((n.v) + sqrt(a^2 + (1 - a^2)(n.v)^2))."""
    nh = h @ n; nv = v @ n
    D = alpha ** 2 / (PI * (nh ** 2 * (alpha ** 2 - 1) + 1) ** 2) * (nh > 0)
    G1 = 2 * nv / (nv + np.sqrt(alpha ** 2 + (1 - alpha ** 2) * nv ** 2))
    return G1 * np.maximum(h @ v, 0) * D / nv


@pytest.mark.parametrize("rough,vz", [(0.5, 0.8), (0.8, 0.35)])
def test_vndf_against_rejection_sampling_of_the_textbook_density(rough, vz):
    """A check that shares nothing with the sampler's construction (the oracle stretches / projects / unstretches, Heitz 2018):
    (i) the oracle's pdf equals the closed form D_vis(h) / (4 v.h) written out independently in world space;
    (ii) half vectors drawn by REJECTION from D_vis (uniform-hemisphere proposals) and reflected give the same histogram of
    directions as the oracle's sampler -- a shared misreading of the density, the frame or the reflection cannot pass both."""
    rng = np.random.default_rng(7)
    n = np.array([0.36, -0.48, 0.8])
    t = np.cross(n, [0, 0, 1.0]); t /= np.linalg.norm(t); b = np.cross(n, t)
    v = vz * n + np.sqrt(1 - vz * vz) * (0.6 * t + 0.8 * b)
    alpha = rough * rough                                                  # PAPER.md:122 "alpha = Roughness^2"
    # (i) pdf of the reflected direction
    L = rng.standard_normal((4000, 3)); L /= np.linalg.norm(L, axis=1, keepdims=True)
    H = L + v; H /= np.linalg.norm(H, axis=1, keepdims=True)
    ref = _dvis_textbook(n, alpha, v, H) / (4 * np.maximum(H @ v, 1e-300))
    got = S.ggx_pdf(n, rough, v, L)
    ok = (H @ n > 1e-6)
    np.testing.assert_allclose(got[ok], ref[ok], rtol=1e-9, atol=1e-12)
    # (ii) rejection sampling of h ~ D_vis, proposal uniform on the hemisphere about n (density 1 / 2 pi)
    M = 2 * PI * alpha ** 2 / (PI * alpha ** 4) / vz * 1.02                # 2 pi max D_vis: D <= 1/(pi a^2), G1 (v.h) <= 1
    keep = []
    while sum(len(k) for k in keep) < 120000:
        z = rng.random(2_000_000); ph = 2 * PI * rng.random(2_000_000)
        r = np.sqrt(1 - z * z)
        h = r[:, None] * np.cos(ph)[:, None] * t + r[:, None] * np.sin(ph)[:, None] * b + z[:, None] * n
        f = 2 * PI * _dvis_textbook(n, alpha, v, h)
        assert f.max() <= M
        keep.append(h[rng.random(len(h)) * M < f])
    h = np.concatenate(keep)
    Lr = 2 * (h @ v)[:, None] * h - v                                      # reflect the view direction about h
    m = 350
    g = (np.arange(m) + 0.5) / m
    u = np.stack(np.meshgrid(g, g, indexing="ij"), -1).reshape(-1, 2)
    Lo = S.ggx_sample(n, rough, v, u)

    def cell(x):
        th = np.arccos(np.clip(x @ n, -1, 1)); ph = np.arctan2(x @ b, x @ t)
        return (np.minimum((th / PI * 10).astype(int), 9)) * 10 + np.minimum(((ph + PI) / (2 * PI) * 10).astype(int), 9)
    e1 = np.bincount(cell(Lr), minlength=100) / len(Lr)
    e2 = np.bincount(cell(Lo), minlength=100) / len(Lo)
    assert np.abs(e1 - e2).max() < 6e-3, np.abs(e1 - e2).max()
    assert e1.max() > 0.05                                                 # the histogram has structure to compare


# ---------------------------------------------------------------------------------------------- stratified sets
def test_stratified_hemisphere_and_sphere():
    rng = np.random.default_rng(4)
    nrm = rng.standard_normal((50, 3)); nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
    nrm = nrm.astype(np.float32)
    Sa, Sb = 8, 8
    d, p = S.sample_stratified(nrm, 50, Sa, Sb, 21)
    n64 = nrm.astype(np.float64); n64 /= np.linalg.norm(n64, axis=1, keepdims=True)
    cos = np.einsum("rsk,rk->rs", d, n64)
    np.testing.assert_allclose(np.linalg.norm(d, axis=-1), 1, atol=1e-6)
    assert np.all(cos > 0)
    np.testing.assert_allclose(p, cos / PI, atol=1e-6)
    a = np.floor((1 - cos ** 2) * Sa).astype(int)                       # u = 1 - z^2 falls in stratum a = slot // Sb
    assert np.array_equal(a, np.tile(np.repeat(np.arange(Sa), Sb), (50, 1)))
    # the azimuthal strata: Sb distinct phi-cells per ring (frame-independent statement: pairwise distinct within a ring)
    # cosine-weighted: E[1/pdf * cos] = pi * E[...]: MC estimate of the hemisphere integral of cos is pi
    assert abs(np.mean(cos / p) - PI) < 1e-6
    d, p = S.sample_stratified(None, 30, 4, 2, 5)
    np.testing.assert_allclose(p, 1 / (4 * PI))
    assert np.array_equal(np.floor((1 - d[..., 2]) / 2 * 4).astype(int), np.tile(np.repeat(np.arange(4), 2), (30, 1)))
    phi = np.arctan2(d[..., 1], d[..., 0]) % (2 * PI)
    assert np.array_equal(np.floor(phi / (2 * PI) * 2).astype(int), np.tile(np.tile(np.arange(2), 4), (30, 1)))
    assert np.abs(d.reshape(-1, 3).mean(0)).max() < 0.08


# ---------------------------------------------------------------------------------------------- the MIS estimator
def test_balance_heuristic_estimator_reproduces_known_integrals():
    """(1 / 2spp) sum f / ((p_light + p_ggx) / 2) over the 2 spp rays is unbiased: constant env L, Lambert a -> a * L;
    a lognormal env -> the quadrature of the same integrand."""
    n = np.array([0.3, 0.2, 0.0]); n[2] = np.sqrt(1 - n @ n)
    wo = np.array([0.0, 0.5, np.sqrt(0.75)])
    N, spp = 4000, 8
    brdf = np.tile(np.concatenate([n, [.5, .5, .5], [0.4]]).astype(np.float32)[None], (N, 1))
    wo32 = np.tile(wo.astype(np.float32)[None], (N, 1))
    n32 = brdf[0, :3].astype(np.float64)
    # constant environment
    env = np.full((8, 16, 3), 2.5, np.float32)
    d, p, _ = S.sample_mis(env, brdf, wo32, spp, 12)
    cos = np.maximum(d @ n32, 0)
    est = (2.5 * (0.5 / PI) * cos / p).mean()
    assert abs(est - 0.5 * 2.5) < 0.01
    # lognormal environment, piecewise-constant radiance per texel (nearest texel, the sampler's own grid)
    env = _env(6, (8, 16))
    d, p, _ = S.sample_mis(env, brdf, wo32, spp, 13)
    def radiance(x):
        th = np.arccos(np.clip(x[..., 2], -1, 1)); ph = np.arctan2(x[..., 1], x[..., 0])
        r = np.minimum((th / PI * 8).astype(int), 7); c = np.minimum(((ph / (2 * PI) + 0.5) * 16).astype(int), 15)
        return env[r, c, 1].astype(np.float64)
    est = (radiance(d) * (0.5 / PI) * np.maximum(d @ n32, 0) / p).mean()
    dq, wq = _sphere_quadrature(720, 1440)
    ref = (radiance(dq) * (0.5 / PI) * np.maximum(dq @ n32, 0) * wq).sum()
    assert abs(est - ref) < 0.02 * ref
    # the two strategies alone, weighted by the same balance heuristic, split the integral: neither is dropped
    light = (radiance(d[:, 0::2]) * (0.5 / PI) * np.maximum(d[:, 0::2] @ n32, 0) / p[:, 0::2]).mean() / 2
    ggx = (radiance(d[:, 1::2]) * (0.5 / PI) * np.maximum(d[:, 1::2] @ n32, 0) / p[:, 1::2]).mean() / 2
    assert light > 0.2 * ref and ggx > 0.02 * ref and abs(light + ggx - est) < 1e-9

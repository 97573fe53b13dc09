"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only, `-m "not gpu"`).

Each test names the SURVEY.md 8(c) pin row it implements.  None of them compares the oracle with itself:
they use closed forms, invariants, library routines (float64 numpy matmul), quadrature, brute force
and an independent literal-recursive numpy re-statement of the whole path.
"""
import math
import os

import numpy as np
import pytest

import gen
from oracle.oracle import Oracle, lib

GOLD = os.path.join(os.path.dirname(__file__), "golden")
PI = math.pi


def blob(*layers):
    return np.concatenate([np.asarray(a, dtype=np.float32).ravel() for a in layers])


def tiny_oracle(L=2, F=2, log2_T=14, res=(4, 8), tables=None, brdf_w=None, irt_w=None, env=None, hidden=4, **kw):
    D = L * F
    T = 1 << log2_T
    if tables is None:
        tables = np.random.default_rng(1).uniform(-1, 1, (L, T, F))
    z = lambda o, i: np.zeros((o, i), np.float32)
    if brdf_w is None:
        brdf_w = blob(z(hidden, D), np.zeros(hidden), z(hidden, hidden), np.zeros(hidden), z(7, hidden), np.zeros(7))
    if irt_w is None:
        irt_w = blob(z(hidden, D + 3), np.zeros(hidden), z(hidden, hidden), np.zeros(hidden), z(2, hidden), np.zeros(2))
    return Oracle(L=L, F=F, log2_T=log2_T, res=np.array(res, np.uint32), tables=tables, brdf_w=brdf_w, irt_w=irt_w,
                  env=env, hidden=hidden, **kw)


# ------------------------------------------------------------------------------------------------ resolutions
def test_resolutions_closed_form():
    """pin 'resolutions': PAPER.md:120 config => growth exactly 2; BASELINE lists."""
    for line in open(os.path.join(GOLD, "resolutions.txt")):
        if line.startswith("#") or not line.strip():
            continue
        head, vals = line.split(":")
        L, lo, hi = map(int, head.split())
        assert gen.resolutions(L, lo, hi).tolist() == list(map(int, vals.split()))


# ------------------------------------------------------------------------------------------------ hash index
def test_hash_known_answers():
    """pin 'hash index': closed-form known answers of the [14] hash (tests/golden/hash_known_answers.txt)."""
    l = lib()
    n = 0
    for line in open(os.path.join(GOLD, "hash_known_answers.txt")):
        if line.startswith("#") or not line.strip():
            continue
        cx, cy, cz, h14, h17, h19 = map(int, line.split())
        assert l.or_hash_index(cx, cy, cz, 14) == h14
        assert l.or_hash_index(cx, cy, cz, 17) == h17
        assert l.or_hash_index(cx, cy, cz, 19) == h19
        n += 1
    assert n == 6
    for T in (14, 17, 19):
        assert l.or_hash_index(0, 0, 0, T) == 0
        for i in (1, 5, 1000, (1 << T) + 3):
            assert l.or_hash_index(i, 0, 0, T) == i % (1 << T)        # prime for x is 1


def test_dense_index_bijection_and_hash_range():
    """pin 'hash index' invariants: dense index is a bijection onto [0,(N+1)^3); hashed index < T."""
    l = lib()
    for Nl, log2_T in ((16, 14), (23, 14)):
        assert l.or_level_is_dense(Nl, log2_T) == 1
        seen = set()
        for cz in range(Nl + 1):
            for cy in range(Nl + 1):
                for cx in range(Nl + 1):
                    seen.add(l.or_grid_index(cx, cy, cz, Nl, log2_T))
        assert seen == set(range((Nl + 1) ** 3))
    assert l.or_level_is_dense(35, 14) == 0 and l.or_level_is_dense(25, 14) == 0     # 26^3 > 2^14
    assert l.or_level_is_dense(58, 19) == 1 and l.or_level_is_dense(80, 19) == 0     # T=2^19 levels 0-4 dense
    rng = np.random.default_rng(0)
    for c in rng.integers(0, 2049, (200, 3)):
        assert l.or_grid_index(int(c[0]), int(c[1]), int(c[2]), 2048, 19) < (1 << 19)


# ------------------------------------------------------------------------------------------------ corners
def test_corner_selection_brute_force():
    """pin 'corner selection': the 8 corners are exactly the vertices of the cell containing x."""
    res = (16, 23)
    o = tiny_oracle(res=res)
    rng = np.random.default_rng(3)
    x = rng.random((300, 3)).astype(np.float32)
    x[:6] = [[0, 0, 0], [1, 1, 1], [0.5, 0.25, 0.125], [1, 0, 0.5], [3 / 16, 5 / 16, 1.0], [1e-8, 1 - 1e-7, 0.999999]]
    _, idx, w = o.encode(x)
    for li, Nl in enumerate(res):
        grid = np.arange(Nl + 1, dtype=np.float64) / Nl                  # vertex positions i/N_l (reading Q4)
        for p in range(x.shape[0]):
            # brute-force search for the cell in double precision
            c0 = []
            for d in range(3):
                xv = float(x[p, d])
                cands = [i for i in range(Nl) if grid[i] <= xv <= grid[i + 1]]
                assert cands, (xv, Nl)
                c0.append(cands)
            got = idx[p, li]
            # decode dense index of corner 0 and check it is one of the admissible cells; other corners = +1 offsets
            s = Nl + 1
            cx, cy, cz = got[0] % s, (got[0] // s) % s, got[0] // (s * s)
            assert cx in c0[0] and cy in c0[1] and cz in c0[2]
            for corner in range(8):
                b = (corner & 1, (corner >> 1) & 1, (corner >> 2) & 1)
                assert got[corner] == (cx + b[0]) + (cy + b[1]) * s + (cz + b[2]) * s * s
            assert np.all(w[p, li] >= 0) and np.all(w[p, li] <= 1)
            # the fp32 index path p = fl32(x * N) is within one fp32 rounding of x*N
            np.testing.assert_allclose((np.array([cx, cy, cz]) + w[p, li].astype(np.float64)) / Nl, x[p].astype(np.float64),
                                       atol=2e-7)
    # x = 1 upper boundary (Q7): c0 = N-1, w = 1
    assert np.all(w[1] == 1.0)
    # out-of-range positions are clamped (Q6)
    _, idx2, w2 = o.encode(np.array([[-0.5, 2.0, 0.3]], np.float32))
    _, idx3, w3 = o.encode(np.array([[0.0, 1.0, 0.3]], np.float32))
    assert np.array_equal(idx2, idx3) and np.array_equal(w2, w3)


# ------------------------------------------------------------------------------------------------ trilinear
def test_vertex_reproduction_bit_exact():
    """pin 'trilinear (i)': at a grid vertex the feature equals that vertex's table row bit-exactly."""
    cfg = gen.make_config("C0")
    m = gen.make_model(cfg)
    o = Oracle.from_gen(cfg, m)
    l = lib()
    rng = np.random.default_rng(5)
    for li in (0, 1, 4, 7):             # dense and hashed levels; N_l = 16, 23, 78, 256
        Nl = int(m["res"][li])
        for _ in range(50):
            c = rng.integers(0, Nl + 1, 3)
            # a vertex i/N_l reproduces exactly when fl32(fl32(i/N)*N) == i; pick only those (true for most)
            x = (c / Nl).astype(np.float32)
            if not np.all((x * np.float32(Nl)).astype(np.float32) == c.astype(np.float32)):
                continue
            feat, idx, w = o.encode(x[None])
            row = l.or_grid_index(int(c[0]), int(c[1]), int(c[2]), Nl, cfg.log2_T)
            expect = m["tables"][li, row].astype(np.float64)
            assert np.array_equal(feat[0, li * cfg.F:(li + 1) * cfg.F], expect)


def test_partition_of_unity_and_affine_reproduction():
    """pins 'trilinear (ii)-(iv)': constant table => constant; affine table on dense levels => affine output."""
    res = (4, 9)
    L, F, log2_T = 2, 2, 14
    T = 1 << log2_T
    rng = np.random.default_rng(7)
    x = rng.random((500, 3)).astype(np.float32)
    o = tiny_oracle(L=L, F=F, log2_T=log2_T, res=res, tables=np.full((L, T, F), 0.625))
    feat, _, _ = o.encode(x)
    np.testing.assert_allclose(feat, 0.625, rtol=0, atol=1e-15)          # weights sum to 1 (double round-off only)
    # affine: tab[l][dense(c)][j] = g_j . (c/N_l) + h_j  (values kept in fp32 => compare against the fp32-rounded table)
    g = np.array([[0.5, -0.25, 0.125], [1.0, 2.0, -3.0]])
    h = np.array([0.75, -0.5])
    tables = np.zeros((L, T, F), np.float32)
    for li, Nl in enumerate(res):
        s = Nl + 1
        cz, cy, cx = np.meshgrid(np.arange(s), np.arange(s), np.arange(s), indexing="ij")
        pos = np.stack([cx, cy, cz], -1).reshape(-1, 3) / Nl
        tables[li, :s ** 3] = (pos @ g.T + h)
    o = tiny_oracle(L=L, F=F, log2_T=log2_T, res=res, tables=tables)
    feat, idx, w = o.encode(x)
    expect = x.astype(np.float64) @ g.T + h
    for li in range(L):
        np.testing.assert_allclose(feat[:, li * F:(li + 1) * F], expect, atol=3e-6)   # fp32 table + fp32 index-path rounding


def test_encode_continuity_across_cell_faces(c0):
    """pin 'trilinear (v)': encode(x-eps) and encode(x+eps) across a cell face differ by O(eps)."""
    cfg, m, fr, o = c0
    Nl = 16
    x0 = np.array([5 / Nl, 0.3371, 0.7113])
    eps = 1e-6
    fa, _, _ = o.encode(np.array([x0 - [eps, 0, 0]], np.float32))
    fb, _, _ = o.encode(np.array([x0 + [eps, 0, 0]], np.float32))
    # slope bound: |df/dx| <= N_l * 2 * max|tab| per level
    bound = 2 * eps * m["res"].astype(np.float64).repeat(cfg.F) * 2 * 1.0 + 1e-6
    assert np.all(np.abs(fa - fb)[0] <= bound)


# ------------------------------------------------------------------------------------------------ MLPs
def test_mlp_equals_float64_matmul(c0):
    """pin 'MLPs': a linear layer is a GEMM => compare with float64 numpy matmul + maximum."""
    cfg, m, fr, o = c0
    rng = np.random.default_rng(11)
    for which, d_in, d_out in (("brdf", cfg.D, 7), ("irt", cfg.D + 3, 2)):
        inp = rng.standard_normal((64, d_in))
        (W1, b1), (W2, b2), (W3, b3) = [(W.astype(np.float64), b.astype(np.float64)) for W, b in
                                        gen.split_mlp(cfg, which, m[which + "_w"])]
        ref = np.maximum(np.maximum(inp @ W1.T + b1, 0) @ W2.T + b2, 0) @ W3.T + b3
        got = o.mlp3(m[which + "_w"], d_in, d_out, inp)
        np.testing.assert_allclose(got, ref, rtol=1e-12, atol=1e-13)


def test_mlp_special_cases():
    """pin 'MLPs': zero weights => bias path; identity-padded weights pass (non-negative) features through."""
    h, d_in, d_out = 4, 3, 2
    o = tiny_oracle(hidden=h)
    z = np.zeros
    b3 = np.array([0.25, -1.5])
    out = o.mlp3(blob(z((h, d_in)), z(h), z((h, h)), z(h), z((d_out, h)), b3), d_in, d_out, np.ones((2, d_in)))
    np.testing.assert_array_equal(out, np.tile(b3, (2, 1)))
    # relu(bias) propagates: W1=0,b1=[1,-1,2,-2] -> h1=[1,0,2,0]; W2=I -> h2=h1; W3 = [[1,1,1,1],[0,0,1,0]]
    out = o.mlp3(blob(z((h, d_in)), [1, -1, 2, -2], np.eye(h), z(h), [[1, 1, 1, 1], [0, 0, 1, 0]], z(d_out)), d_in, d_out,
                 np.ones((1, d_in)))
    np.testing.assert_array_equal(out, [[3.0, 2.0]])
    # identity padding: h1 = relu(in) for the first 3 rows; W2 = I; W3 picks rows 0 and 2 -> transposition would fail
    W1 = np.zeros((h, d_in)); W1[0, 0] = W1[1, 1] = W1[2, 2] = 1
    inp = np.array([[0.5, -0.25, 2.0]])
    out = o.mlp3(blob(W1, z(h), np.eye(h), z(h), [[1, 0, 0, 0], [0, 0, 1, 0]], z(d_out)), d_in, d_out, inp)
    np.testing.assert_array_equal(out, [[0.5, 2.0]])
    W1 = np.zeros((h, d_in)); W1[3, 1] = -1            # asymmetric: only a [out][in] layout gives 0.25
    out = o.mlp3(blob(W1, z(h), np.eye(h), z(h), [[0, 0, 0, 1], [0, 0, 0, 0]], z(d_out)), d_in, d_out, inp)
    np.testing.assert_array_equal(out, [[0.25, 0.0]])


def test_output_maps(c0):
    """pin 'output maps': ||n||=1, a in (0,1), r in [0.09,1], r(0)=0.545; t in [near,far]."""
    cfg, m, fr, o = c0
    feat, _, _ = o.encode(fr["x"][:256])
    brdf = o.decode(feat)
    np.testing.assert_allclose(np.linalg.norm(brdf[:, :3], axis=1), 1.0, atol=1e-12)
    assert np.all((brdf[:, 3:6] > 0) & (brdf[:, 3:6] < 1))
    assert np.all((brdf[:, 6] >= 0.09) & (brdf[:, 6] <= 1.0))
    vis, zv, t, xs = o.trace(fr["x"][:256], feat, fr["dir_d"][:256])
    assert np.all((t >= cfg.near_t) & (t <= cfg.far_t))
    np.testing.assert_allclose(vis, 1 / (1 + np.exp(-zv)), rtol=1e-14)
    # zero network: sigma(0) = 1/2 everywhere, r(0) = 0.09 + 0.91/2 = 0.545, albedo 0.5
    oz = tiny_oracle()
    bz = oz.decode(np.zeros((1, 4)))
    assert bz[0, 6] == pytest.approx(0.545, abs=1e-7) and np.allclose(bz[0, 3:6], 0.5)
    v, z, t, _ = oz.trace(np.zeros((1, 3), np.float32), np.zeros((1, 4)), np.array([[[0, 0, 1.0]]]))
    assert v[0, 0] == 0.5 and t[0, 0] == pytest.approx(0.05 + math.log(2.0) * 1.45, abs=1e-7)   # softplus(0) = ln 2
    # z_t -> +inf => d clamps at 1 => t = far ("clamp all outputs to 1 (corresponding to far)")
    big = blob(np.zeros((4, 7)), np.zeros(4), np.zeros((4, 4)), np.zeros(4), np.zeros((2, 4)), [0.0, 50.0])
    ob = tiny_oracle(irt_w=big)
    _, _, t, _ = ob.trace(np.zeros((1, 3), np.float32), np.zeros((1, 4)), np.array([[[0, 0, 1.0]]]))
    assert t[0, 0] == pytest.approx(1.5, abs=1e-7)
    # hard mode: v = [z_v > 0], tie -> occluded (Q14)
    ob.set_modes(vis_mode=1)
    v, _, _, _ = ob.trace(np.zeros((1, 3), np.float32), np.zeros((1, 4)), np.array([[[0, 0, 1.0]]]))
    assert v[0, 0] == 0.0


# ------------------------------------------------------------------------------------------------ trace
def test_trace_secondary_hit():
    """pin 'trace': t=0 => x'=x; axis-aligned omega moves one coordinate only; clamp to [0,1]."""
    neg = blob(np.zeros((4, 7)), np.zeros(4), np.zeros((4, 4)), np.zeros(4), np.zeros((2, 4)), [0.0, -800.0])
    o = tiny_oracle(irt_w=neg, near_t=0.0, far_t=1.0)              # softplus(-800) = 0 => t = near = 0
    x = np.array([[0.3, 0.6, 0.9]], np.float32)
    _, _, t, xs = o.trace(x, np.zeros((1, 4)), np.array([[[0.6, 0.0, 0.8]]]))
    assert t[0, 0] == 0.0 and np.array_equal(xs[0, 0], x[0])
    o = tiny_oracle()                                              # zero net: t = 0.05 + ln2*1.45 = 1.0551
    tt = 0.05 + math.log(2.0) * 1.45
    _, _, t, xs = o.trace(x, np.zeros((1, 4)), np.array([[[0, -1.0, 0], [0, 0, 1.0], [-0.25, 0, 0]]]))
    assert np.array_equal(xs[0, 0], np.array([0.3, 0.0, 0.9], np.float32))          # 0.6 - 1.055 clamps to 0
    assert np.array_equal(xs[0, 1], np.array([0.3, 0.6, 1.0], np.float32))          # clamps to 1
    np.testing.assert_allclose(xs[0, 2], [np.float32(0.3) - 0.25 * tt, 0.6, 0.9], atol=1e-7)
    assert xs[0, 2, 1] == np.float32(0.6) and xs[0, 2, 2] == np.float32(0.9)


# ------------------------------------------------------------------------------------------------ env lookup
def test_env_lookup():
    """pin 'env lookup': constant map; texel-centre exactness; continuity across phi=+-pi; linear-in-row map."""
    rng = np.random.default_rng(13)
    He, We = 8, 16
    d = rng.standard_normal((200, 3)); d /= np.linalg.norm(d, axis=1, keepdims=True)
    o = tiny_oracle(env=np.full((He, We, 3), 2.5))
    np.testing.assert_allclose(o.env_lookup(d), 2.5, atol=1e-14)
    env = rng.random((He, We, 3)).astype(np.float32)
    o = tiny_oracle(env=env)
    for (r, c) in ((0, 0), (3, 5), (7, 15), (4, 8)):
        th = (r + 0.5) / He * PI
        ph = ((c + 0.5) / We - 0.5) * 2 * PI
        w = [math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)]
        np.testing.assert_allclose(o.env_lookup([w])[0], env[r, c].astype(np.float64), atol=1e-12)
    # halfway between two texel centres in u: average of the two texels
    th = (3 + 0.5) / He * PI; ph = ((5 + 1.0) / We - 0.5) * 2 * PI
    w = [math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)]
    np.testing.assert_allclose(o.env_lookup([w])[0], 0.5 * (env[3, 5].astype(np.float64) + env[3, 6]), atol=1e-12)
    # wrap: phi = pi - eps and -pi + eps give (nearly) the same colour = average of columns We-1 and 0
    e = 1e-9
    a = o.env_lookup([[-math.cos(e), math.sin(e), 0.3], [-math.cos(e), -math.sin(e), 0.3]])
    np.testing.assert_allclose(a[0], a[1], atol=1e-7)
    # rows vary linearly with the row index => lookup reproduces theta/pi*He - 1/2 away from the poles
    env = np.repeat(np.arange(He, dtype=np.float32)[:, None, None], We, 1).repeat(3, 2)
    o = tiny_oracle(env=env)
    dd = d[np.abs(np.arccos(d[:, 2]) / PI - 0.5) < 0.4]
    np.testing.assert_allclose(o.env_lookup(dd)[:, 0], np.arccos(dd[:, 2]) / PI * He - 0.5, atol=1e-12)
    # poles clamp (Q25): theta=0 -> row 0
    np.testing.assert_allclose(o.env_lookup([[0, 0, 1.0]])[0], 0.0, atol=1e-12)


# ------------------------------------------------------------------------------------------------ BRDF
def _brdf7(n, a, r):
    return np.array(list(n) + list(a) + [r], dtype=np.float64)


def test_brdf_lambert_reciprocity_fresnel():
    """pin 'BRDF': Lambert closed form a/pi; reciprocity; F(VoH=1)=F0=0.04; finite at grazing."""
    o = tiny_oracle(brdf_model=0)
    n = [0, 0, 1.0]
    b = _brdf7(n, [0.2, 0.5, 0.8], 0.3)
    wi = np.array([0.6, 0.0, 0.8]); wo = np.array([0.0, -0.6, 0.8])
    np.testing.assert_allclose(o.brdf_eval(b, wi, wo), np.array([0.2, 0.5, 0.8]) / PI, rtol=1e-14)
    assert np.all(o.brdf_eval(b, [0.6, 0, -0.8], wo) == 0)               # NoL <= 0 => 0 (Q22)
    o = tiny_oracle(brdf_model=1)
    rng = np.random.default_rng(17)
    for _ in range(50):
        wi = rng.standard_normal(3); wi[2] = abs(wi[2]) + 0.05; wi /= np.linalg.norm(wi)
        wo = rng.standard_normal(3); wo[2] = abs(wo[2]) + 0.05; wo /= np.linalg.norm(wo)
        b = _brdf7(n, rng.random(3), 0.09 + 0.91 * rng.random())
        np.testing.assert_allclose(o.brdf_eval(b, wi, wo), o.brdf_eval(b, wo, wi), rtol=1e-12)
    # wi = wo = n: NoL=NoV=NoH=VoH=1 => D = 1/(pi k), F = F0, Gv = 0.5/(2) => spec = F0/(4 pi k), k = r^4
    r = 0.5
    b = _brdf7(n, [0, 0, 0], r)
    F0 = float(np.float32(0.04))                 # the config carries F0 as fp32
    np.testing.assert_allclose(o.brdf_eval(b, n, n), F0 / (4 * PI * r ** 4), rtol=1e-12)
    # k = 1 (r = 1): D = 1/pi, Gv = 0.5/(NoL+NoV) (textbook height-correlated Smith at alpha = 1)
    b = _brdf7(n, [0, 0, 0], 1.0)
    wi = np.array([0.6, 0, 0.8]); wo = np.array([-0.28, 0, 0.96])
    hvec = (wi + wo) / np.linalg.norm(wi + wo)
    F = F0 + (1 - F0) * (1 - wo @ hvec) ** 5
    np.testing.assert_allclose(o.brdf_eval(b, wi, wo), (1 / PI) * F * 0.5 / (0.8 + 0.96), rtol=1e-12)
    # grazing stays finite
    g = o.brdf_eval(_brdf7(n, [0.5] * 3, 0.2), [math.sqrt(1 - 1e-12), 0, 1e-6], wo)
    assert np.all(np.isfinite(g))


def test_ggx_normalisation_quadrature():
    """pin 'BRDF': int D(h) (n.h) dw_h = 1 by quadrature, D isolated through wi = wo = h with F0 = 1.

    With wi = wo = h: VoH = 1 => F = F0 = 1, NoL = NoV = NoH = c, Gv = 0.5 / (2 c sqrt(c^2 (1-k) + k)) in closed form.
    """
    o = tiny_oracle(brdf_model=1, fresnel_f0=1.0)
    for r in (0.3, 0.6, 1.0):
        k = r ** 4
        nth = 4000
        th = (np.arange(nth) + 0.5) / nth * (PI / 2)
        tot = 0.0
        for t in th:
            c = math.cos(t)
            hvec = [math.sin(t), 0, c]
            spec = o.brdf_eval(_brdf7([0, 0, 1.0], [0, 0, 0], r), hvec, hvec)[0]
            Gv = 0.5 / (2 * c * math.sqrt(c * c * (1 - k) + k))
            D = spec / Gv
            tot += D * c * math.sin(t) * 2 * PI * (PI / 2 / nth)
        assert tot == pytest.approx(1.0, abs=2e-3)


# ------------------------------------------------------------------------------------------------ rendering sum
def _const_brdf_blob(h, D, n, a_logit, r_logit=0.0):
    return blob(np.zeros((h, D)), np.zeros(h), np.zeros((h, h)), np.zeros(h), np.zeros((7, h)),
                list(n) + [a_logit] * 3 + [r_logit])


def _cos_dirs(n, S, rng):
    """S cosine-weighted directions about unit n with pdf = cos/pi (test-local sampler)."""
    u1, u2 = rng.random(S), rng.random(S)
    r, ph = np.sqrt(u1), 2 * PI * u2
    lz = np.sqrt(1 - u1)
    n = np.asarray(n, float)
    t = np.cross(n, [1, 0, 0] if abs(n[0]) < 0.9 else [0, 1, 0]); t /= np.linalg.norm(t)
    b = np.cross(n, t)
    d = (r * np.cos(ph))[:, None] * t + (r * np.sin(ph))[:, None] * b + lz[:, None] * n
    d = d.astype(np.float32)
    pdf = (d.astype(np.float64) @ n / PI).astype(np.float32)       # pdf consistent with the fp32-rounded direction
    return d, pdf


def test_closed_form_albedo_times_L():
    """pin 'rendering sum' closed form 1: Lambert, v==1, constant env L, cosine pdf => every term is a*L (Eq. 1)."""
    rng = np.random.default_rng(19)
    Lc = 1.75
    o = tiny_oracle(env=np.full((4, 8, 3), Lc), brdf_model=0)
    n = np.array([0.36, -0.48, 0.8])
    a = np.array([0.2, 0.55, 0.9])
    for S in (1, 7, 64):
        d, pdf = _cos_dirs(n, S, rng)
        brdf = np.array([list(n) + list(a) + [0.5]], np.float32)
        r = o.render_frame(np.array([[0.4, 0.5, 0.6]], np.float32), np.array([[0, 0, 1.0]], np.float32), (d[None], pdf[None]),
                           flags=1, brdf=brdf)                       # no SHADOW flag => v == 1
        np.testing.assert_allclose(r["rgb"][0], a.astype(np.float32).astype(np.float64) * Lc, rtol=2e-6)


def test_indirect_vanishes_when_visible_and_closed_form_a_a_L():
    """pins 'rendering sum' closed forms 2 and 3 (Eq. 2).

    z_v = -K * omega_z through a hand-built I (hard mode): directions with omega_z > 0 are occluded, omega_z < 0 visible.
    Primary normal +z with cosine secondary set (all occluded), secondary normal -z (from B's bias) with a cosine
    tertiary set about -z (all visible) => pixel = a * a' * L for any S.  Flipping K's sign makes every secondary
    direction visible => the indirect term is exactly 0.
    """
    rng = np.random.default_rng(23)
    h, L, F = 4, 2, 2
    D = L * F
    Lc = 0.8
    a = np.array([0.3, 0.6, 0.9], np.float32)
    a2_logit = 0.4
    a2 = 1 / (1 + math.exp(-a2_logit))

    def irt(K):
        W1 = np.zeros((h, D + 3)); W1[0, D + 2] = 1.0; W1[1, D + 2] = -1.0        # h = relu(+-omega_z)
        W3 = np.zeros((2, h)); W3[0, 0] = -K; W3[0, 1] = K                         # z_v = -K omega_z
        return blob(W1, np.zeros(h), np.eye(h), np.zeros(h), W3, [0.0, -1.0])
    for S_i, S_2 in ((1, 1), (16, 8), (5, 3)):
        ds, ps = _cos_dirs([0, 0, 1.0], S_i, rng)
        dt, pt = _cos_dirs([0, 0, -1.0], S_2, rng)
        x = np.array([[0.5, 0.5, 0.2]], np.float32)
        brdf = np.array([[0, 0, 1.0, *a, 0.5]], np.float32)
        wo = np.array([[0, 0.6, 0.8]], np.float32)
        common = dict(L=L, F=F, res=(4, 8), hidden=h, env=np.full((4, 8, 3), Lc), brdf_model=0, vis_mode=1,
                      brdf_w=_const_brdf_blob(h, D, [0, 0, -2.0], a2_logit))
        o = tiny_oracle(irt_w=irt(1e4), **common)
        r = o.render_frame(x, wo, (ds[None], ps[None]), (ds[None], ps[None]), (dt, pt), flags=7, brdf=brdf)
        # direct term: all occluded => 0; indirect: a * a' * L
        np.testing.assert_allclose(r["rgb"][0], a.astype(np.float64) * a2 * Lc, rtol=3e-6)
        o = tiny_oracle(irt_w=irt(-1e4), **common)
        r2 = o.render_frame(x, wo, (ds[None], ps[None]), (ds[None], ps[None]), (dt, pt), flags=7, brdf=brdf)
        r1 = o.render_frame(x, wo, (ds[None], ps[None]), flags=3, brdf=brdf)
        assert np.array_equal(r2["rgb"], r1["rgb"])                               # V == 1 => indirect == 0 exactly
        np.testing.assert_allclose(r1["rgb"][0], a.astype(np.float64) * Lc, rtol=3e-6)


def test_linearity_in_env_and_permutation_invariance(c0):
    """pin 'rendering sum': linear in the env map; invariant under permuting the direction set."""
    cfg, m, fr, o = c0
    sl = slice(100, 132)
    args = (fr["x"][sl], fr["wo"][sl])
    r1 = o.render_frame(*args, (fr["dir_d"][sl], fr["pdf_d"][sl]))["rgb"]
    o2 = Oracle.from_gen(cfg, {**m, "env": (m["env"] * np.float32(2.0))})
    r2 = o2.render_frame(*args, (fr["dir_d"][sl], fr["pdf_d"][sl]))["rgb"]
    np.testing.assert_allclose(r2, 2 * r1, rtol=1e-12)
    perm = np.random.default_rng(29).permutation(cfg.S_d)
    r3 = o.render_frame(*args, (fr["dir_d"][sl][:, perm], fr["pdf_d"][sl][:, perm]))["rgb"]
    np.testing.assert_allclose(r3, r1, rtol=1e-12)


def test_mask_and_flags(c0):
    cfg, m, fr, o = c0
    sl = slice(0, 8)
    mask = np.array([1, 0, 1, 1, 0, 1, 1, 1], np.uint8)
    r = o.render_frame(fr["x"][sl], fr["wo"][sl], (fr["dir_d"][sl], fr["pdf_d"][sl]), mask=mask)["rgb"]
    r0 = o.render_frame(fr["x"][sl], fr["wo"][sl], (fr["dir_d"][sl], fr["pdf_d"][sl]))["rgb"]
    assert np.all(r[mask == 0] == 0) and np.array_equal(r[mask == 1], r0[mask == 1])


# ------------------------------------------------------------------------------------------------ whole frame
def _naive_frame(cfg, m, x, wo, dd, pd, dsec, psec, dt, pt, vis_mode, flags):
    """Independent literal re-statement in numpy float64: re-encodes per direction, un-factored layer 1,
    recursion written as a recursive function.  Shares no code with oracle/ (pin 'whole frame')."""
    res, tab, env = m["res"], m["tables"].astype(np.float64), m["env"].astype(np.float64)
    T = cfg.T
    f32 = lambda v: float(np.float32(v))                      # the config carries these scalars as fp32
    near_t, far_t, rough_min, f0 = f32(cfg.near_t), f32(cfg.far_t), f32(cfg.rough_min), f32(cfg.fresnel_f0)

    def H(p):
        p = np.clip(np.asarray(p, np.float32), np.float32(0), np.float32(1))
        out = []
        for l in range(cfg.L):
            N = int(res[l])
            q = (p * np.float32(N)).astype(np.float32)
            c0 = np.minimum(np.floor(q).astype(np.int64), N - 1)
            w = (q - c0.astype(np.float32)).astype(np.float64)
            acc = np.zeros(cfg.F)
            for bz in (0, 1):
                for by in (0, 1):
                    for bx in (0, 1):
                        c = c0 + [bx, by, bz]
                        if (N + 1) ** 3 <= T:
                            i = int(c[0] + c[1] * (N + 1) + c[2] * (N + 1) ** 2)
                        else:
                            i = int(((int(c[0]) * 1) ^ ((int(c[1]) * 2654435761) & 0xFFFFFFFF) ^ ((int(c[2]) * 805459861) & 0xFFFFFFFF)) % T)
                        wt = (w[0] if bx else 1 - w[0]) * (w[1] if by else 1 - w[1]) * (w[2] if bz else 1 - w[2])
                        acc += wt * tab[l, i]
            out.append(acc)
        return np.concatenate(out)

    def mlp(which, v):
        for k, (W, b) in enumerate(gen.split_mlp(cfg, which, m[which + "_w"])):
            v = W.astype(np.float64) @ v + b.astype(np.float64)
            if k < 2:
                v = np.maximum(v, 0)
        return v

    def B(f):
        o = mlp("brdf", f)
        sg = lambda z: 1 / (1 + np.exp(-z))
        return o[:3] / np.linalg.norm(o[:3]), sg(o[3:6]), rough_min + sg(o[6]) * (1 - rough_min)

    def I(p, w):
        o = mlp("irt", np.concatenate([H(p), np.asarray(w, np.float64)]))
        v = (1.0 if o[0] > 0 else 0.0) if vis_mode else 1 / (1 + math.exp(-o[0]))
        return v, near_t + min(math.log1p(math.exp(o[1])), 1.0) * (far_t - near_t)

    def Li(w):
        He, We = env.shape[:2]
        th, ph = math.acos(max(-1, min(1, w[2]))), math.atan2(w[1], w[0])
        u, s = (ph / (2 * PI) + 0.5) * We - 0.5, th / PI * He - 0.5
        u0, s0 = math.floor(u), math.floor(s)
        fu, fs = u - u0, s - s0
        r0, r1 = min(max(s0, 0), He - 1), min(max(s0 + 1, 0), He - 1)
        return ((1 - fs) * ((1 - fu) * env[r0, u0 % We] + fu * env[r0, (u0 + 1) % We])
                + fs * ((1 - fu) * env[r1, u0 % We] + fu * env[r1, (u0 + 1) % We]))

    def fr_cos_pdf(n, a, r, wi, wov, pdf):
        NoL = n @ wi
        if NoL <= 0 or pdf <= 0:
            return np.zeros(3)
        NoV = max(n @ wov, 1e-4)
        hv = (wi + wov); hv = hv / max(np.linalg.norm(hv), 1e-12)
        NoH, VoH = max(n @ hv, 0), max(wov @ hv, 0)
        k = r ** 4
        Dg = k / (PI * (NoH * NoH * (k - 1) + 1) ** 2)
        Fr = f0 + (1 - f0) * (1 - VoH) ** 5
        G = 0.5 / (NoL * math.sqrt(NoV * NoV * (1 - k) + k) + NoV * math.sqrt(NoL * NoL * (1 - k) + k))
        return (a / PI + Dg * Fr * G) * NoL / pdf

    def radiance(p, wov, depth, dirs, pdfs, sdirs, spdfs):
        """Eq. 1 at p; at depth 0 also the (1-V) L'_o term of Eq. 2 over the secondary set, recursing once."""
        n, a, r = B(H(p))
        tot = np.zeros(3)
        for w, q in zip(dirs, pdfs):
            w64 = w.astype(np.float64)
            v = I(p, w)[0] if (flags & 2) or depth else 1.0
            tot += v * Li(w64) * fr_cos_pdf(n, a, r, w64, wov, float(q)) / len(dirs)
        if depth == 0 and (flags & 4):
            for w, q in zip(sdirs, spdfs):
                w64 = w.astype(np.float64)
                v, t = I(p, w)
                xs = np.clip(p.astype(np.float64) + t * w64, 0, 1).astype(np.float32)
                Lo = radiance(xs, -w64, 1, dt, pt, None, None)
                tot += (1 - v) * Lo * fr_cos_pdf(n, a, r, w64, wov, float(q)) / len(sdirs)
        return tot

    return np.array([radiance(x[i], wo[i].astype(np.float64), 0, dd[i], pd[i], None if dsec is None else dsec[i],
                              None if psec is None else psec[i]) for i in range(len(x))])


@pytest.mark.parametrize("vis_mode", [0, 1])
def test_whole_frame_brute_force(vis_mode):
    """pin 'whole frame': naive literal-recursive numpy evaluation of a few C0-like pixels == batched oracle to 1e-12."""
    cfg = gen.make_config("C0", S_i=4, S_2=3, flags=7, N=4096)
    m = gen.make_model(cfg)
    pix = np.array([0, 17, 301, 1022, 2048, 4095])
    fr = gen.make_frame(cfg, m["env"], pix)
    o = Oracle.from_gen(cfg, m, vis_mode=vis_mode)
    got = o.render_frame(fr["x"], fr["wo"], (fr["dir_d"], fr["pdf_d"]), (fr["dir_s"], fr["pdf_s"]), (fr["dir_t"], fr["pdf_t"]),
                         flags=7)["rgb"]
    ref = _naive_frame(cfg, m, fr["x"], fr["wo"], fr["dir_d"], fr["pdf_d"], fr["dir_s"], fr["pdf_s"], fr["dir_t"], fr["pdf_t"],
                       vis_mode, 7)
    np.testing.assert_allclose(got, ref, rtol=1e-11, atol=1e-13)
    assert (np.abs(ref).max(axis=1) > 1e-3).sum() >= 3


def test_frame_equals_stage_composition(c0):
    """render_frame == encode -> decode -> trace -> shade (the C-ABI's stage calls must compose the same way)."""
    cfg, m, fr, o = c0
    sl = slice(200, 264)
    x, wo, d, p = fr["x"][sl], fr["wo"][sl], fr["dir_d"][sl], fr["pdf_d"][sl]
    feat, _, _ = o.encode(x)
    brdf = o.decode(feat)
    vis, zv, t, xs = o.trace(x, feat, d)
    rgb = o.shade(brdf, wo, d, p, vis, terms=1)
    ref = o.render_frame(x, wo, (d, p), flags=3)["rgb"]
    np.testing.assert_allclose(rgb, ref, rtol=1e-13, atol=1e-15)


def test_flipbound_covers_a_forced_flip():
    """Q33: with hard visibility, flipping every near-threshold sample changes the pixel by at most flipbound."""
    cfg = gen.make_config("C0", S_i=4, S_2=3, flags=7)
    m = gen.make_model(cfg)
    pix = np.arange(0, 4096, 128)
    fr = gen.make_frame(cfg, m["env"], pix)
    args = (fr["x"], fr["wo"], (fr["dir_d"], fr["pdf_d"]), (fr["dir_s"], fr["pdf_s"]), (fr["dir_t"], fr["pdf_t"]))
    o = Oracle.from_gen(cfg, m, vis_mode=1)
    delta = 0.02
    base = o.render_frame(*args, flags=7, delta=delta)
    assert base["flipbound"].max() > 0
    # perturb the visibility bias by +-delta: only samples with |z_v| < delta can flip
    for sgn in (+1, -1):
        w = m["irt_w"].copy()
        w[-2] += sgn * delta * 0.999
        o2 = Oracle.from_gen(cfg, {**m, "irt_w": w}, vis_mode=1)
        pert = o2.render_frame(*args, flags=7)["rgb"]
        assert np.all(np.abs(pert - base["rgb"]) <= base["flipbound"] * (1 + 1e-9) + 1e-15)

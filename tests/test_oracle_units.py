"""Pins for the oracle's per-fragment functions: each is checked against
something other than itself -- a library routine, a closed form, a cited worked example."""
import os

import numpy as np
import pytest

import oracle


# ---- fp16 decode: all 65536 bit patterns against numpy's float16 -------------------------------
def test_half_to_double_all_patterns():
    bits = np.arange(65536, dtype=np.uint16)
    ref = bits.view(np.float16).astype(np.float64)
    got = np.array([oracle.half_to_double(int(b)) for b in bits])
    nan = np.isnan(ref)
    assert np.array_equal(np.isnan(got), nan)
    assert np.array_equal(got[~nan], ref[~nan])
    assert np.array_equal(np.signbit(got[~nan]), np.signbit(ref[~nan]))


# ---- SH basis -----------------------------------------------------------------------------------
def _real_sh_scipy(deg, v):
    """Real SH built from scipy's complex Y_l^m (library routine), without Condon-Shortley sign."""
    from scipy.special import sph_harm_y
    x, y, z = v
    theta = np.arccos(np.clip(z, -1, 1))
    phi = np.arctan2(y, x)
    out = []
    for l in range(deg + 1):
        for m in range(-l, l + 1):
            if m == 0:
                out.append(sph_harm_y(l, 0, theta, phi).real)
            elif m > 0:
                out.append(np.sqrt(2) * (-1) ** m * sph_harm_y(l, m, theta, phi).real)
            else:
                out.append(np.sqrt(2) * (-1) ** m * sph_harm_y(l, -m, theta, phi).imag)
    return np.array(out)


def test_sh_matches_scipy():
    rng = np.random.default_rng(1)
    for _ in range(200):
        v = rng.standard_normal(3)
        v /= np.linalg.norm(v)
        np.testing.assert_allclose(oracle.sh_basis(3, v), _real_sh_scipy(3, v), atol=1e-13)


def test_sh_band0_constant_and_symmetry(golden_dir):
    consts = {}
    for line in open(os.path.join(golden_dir, "sh_constants.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            consts[line[0]] = float(line[1])
    for v in ([0, 0, 1.0], [1.0, 0, 0], [0.6, 0.0, 0.8]):
        assert abs(oracle.sh_basis(0, v)[0] - consts["Y00"]) < 1e-9
    Y = oracle.sh_basis(3, [0.0, 0.0, 1.0])
    assert Y[1] == 0 and Y[3] == 0
    assert abs(Y[2] - consts["c1"]) < 1e-9
    assert abs(Y[6] - 2 * consts["c2b"]) < 1e-9                           # 3z^2-1 = 2
    assert abs(Y[12] - 2 * consts["c3d"]) < 1e-9                          # z(5z^2-3) = 2
    Y = oracle.sh_basis(3, [1.0, 0.0, 0.0])
    assert abs(Y[3] - consts["c1"]) < 1e-9 and abs(Y[8] - consts["c2c"]) < 1e-9
    assert abs(Y[15] - consts["c3a"]) < 1e-9 and abs(Y[13] + consts["c3c"]) < 1e-9
    Y = oracle.sh_basis(3, [0.0, 1.0, 0.0])
    assert abs(Y[1] - consts["c1"]) < 1e-9 and abs(Y[9] + consts["c3a"]) < 1e-9
    s = 1 / np.sqrt(3.0)
    Y = oracle.sh_basis(3, [s, s, s])
    assert abs(Y[4] - consts["c2a"] / 3) < 1e-9 and abs(Y[10] - consts["c3b"] * s ** 3) < 1e-9
    assert abs(Y[14]) < 1e-12 and abs(Y[11] - consts["c3c"] * s * (5 / 3 - 1)) < 1e-9


def test_sh_orthonormal_by_quadrature():
    # Gauss-Legendre in cos(theta) x uniform azimuth integrates degree <= 6 products exactly
    xs, ws = np.polynomial.legendre.leggauss(16)
    G = np.zeros((16, 16))
    naz = 32
    for ct, w in zip(xs, ws):
        st = np.sqrt(1 - ct * ct)
        for a in range(naz):
            ph = 2 * np.pi * (a + 0.5) / naz
            Y = oracle.sh_basis(3, [st * np.cos(ph), st * np.sin(ph), ct])
            G += w * (2 * np.pi / naz) * np.outer(Y, Y)
    assert np.abs(G - np.eye(16)).max() < 1e-12


# ---- bilinear sampling at texel centres, clamp-to-edge -----------------------------------------
@pytest.mark.parametrize("dtype", [np.float32, np.float16])
def test_bilinear_matches_grid_sample(dtype):
    """torch grid_sample(align_corners=False, padding_mode='border') is the texel-centre bilinear
    filter with clamp-to-edge that the paper says it mimics."""
    import torch
    rng = np.random.default_rng(2)
    H, W, n = 7, 5, 4
    tex = rng.standard_normal((H, W, n, 4)).astype(dtype)
    uv = rng.uniform(-0.1, 1.1, size=(400, 2))
    uv[:8] = [[0, 0], [1, 1], [0, 1], [1, 0], [0.5, 0.5], [0.1, 0.9], [1.0 - 1e-9, 0.3], [1e-9, 0.7]]
    t = torch.from_numpy(tex.astype(np.float64)).reshape(H, W, n * 4).permute(2, 0, 1)[None]
    grid = torch.from_numpy(uv * 2 - 1).reshape(1, 1, -1, 2)
    ref = torch.nn.functional.grid_sample(t, grid, mode="bilinear", padding_mode="border",
                                          align_corners=False)[0, :, 0].T.numpy().reshape(-1, n, 4)
    for i, (u, v) in enumerate(uv):
        np.testing.assert_allclose(oracle.sample_bilinear(tex, u, v), ref[i], atol=1e-12)


def test_bilinear_centre_midpoint_clamp():
    rng = np.random.default_rng(3)
    H, W, n = 6, 8, 9
    tex = rng.standard_normal((H, W, n, 4)).astype(np.float32)
    for (i, j) in [(0, 0), (3, 2), (7, 5)]:
        got = oracle.sample_bilinear(tex, (i + 0.5) / W, (j + 0.5) / H)
        assert np.array_equal(got, tex[j, i].astype(np.float64))
    got = oracle.sample_bilinear(tex, 3.0 / W, 2.5 / H)
    np.testing.assert_allclose(got, 0.5 * (tex[2, 2].astype(np.float64) + tex[2, 3]), atol=1e-15)
    assert np.array_equal(oracle.sample_bilinear(tex, -3.0, 2.5 / H), tex[2, 0].astype(np.float64))
    assert np.array_equal(oracle.sample_bilinear(tex, 0.5 / W, 9.0), tex[H - 1, 0].astype(np.float64))
    # rows are v, columns are u, no flip: a texture that is 1 only at (row 4, col 1)
    one = np.zeros((H, W, 1, 4), dtype=np.float32)
    one[4, 1] = 1.0
    assert oracle.sample_bilinear(one, 1.5 / W, 4.5 / H)[0, 0] == 1.0
    assert oracle.sample_bilinear(one, 4.5 / W, 1.5 / H)[0, 0] == 0.0


# ---- decode --------------------------------------------------------------------------------------
def test_decode_band0_closed_form():
    for s in (-3.0, 0.0, 0.7, 12.5):
        coef = np.zeros((16, 4))
        coef[0] = [s, -s, 2 * s, 0.5 * s]
        Y = oracle.sh_basis(3, [0.36, 0.48, 0.8])
        got = oracle.decode_rgba(coef, Y)
        want = 1 / (1 + np.exp(-0.28209479177387814 * np.array([s, -s, 2 * s, 0.5 * s])))
        np.testing.assert_allclose(got, want, atol=1e-15)


def test_decode_is_dot_then_logistic():
    rng = np.random.default_rng(4)
    from scipy.special import expit
    for _ in range(20):
        coef = rng.standard_normal((16, 4))
        v = rng.standard_normal(3)
        v /= np.linalg.norm(v)
        Y = oracle.sh_basis(3, v)
        np.testing.assert_allclose(oracle.decode_rgba(coef, Y), expit(_real_sh_scipy(3, v) @ coef), atol=1e-13)


# ---- blend ---------------------------------------------------------------------------------------
def test_blend_golden(golden_dir):
    n = 0
    for line in open(os.path.join(golden_dir, "blend_examples.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        k, layers, want = line.split("|")
        layers = np.array(layers.split(), dtype=np.float64).reshape(int(k), 4)
        want = np.array(want.split(), dtype=np.float64)
        np.testing.assert_allclose(oracle.blend(layers), want, atol=1e-15)
        n += 1
    assert n == 4


def test_blend_closed_form_and_misses():
    rng = np.random.default_rng(5)
    for _ in range(50):
        k = int(rng.integers(1, 10))
        L = rng.uniform(0, 1, size=(k, 4))
        hit = rng.integers(0, 2, size=k).astype(np.int32)
        bg = rng.uniform(0, 1, size=3)
        A = L[:, 3] * hit
        T = np.concatenate([[1.0], np.cumprod(1 - A)])
        want_rgb = (L[:, :3] * (A * T[:-1])[:, None]).sum(0) + T[-1] * bg
        got = oracle.blend(L, hit, 0.0, bg)
        np.testing.assert_allclose(got[:3], want_rgb, atol=1e-14)
        assert abs(got[3] - (1 - T[-1])) < 1e-14
    # k = 1 limit: a single opaque layer is a single-surface render (pins reading Q1)
    assert np.array_equal(oracle.blend([[0.2, 0.5, 0.7, 1.0]]), [0.2, 0.5, 0.7, 1.0])
    # nothing hit -> background, alpha 0
    assert np.array_equal(oracle.blend([[1, 1, 1, 1.0]], [0], 0.0, (0.1, 0.2, 0.3)), [0.1, 0.2, 0.3, 0.0])


def test_blend_early_exit_bound():
    rng = np.random.default_rng(6)
    for _ in range(200):
        L = rng.uniform(0, 1, size=(9, 4))
        L[:, 3] = rng.uniform(0.5, 1.0, size=9)
        tm = 2.0 ** -6
        a, b = oracle.blend(L, None, tm), oracle.blend(L, None, 0.0)
        assert np.abs(a - b).max() <= tm


# ---- vertex transform ------------------------------------------------------------------------------
def test_transform_matches_double_pinhole():
    from paper_2409_02482_b200 import synth
    rng = np.random.default_rng(7)
    cam = synth.look_at_camera((1.0, 0.7, -2.5), 640, 480)
    R = cam[4:13].astype(np.float64).reshape(3, 3)
    t = cam[13:16].astype(np.float64)
    for _ in range(300):
        p = rng.uniform(-1, 1, 3).astype(np.float32)
        X, Y, q, bad = oracle.transform_vertex(cam, 0.05, p)
        pc = R @ p.astype(np.float64) + t
        assert bad == 0
        xs = cam[0] * pc[0] / pc[2] + cam[2]
        ys = cam[1] * pc[1] / pc[2] + cam[3]
        assert abs(X / 256.0 - xs) <= 0.5 / 256 + 1e-3 and abs(Y / 256.0 - ys) <= 0.5 / 256 + 1e-3
        assert abs(q * pc[2] - 1) < 1e-5
    # exactly representable case: snapping is exact and round-half-even
    cam = np.array([64, 64, 8, 8, 1, 0, 0, 0, 1, 0, 0, 0, 1, 0, 0, 0], dtype=np.float32)
    assert oracle.transform_vertex(cam, 0.05, [0.25, -0.25, 2.0])[:2] == (16 * 256, 0)
    assert oracle.transform_vertex(cam, 0.05, [1.0 / 512 / 64 * 2, 0, 2.0])[0] == 8 * 256       # +0.5 -> even
    assert oracle.transform_vertex(cam, 0.05, [3.0 / 512 / 64 * 2, 0, 2.0])[0] == 8 * 256 + 2   # +1.5 -> even
    assert oracle.transform_vertex(cam, 0.05, [0, 0, 0.01])[3] == 1                               # behind near
    assert oracle.transform_vertex(cam, 0.05, [0, 0, -1.0])[3] == 1
    assert oracle.transform_vertex(cam, 0.05, [600.0, 0, 2.0])[3] == 2                            # guard band

"""Pins for the oracle's transparency attenuation (§4.2
"Transparency Attenuation": alpha_w = 2 Sigmoid(10 |v . n|) - 1 multiplies every fragment's opacity).
CPU only.  What is pinned: the function against the values SPEC.md prints and against tanh(5x); the face
normal against a numpy cross product; and the rendered effect against closed forms on quads whose
normal and view directions are known analytically (facing, tilted, back-facing, off-axis pixels)."""
import math
import os
import types

import numpy as np

import oracle

Y00 = 0.28209479177387814


def L(pos, uv, idx, tex):
    return types.SimpleNamespace(positions=np.asarray(pos, np.float32), uvs=np.asarray(uv, np.float32),
                                 indices=np.asarray(idx, np.uint32), texture=tex)


def ident_cam(f, W, H):
    return np.array([f, f, W / 2, H / 2, 1, 0, 0, 0, 1, 0, 0, 0, 1, 0, 0, 0], dtype=np.float32)


def const_tex(rgba_logit, size=4):
    t = np.zeros((size, size, 1, 4), dtype=np.float32)
    t[:, :, 0, :] = np.asarray(rgba_logit) / Y00
    return t


def sigmoid(x):
    return 1 / (1 + np.exp(-x))


def test_attenuation_golden(golden_dir):
    n = np.array([0.0, 0.0, 1.0])
    rows = [l.split() for l in open(os.path.join(golden_dir, "attenuation_examples.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for d, want, tol in rows:
        d, want, tol = float(d), float(want), float(tol)
        v = np.array([math.sqrt(1 - d * d), 0.0, d])
        assert abs(oracle.alpha_attenuation(v, n) - want) <= tol
        assert abs(oracle.alpha_attenuation(v, -n) - want) <= tol          # |v . n|: the sign of n is irrelevant


def test_attenuation_is_tanh_5x_and_monotone():
    rng = np.random.default_rng(3)
    prev = -1.0
    for d in np.linspace(0.0, 1.0, 101):
        phi = rng.uniform(0, 2 * math.pi)
        s = math.sqrt(max(0.0, 1 - d * d))
        v = np.array([s * math.cos(phi), s * math.sin(phi), -d])           # v . n = -d
        a = oracle.alpha_attenuation(v, [0, 0, 1])
        assert abs(a - math.tanh(5 * d)) <= 1e-15
        assert a > prev or d == 0.0
        prev = a


def test_face_normal_matches_cross_product():
    rng = np.random.default_rng(4)
    for _ in range(100):
        p = rng.normal(size=(3, 3)).astype(np.float32)
        n = oracle.face_normal(p[0], p[1], p[2])
        c = np.cross(p[1].astype(np.float64) - p[0], p[2].astype(np.float64) - p[0])
        np.testing.assert_allclose(n, c / np.linalg.norm(c), atol=1e-14)
        # reversing the winding flips the sign only
        np.testing.assert_allclose(oracle.face_normal(p[0], p[2], p[1]), -n, atol=1e-14)
    assert np.array_equal(oracle.face_normal([0, 0, 0], [1, 1, 1], [2, 2, 2]), np.zeros(3))   # zero area -> 0


def _quad(tilt_deg, d=2.0, hw=0.6):
    """Square of half-width hw centred on the optical axis at depth d, rotated by `tilt_deg` about the x axis
    (camera frame == world frame).  Its unit normal is (0, -sin t, cos t) up to sign."""
    t = math.radians(tilt_deg)
    corners = [(-hw, -hw), (hw, -hw), (hw, hw), (-hw, hw)]
    pos = [[x, y * math.cos(t), d + y * math.sin(t)] for x, y in corners]
    n = np.array([0.0, -math.sin(t), math.cos(t)])
    return pos, n


def _closed_form(W, H, f, n, logits):
    pi, pj = np.meshgrid(np.arange(W), np.arange(H), indexing="xy")
    dx, dy = (pi + 0.5 - W / 2) / f, (pj + 0.5 - H / 2) / f
    vdotn = np.abs(dx * n[0] + dy * n[1] + n[2]) / np.sqrt(dx * dx + dy * dy + 1.0)
    A = sigmoid(logits[3]) * np.tanh(5.0 * vdotn)
    rgb = sigmoid(np.asarray(logits[:3], dtype=np.float64))
    return np.concatenate([A[..., None] * rgb, A[..., None]], -1), vdotn


def test_quad_attenuation_closed_form():
    """k = 1, constant texture, background 0: rgba = (rgb A alpha_w, A alpha_w) with alpha_w from the analytic
    |v . n| of every pixel.  A wrong normal (tilted quads), a wrong v (off-axis pixels), a missing |.| (reversed
    winding) or a wrong constant (10) each break it."""
    W, H, f = 24, 16, 40.0
    cam = ident_cam(f, W, H)
    logits = [0.4, -0.3, 0.9, 1.2]
    uv = [[0, 0], [1, 0], [1, 1], [0, 1]]
    for tilt in (0.0, 35.0, -60.0, 80.0):
        pos, n = _quad(tilt)
        for idx in ([[0, 1, 2], [0, 2, 3]], [[0, 2, 1], [0, 3, 2]]):      # both windings
            lay = [L(pos, uv, idx, const_tex(logits))]
            r = oracle.render_view(lay, 0, cam, W, H, attenuation=True, want_layer_rgba=True)
            want, vdotn = _closed_form(W, H, f, n, logits)
            hit = r["ids"][0] != oracle.MISS
            assert hit.sum() > 40
            np.testing.assert_allclose(r["rgba"][hit], want[hit], atol=1e-7)   # fp32 vertex positions: ~1e-8 in n
            np.testing.assert_allclose(r["layer_rgba"][0][hit][:, 3], want[hit][:, 3], atol=1e-7)
            assert np.all(r["rgba"][~hit] == 0.0)
            # without the flag the same call gives the unattenuated opacity
            r0 = oracle.render_view(lay, 0, cam, W, H)
            np.testing.assert_allclose(r0["rgba"][hit][:, 3], sigmoid(logits[3]), atol=1e-12)
            if tilt == 0.0:    # head-on at the principal point: tanh(5 cos) with cos ~ 1
                assert abs(vdotn[H // 2, W // 2] - 1.0) < 2e-4
    # grazing: a quad containing the optical axis' direction is seen edge-on -> |v . n| -> 0 -> invisible
    pos, n = _quad(89.9)
    r = oracle.render_view([L(pos, uv, [[0, 1, 2], [0, 2, 3]], const_tex(logits))], 0, cam, W, H, attenuation=True)
    want, _ = _closed_form(W, H, f, n, logits)
    hit = r["ids"][0] != oracle.MISS
    np.testing.assert_allclose(r["rgba"][hit], want[hit], atol=1e-6)


def test_attenuated_blend_two_layers():
    """Two facing quads, front (layer 0) tilted: C = c0 A0 w0 + (1 - A0 w0) c1 A1 w1 with per-pixel analytic w."""
    W, H, f = 16, 16, 32.0
    cam = ident_cam(f, W, H)
    uv = [[0, 0], [1, 0], [1, 1], [0, 1]]
    idx = [[0, 1, 2], [0, 2, 3]]
    l0, l1 = [0.5, 0.1, -0.7, 0.3], [-0.2, 0.8, 0.6, 2.0]
    p0, n0 = _quad(40.0, d=2.0, hw=0.8)
    p1, n1 = _quad(0.0, d=3.0, hw=2.0)
    r = oracle.render_view([L(p0, uv, idx, const_tex(l0)), L(p1, uv, idx, const_tex(l1))], 0, cam, W, H,
                           attenuation=True, t_min=0.0)
    w0, _ = _closed_form(W, H, f, n0, l0)
    w1, _ = _closed_form(W, H, f, n1, l1)
    both = (r["ids"][0] != oracle.MISS) & (r["ids"][1] != oracle.MISS)
    assert both.sum() > 50
    want_rgb = w0[..., :3] + (1 - w0[..., 3:]) * w1[..., :3]
    want_a = 1 - (1 - w0[..., 3]) * (1 - w1[..., 3])
    np.testing.assert_allclose(r["rgba"][both][:, :3], want_rgb[both], atol=1e-7)
    np.testing.assert_allclose(r["rgba"][both][:, 3], want_a[both], atol=1e-7)

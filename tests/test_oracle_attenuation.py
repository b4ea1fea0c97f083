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
from paper_2409_02482_b200 import synth

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


# ---- optional per-vertex normals ----------------------------------

def test_interp_normal_unit_function():
    n = oracle.interp_normal([0.2, 0.3, 0.5], [1, 0, 0], [0, 1, 0], [0, 0, 1])
    want = np.array([0.2, 0.3, 0.5]) / np.linalg.norm([0.2, 0.3, 0.5])
    np.testing.assert_allclose(n, want, atol=1e-15)
    np.testing.assert_allclose(oracle.interp_normal([1, 0, 0], [0, 0, 3], [5, 0, 0], [0, 7, 0]), [0, 0, 1], atol=1e-15)   # need not be unit
    assert np.all(oracle.interp_normal([0.5, 0.5, 0.0], [0, 0, 1], [0, 0, -1], [1, 0, 0]) == 0.0)                        # vanishing sum -> 0


def test_radial_vertex_normals_of_a_sphere_mesh_give_the_hit_direction():
    """Icospheres centred at the origin with vertex normal = vertex position / radius.  The perspective-correct barycentrics
    interpolate the 3-D hit point p on the facet, so sum b_i n_i = p / r and the renormalised normal is EXACTLY p / |p|:
    alpha_w = 2 Sigmoid(10 |v . p/|p||) - 1 in closed form from the depth buffer.  The face normal differs from it by up to
    the facet angle, so the test also tells the two paths apart."""
    sc = synth.make_config(1, width=96, height=96, num_cameras=2)
    for ly in sc.layers:
        ly.texture[...] = 0.0
        ly.texture[:, :, 0, 3] = 0.9 / Y00                     # constant opacity sigmoid(0.9) everywhere, view independent
        ly.normals = (ly.positions / np.linalg.norm(ly.positions, axis=1, keepdims=True)).astype(np.float32)
    a0 = 1.0 / (1.0 + math.exp(-float(np.float32(0.9 / Y00)) * Y00))
    for vi in (0, 1):
        cam = sc.cameras[vi]
        r = oracle.render_scene(sc, [vi], attenuation=True, want_layer_rgba=True, want_qp=True, want_layer_normal=True)[0]
        rf = None
        R, t = cam[4:13].reshape(3, 3).astype(np.float64), cam[13:16].astype(np.float64)
        W, H = sc.width, sc.height
        pi, pj = np.meshgrid(np.arange(W), np.arange(H), indexing="xy")
        dcam = np.stack([(pi + 0.5 - cam[2]) / cam[0], (pj + 0.5 - cam[3]) / cam[1], np.ones_like(pi, dtype=np.float64)], -1)
        vdir = dcam @ R                                         # world = R^T cam
        vdir /= np.linalg.norm(vdir, axis=-1, keepdims=True)
        for l in range(sc.k):
            hit = r["ids"][l] != oracle.MISS
            z = 1.0 / r["qp"][l][hit].astype(np.float64)
            pw = (dcam[hit] * z[:, None] - t) @ R
            nrm = pw / np.linalg.norm(pw, axis=1, keepdims=True)
            d = np.abs((vdir[hit] * nrm).sum(-1))
            want = a0 * (2.0 / (1.0 + np.exp(-10.0 * d)) - 1.0)
            got = r["layer_rgba"][l][hit][:, 3]
            # the rasteriser's barycentrics belong to the triangle of the SNAPPED vertices (1/256 px): against the exact ray
            # hit they are off by ~1e-4 relative, which the facet angle (0.1 rad) and the slope of alpha_w (<= 5) turn into
            # <= ~1e-4 in alpha_w; the face-normal path below is two orders of magnitude away
            np.testing.assert_allclose(got, want, atol=1.5e-4)
            # the normal buffer holds the interpolated normal, facing the viewer
            np.testing.assert_allclose(np.abs((r["layer_normal"][l][hit] * nrm).sum(-1)), 1.0, atol=1e-9)
            assert np.all((r["layer_normal"][l][hit] * vdir[hit]).sum(-1) <= 1e-12)
        # negative control: with the FACE normals the opacities differ measurably near the silhouette
        for ly in sc.layers:
            ly.normals_saved, ly.normals = ly.normals, None
        rf = oracle.render_scene(sc, [vi], attenuation=True, want_layer_rgba=True)[0]
        for ly in sc.layers:
            ly.normals = ly.normals_saved
        hit0 = r["ids"][0] != oracle.MISS
        assert np.abs(rf["layer_rgba"][0][hit0][:, 3] - r["layer_rgba"][0][hit0][:, 3]).max() > 1.5e-2


def test_vertex_normals_equal_to_the_face_normal_change_nothing():
    """A tilted flat quad whose four vertex normals are its face normal: interpolation and renormalisation return that
    normal, so the render coincides with the face-normal path (and with -n: only |v . n| matters)."""
    W, H, f = 40, 30, 64.0
    tilt = 0.6
    pos = np.array([[-1.2, -0.9, 3.0 - 1.2 * tilt], [1.2, -0.9, 3.0 + 1.2 * tilt], [1.2, 0.9, 3.0 + 1.2 * tilt], [-1.2, 0.9, 3.0 - 1.2 * tilt]], np.float32)
    uv = [[0, 0], [1, 0], [1, 1], [0, 1]]
    idx = [[0, 1, 2], [0, 2, 3]]
    tex = np.zeros((8, 8, 1, 4), np.float32)
    tex[..., 0, :] = np.array([0.3, -0.2, 0.5, 1.3]) / Y00
    n = oracle.face_normal(pos[0], pos[1], pos[2])
    base = L(pos, uv, idx, tex)
    ref = oracle.render_view([base], 0, ident_cam(f, W, H), W, H, attenuation=True, want_layer_rgba=True)
    for sign in (1.0, -1.0):
        lv = L(pos, uv, idx, tex)
        lv.normals = np.tile((sign * n).astype(np.float32), (4, 1))
        got = oracle.render_view([lv], 0, ident_cam(f, W, H), W, H, attenuation=True, want_layer_rgba=True)
        assert np.array_equal(got["ids"], ref["ids"]) and (ref["ids"] != oracle.MISS).sum() > 100
        np.testing.assert_allclose(got["rgba"], ref["rgba"], atol=1e-7)       # n is stored as fp32: 6e-8 relative
        np.testing.assert_allclose(got["layer_rgba"], ref["layer_rgba"], atol=1e-7)


def test_linearly_varying_vertex_normals_closed_form():
    """Viewport-filling quad at constant depth facing the camera (perspective-correct == affine in the pixel position) with
    vertex normals (sx, 0, -1): the interpolated normal at pixel column i is normalize((x(i), 0, -1)), x affine from -s to s;
    alpha_w = 2 Sigmoid(10 |v . n|) - 1 with the pixel's own view direction -- recomputed here with numpy only."""
    W, H, f, d, s = 32, 20, 64.0, 2.0, 1.5
    hx, hy = (W / 2) * d / f, (H / 2) * d / f
    pos = [[-hx, -hy, d], [hx, -hy, d], [hx, hy, d], [-hx, hy, d]]
    uv = [[0, 0], [1, 0], [1, 1], [0, 1]]
    tex = np.zeros((4, 4, 1, 4), np.float32)
    tex[..., 0, 3] = 0.4 / Y00
    ly = L(pos, uv, [[0, 1, 2], [0, 2, 3]], tex)
    ly.normals = np.array([[-s, 0, -1], [s, 0, -1], [s, 0, -1], [-s, 0, -1]], np.float32)
    r = oracle.render_view([ly], 0, ident_cam(f, W, H), W, H, attenuation=True, want_layer_rgba=True)
    a0 = 1.0 / (1.0 + math.exp(-float(np.float32(0.4 / Y00)) * Y00))
    i = np.arange(W) + 0.5
    x = -s + 2.0 * s * i / W
    for j in (0, 7, 19):
        n = np.stack([x, np.zeros(W), -np.ones(W)], -1)
        n /= np.linalg.norm(n, axis=1, keepdims=True)
        v = np.stack([(i - W / 2) / f, np.full(W, (j + 0.5 - H / 2) / f), np.ones(W)], -1)
        v /= np.linalg.norm(v, axis=1, keepdims=True)
        want = a0 * (2.0 / (1.0 + np.exp(-10.0 * np.abs((v * n).sum(-1)))) - 1.0)
        np.testing.assert_allclose(r["layer_rgba"][0, j, :, 3], want, atol=1e-6)

"""Pins for the oracle's per-layer render buffers (PAPER.md:L763-803 supplement Fig. "render
buffers": surface normals, surface UVs, surface opacity, surface colours per layer).  CPU only."""
import math
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


def test_fullscreen_quad_buffers_closed_form():
    """Viewport-filling quad at constant depth with UVs affine in the pixel position: the UV buffer is ((i+.5)/W,
    (j+.5)/H) exactly (perspective-correct == affine at constant depth), the colour / opacity buffers are
    sigmoid(Y00 coef) of a constant texture (NOT premultiplied, NOT composited), the normal faces the viewer."""
    W, H, f, d = 16, 12, 64.0, 2.0
    hx, hy = (W / 2) * d / f, (H / 2) * d / f
    pos = [[-hx, -hy, d], [hx, -hy, d], [hx, hy, d], [-hx, hy, d]]
    uv = [[0, 0], [1, 0], [1, 1], [0, 1]]
    logits = np.array([0.7, -0.4, 0.2, -1.1])
    tex = np.zeros((4, 4, 1, 4), np.float32)
    tex[:, :, 0, :] = logits / Y00
    behind = np.zeros((4, 4, 1, 4), np.float32)
    behind[:, :, 0, :] = np.array([2.0, 2.0, 2.0, 30.0]) / Y00
    pos2 = [[p[0] * 2, p[1] * 2, 2 * d] for p in pos]
    for idx in ([[0, 1, 2], [0, 2, 3]], [[0, 2, 1], [0, 3, 2]]):
        r = oracle.render_view([L(pos, uv, idx, tex), L(pos2, uv, idx, behind)], 0, ident_cam(f, W, H), W, H,
                               want_layer_rgba=True, want_layer_uv=True, want_layer_normal=True)
        pi, pj = np.meshgrid(np.arange(W), np.arange(H), indexing="xy")
        np.testing.assert_allclose(r["layer_uv"][0][..., 0], (pi + 0.5) / W, atol=1e-7)
        np.testing.assert_allclose(r["layer_uv"][0][..., 1], (pj + 0.5) / H, atol=1e-7)
        want = 1 / (1 + np.exp(-logits.astype(np.float32).astype(np.float64) / np.float32(Y00) * Y00))
        np.testing.assert_allclose(r["layer_rgba"][0], np.broadcast_to(want, (H, W, 4)), atol=1e-7)
        # the buffer of the layer behind is its own colour/opacity, untouched by the layer in front
        np.testing.assert_allclose(r["layer_rgba"][1][..., 3], 1.0, atol=1e-12)
        np.testing.assert_allclose(r["layer_rgba"][1][..., 0], 1 / (1 + math.exp(-2.0)), atol=1e-7)
        # camera looks down +z from the origin: the normal that faces the viewer is (0, 0, -1), whatever the winding
        np.testing.assert_allclose(r["layer_normal"][0], np.broadcast_to([0.0, 0.0, -1.0], (H, W, 3)), atol=1e-12)


def test_buffers_zero_on_miss_and_with_early_exit():
    sc = synth.make_config(1, width=48, height=40, num_cameras=1, tex_size=32)
    for ly in sc.layers:
        ly.texture[:, :, 0, 3] += 40.0          # opaque outer layer: compositing stops after it ...
    r = oracle.render_scene(sc, [0], want_layer_rgba=True, want_layer_uv=True, want_layer_normal=True, t_min=2.0 ** -6)[0]
    miss = r["ids"] == oracle.MISS
    assert miss.any() and (~miss).any()
    for key in ("layer_rgba", "layer_uv", "layer_normal"):
        assert np.all(r[key][miss] == 0.0)
    # ... but the buffers of the layers behind it are still filled (they are per-layer, not composited)
    inner = ~miss[2]
    assert inner.sum() > 50 and np.all(r["layer_rgba"][2][inner][:, 3] > 0.99)
    assert np.all(np.abs(np.linalg.norm(r["layer_normal"][2][inner], axis=-1) - 1.0) < 1e-12)


def test_sphere_normals_face_the_viewer_and_follow_the_surface():
    """Icospheres centred at the origin seen from outside: the facing normal of a hit is close to the outward radial
    direction of the hit point (within the facet angle) and always satisfies v . n <= 0."""
    sc = synth.make_config(1)
    cam = sc.cameras[1]
    r = oracle.render_scene(sc, [1], want_layer_normal=True, want_qp=True)[0]
    R, t = cam[4:13].reshape(3, 3).astype(np.float64), cam[13:16].astype(np.float64)
    W, H = sc.width, sc.height
    pi, pj = np.meshgrid(np.arange(W), np.arange(H), indexing="xy")
    dcam = np.stack([(pi + 0.5 - cam[2]) / cam[0], (pj + 0.5 - cam[3]) / cam[1], np.ones_like(pi, dtype=np.float64)], -1)
    for l in range(sc.k):
        hit = r["ids"][l] != oracle.MISS
        z = 1.0 / r["qp"][l][hit].astype(np.float64)                  # camera depth of the fragment
        pw = (dcam[hit] * z[:, None] - t) @ R                            # x_world = R^T (x_cam - t)
        radial = pw / np.linalg.norm(pw, axis=-1, keepdims=True)
        n = r["layer_normal"][l][hit]
        assert np.all(np.sum(n * radial, -1) > math.cos(math.radians(12.0)))   # subdivision-3 facets: < ~10 degrees
        v = dcam[hit] @ R
        assert np.all(np.sum(n * v, -1) <= 1e-12)

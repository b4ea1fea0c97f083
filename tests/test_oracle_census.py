"""Pins for the oracle's footprint census `vso_count_footprints` (B_tex = unique texels referenced by the
2x2 footprints of shaded fragments, "counted, not assumed: an instrumented pass or the oracle").  The census is the
numerator of every roofline fraction bench.py prints, so it is pinned on scenes whose count is known by hand.  CPU only."""
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


def quad(W, H, f, d, x0, x1, y0, y1, u0, u1, v0, v1):
    """Axis-aligned quad at depth d whose edges fall on the pixel BOUNDARIES x0, x1 / y0, y1 (so it covers exactly the
    pixels x0 <= i < x1, y0 <= j < y1) with UV affine in the pixel position: u = u0 at pixel boundary x0, u1 at x1."""
    def wx(x): return (x - W / 2) * d / f
    def wy(y): return (y - H / 2) * d / f
    pos = [[wx(x0), wy(y0), d], [wx(x1), wy(y0), d], [wx(x1), wy(y1), d], [wx(x0), wy(y1), d]]
    uv = [[u0, v0], [u1, v0], [u1, v1], [u0, v1]]
    return pos, uv, [[0, 1, 2], [0, 2, 3]]


def const_tex(w, h, alpha_logit):
    t = np.zeros((h, w, 1, 4), np.float32)
    t[:, :, 0, 3] = alpha_logit / Y00
    return t


def census(layers, W, H, t_min=2.0 ** -14, marks=None):
    r = oracle.render_view(layers, 0, ident_cam(64.0, W, H), W, H, t_min=t_min, want_layer_rgba=True, want_layer_uv=True)
    return oracle.count_footprints(layers, W, H, r, t_min=t_min, marks=marks), r


def test_magnified_quad_two_texels_per_pixel_axis():
    """Full-screen quad, texture 2W x 2H: pixel i maps to x = 2 i + 0.5, so its footprint is columns {2i, 2i+1} (fraction 0.5,
    far from every rounding edge): the footprints tile the texture, every texel is referenced exactly once."""
    W, H = 16, 12
    pos, uv, idx = quad(W, H, 64.0, 2.0, 0, W, 0, H, 0, 1, 0, 1)
    (frags, fresh, marks), _ = census([L(pos, uv, idx, const_tex(2 * W, 2 * H, 0.0))], W, H)
    assert frags == W * H
    assert fresh == 4 * W * H and marks[0].all()


def test_sub_rectangle_and_texture_window():
    """A quad over pixels [3, 11) x [2, 7) whose UVs address the texel window [8, 24) x [4, 14) of a 40 x 30 texture at two
    texels per pixel: 8 x 5 fragments, and exactly the 16 x 10 texels of the window -- nothing outside it."""
    W, H, tw, th = 16, 12, 40, 30
    pos, uv, idx = quad(W, H, 64.0, 2.0, 3, 11, 2, 7, 8 / tw, 24 / tw, 4 / th, 14 / th)
    (frags, fresh, marks), _ = census([L(pos, uv, idx, const_tex(tw, th, 0.0))], W, H)
    assert frags == 8 * 5
    want = np.zeros((th, tw), np.uint8)
    want[4:14, 8:24] = 1
    assert fresh == 160 and np.array_equal(marks[0], want)


def test_minified_quad_skips_texels():
    """Texture 4W wide, W pixels across: x = 4 i + 1.5, footprint columns {4i+1, 4i+2}: half of the columns are never
    fetched.  Rows at one texel per two... (th = H/2: y = j/2 - 0.25): rows floor(j/2 - 0.25) and +1, clamped at both ends,
    reference every row."""
    W, H = 16, 12
    tw, th = 4 * W, H // 2
    pos, uv, idx = quad(W, H, 64.0, 2.0, 0, W, 0, H, 0, 1, 0, 1)
    (frags, fresh, marks), _ = census([L(pos, uv, idx, const_tex(tw, th, 0.0))], W, H)
    cols = np.zeros(tw, bool)
    for i in range(W):
        cols[4 * i + 1] = cols[4 * i + 2] = True
    want = np.zeros((th, tw), np.uint8)
    want[:, cols] = 1
    assert frags == W * H and fresh == th * 2 * W and np.array_equal(marks[0], want)


def test_early_exit_stops_the_census_and_misses_do_not_count():
    """Three layers: the first covers the left half, the second (opaque: alpha = 1 up to 1e-18, T < t_min) everything, the
    third everything.  Fragments: left half 2 (layer 0 + the stopping layer 1), right half 1 (layer 1); layer 2 is never
    composited, so none of its texels is referenced.  With t_min = 0 nothing stops: layer 2 counts everywhere."""
    W, H = 16, 12
    p0, uv0, idx = quad(W, H, 64.0, 2.0, 0, W // 2, 0, H, 0, 0.5, 0, 1)
    p1, uv1, _ = quad(W, H, 64.0, 3.0, 0, W, 0, H, 0, 1, 0, 1)
    p2, uv2, _ = quad(W, H, 64.0, 4.0, 0, W, 0, H, 0, 1, 0, 1)
    layers = [L(p0, uv0, idx, const_tex(2 * W, 2 * H, 0.0)), L(p1, uv1, idx, const_tex(2 * W, 2 * H, 60.0)),
              L(p2, uv2, idx, const_tex(2 * W, 2 * H, 0.0))]
    (frags, fresh, marks), r = census(layers, W, H)
    assert (r["ids"][0][:, W // 2:] == oracle.MISS).all() and (r["ids"][2] != oracle.MISS).all()
    assert frags == (W // 2) * H * 2 + (W // 2) * H
    assert marks[0][:, :W].all() and not marks[0][:, W:].any()
    assert marks[1].all() and not marks[2].any()
    assert fresh == 2 * W * H + 4 * W * H
    (frags0, fresh0, marks0), _ = census(layers, W, H, t_min=0.0)
    assert frags0 == frags + W * H and marks0[2].all() and fresh0 == fresh + 4 * W * H


def test_marks_accumulate_over_views():
    """`fresh` counts texels newly marked by the call: rendering the same view twice adds fragments but no texels."""
    sc = synth.make_config(1, width=48, height=40, num_cameras=2, tex_size=64)
    kw = dict(want_layer_rgba=True, want_layer_uv=True)
    r0, r1 = oracle.render_scene(sc, [0, 1], **kw)
    f0, t0, marks = oracle.count_footprints(sc.layers, sc.width, sc.height, r0, t_min=sc.t_min)
    assert f0 == int((r0["ids"] != oracle.MISS).sum())          # C1 opacities ~ 0.5: no early exit at 3 layers
    assert t0 == sum(int(m.sum()) for m in marks) and 0 < t0 <= 4 * f0
    f0b, t0b, _ = oracle.count_footprints(sc.layers, sc.width, sc.height, r0, t_min=sc.t_min, marks=marks)
    assert f0b == f0 and t0b == 0
    _, t1, _ = oracle.count_footprints(sc.layers, sc.width, sc.height, r1, t_min=sc.t_min, marks=marks)
    _, t1_alone, _ = oracle.count_footprints(sc.layers, sc.width, sc.height, r1, t_min=sc.t_min)
    assert 0 < t1 <= t1_alone and t0 + t1 == sum(int(m.sum()) for m in marks)


def test_footprint_is_the_one_bilinear_sampling_reads():
    """The census addresses the same four texels as vso_sample_bilinear: put a huge value into exactly the marked texels of a
    zero texture and re-render -- every hit pixel's sampled opacity logit must then be that value (weights sum to 1); put it
    into the UNMARKED texels instead and no pixel may change."""
    sc = synth.make_config(1, width=40, height=40, num_cameras=1, tex_size=48)
    k = sc.k
    for ly in sc.layers:
        ly.texture[...] = 0.0
    r = oracle.render_scene(sc, [0], want_layer_rgba=True, want_layer_uv=True, t_min=0.0)[0]
    _, _, marks = oracle.count_footprints(sc.layers, sc.width, sc.height, r, t_min=0.0)
    for l, ly in enumerate(sc.layers):
        ly.texture[:, :, 0, 3] = np.where(marks[l] != 0, 8.0 / Y00, 0.0)
    r2 = oracle.render_scene(sc, [0], want_layer_rgba=True, t_min=0.0)[0]
    hit = r["ids"] != oracle.MISS
    assert hit.sum() > 500
    np.testing.assert_allclose(r2["layer_rgba"][hit][:, 3], 1 / (1 + np.exp(-8.0)), atol=1e-6)
    for l, ly in enumerate(sc.layers):
        ly.texture[:, :, 0, 3] = np.where(marks[l] != 0, 0.0, 8.0 / Y00)
    r3 = oracle.render_scene(sc, [0], want_layer_rgba=True, t_min=0.0)[0]
    np.testing.assert_allclose(r3["layer_rgba"][hit][:, 3], 0.5, atol=1e-12)
    assert k == 3

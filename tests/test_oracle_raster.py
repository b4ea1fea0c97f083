"""Pins for the oracle's rasteriser + compositor (the five `north_star` self-checks, SURVEY.md §8(c),
plus the sorting-free theorem check).  Everything here is CPU-only."""
import os
import types

import numpy as np
import pytest

import oracle
from paper_2409_02482_b200 import synth

Y00 = 0.28209479177387814
MISS = oracle.MISS


def L(pos, uv, idx, tex):
    return types.SimpleNamespace(positions=np.asarray(pos, np.float32), uvs=np.asarray(uv, np.float32),
                                 indices=np.asarray(idx, np.uint32), texture=tex)


def ident_cam(f, W, H):
    return np.array([f, f, W / 2, H / 2, 1, 0, 0, 0, 1, 0, 0, 0, 1, 0, 0, 0], dtype=np.float32)


def const_tex(rgba_logit, n=1, size=4, dtype=np.float32):
    t = np.zeros((size, size, n, 4), dtype=dtype)
    t[:, :, 0, :] = np.asarray(rgba_logit) / Y00
    return t


def sigmoid(x):
    return 1 / (1 + np.exp(-x))


# ---- 1. closed-form full-screen textured quad -------------------------------------------------------
def test_fullscreen_quad_closed_form():
    W = H = 16
    f, d = 64.0, 2.0
    hw = (W / 2) * d / f          # 0.25: projects exactly onto the viewport corners
    pos = [[-hw, -hw, d], [hw, -hw, d], [hw, hw, d], [-hw, hw, d]]
    uv = [[0, 0], [1, 0], [1, 1], [0, 1]]
    Wt, Ht = 2 * W, 2 * H
    ii, jj = np.meshgrid(np.arange(Wt), np.arange(Ht), indexing="xy")
    a = np.array([0.3, -0.2, 0.1, 0.5])
    b = np.array([0.05, 0.02, -0.03, 0.01])
    c = np.array([-0.04, 0.03, 0.02, 0.06])
    tex = np.zeros((Ht, Wt, 4, 4), dtype=np.float32)      # degree 1, higher bands zero
    tex[:, :, 0, :] = a + ii[..., None] * b + jj[..., None] * c
    cam = ident_cam(f, W, H)
    # both triangles in one layer: ids give the diagonal ownership
    r = oracle.render_view([L(pos, uv, [[0, 1, 2], [0, 2, 3]], tex)], 1, cam, W, H)
    pi, pj = np.meshgrid(np.arange(W), np.arange(H), indexing="xy")
    x = (pi + 0.5) / W * Wt - 0.5          # texel coordinates of the pixel centre
    y = (pj + 0.5) / H * Ht - 0.5
    s = tex[0, 0, 0].astype(np.float64) * 0 + (a.astype(np.float32).astype(np.float64)) \
        + x[..., None] * b.astype(np.float32).astype(np.float64) \
        + y[..., None] * c.astype(np.float32).astype(np.float64)
    rgba = sigmoid(Y00 * s)
    want = np.concatenate([rgba[..., :3] * rgba[..., 3:], rgba[..., 3:]], -1)   # bg = 0: C = rgb*A
    # float32 texel values a + i b + j c are rounded: tolerance 64 * 2^-24
    np.testing.assert_allclose(r["rgba"], want, atol=5e-6)
    # upper-right triangle (0) owns the diagonal: it is its LEFT edge; lower-left triangle is 1
    assert np.array_equal(r["ids"][0], np.where(pi >= pj, 0, 1).astype(np.uint32))
    # one triangle per layer: every pixel is covered exactly once across the shared diagonal
    r2 = oracle.render_view([L(pos, uv, [[0, 1, 2]], tex), L(pos, uv, [[0, 2, 3]], tex)], 1, cam, W, H)
    c0, c1 = r2["ids"][0] != MISS, r2["ids"][1] != MISS
    assert np.all(c0 ^ c1)
    # orientation does not matter (no culling, reading Q9): flipped winding, same coverage
    r3 = oracle.render_view([L(pos, uv, [[0, 2, 1], [0, 3, 2]], tex)], 1, cam, W, H)
    assert np.array_equal(r3["ids"], r["ids"])
    np.testing.assert_array_equal(r3["rgba"], r["rgba"])


# ---- top-left rule, hand-counted fixture ------------------------------------------------------------
def test_topleft_golden(golden_dir):
    rows = [l.split() for l in open(os.path.join(golden_dir, "topleft_triangle.txt"))
            if l.strip() and not l.startswith("#")]
    want = np.array(rows, dtype=np.int64).astype(bool)
    W = H = 6
    f, d = 8.0, 1.0
    cam = ident_cam(f, W, H)
    to_world = lambda px, py: [(px - W / 2) / f * d, (py - H / 2) / f * d, d]   # exact in fp32
    tri = [to_world(0.5, 0.5), to_world(4.5, 0.5), to_world(0.5, 4.5)]
    uv = [[0, 0], [1, 0], [0, 1]]
    for idx in ([[0, 1, 2]], [[0, 2, 1]], [[1, 2, 0]]):
        r = oracle.render_view([L(tri, uv, idx, const_tex([0, 0, 0, 0]))], 0, cam, W, H)
        assert np.array_equal(r["ids"][0] != MISS, want)
    assert want.sum() == 10
    # two triangles sharing the hypotenuse: every sample on it belongs to exactly one of them
    quad = tri + [to_world(4.5, 4.5)]
    ra = oracle.render_view([L(quad, uv + [[1, 1]], [[0, 1, 2]], const_tex([0, 0, 0, 0])),
                             L(quad, uv + [[1, 1]], [[1, 3, 2]], const_tex([0, 0, 0, 0]))], 0, cam, W, H)
    ca, cb = ra["ids"][0] != MISS, ra["ids"][1] != MISS
    assert not np.any(ca & cb)
    ii, jj = np.meshgrid(np.arange(W), np.arange(H), indexing="xy")
    assert np.array_equal(ca | cb, (ii < 4) & (jj < 4))       # right and bottom edges excluded


# ---- 5(i). exact brute force: every pixel x every triangle, no bounding boxes ---------------------
def _snap_all(cam, near, pos):
    out = [oracle.transform_vertex(cam, near, p) for p in pos]
    return out


def _brute_ids(layer, cam, W, H, near=0.05):
    """Independent restatement of DESIGN.md §3.2-3.4 with Python integers and numpy float32."""
    vt = _snap_all(cam, near, layer.positions)
    best = {}
    f32 = np.float32
    for t, (i0, i1, i2) in enumerate(layer.indices.tolist()):
        v = [vt[i0], vt[i1], vt[i2]]
        if any(x[3] for x in v):
            continue
        A2 = (v[1][0] - v[0][0]) * (v[2][1] - v[0][1]) - (v[2][0] - v[0][0]) * (v[1][1] - v[0][1])
        if A2 == 0:
            continue
        if A2 < 0:
            v[1], v[2] = v[2], v[1]
            A2 = -A2
        for j in range(H):
            for i in range(W):
                Sx, Sy = 256 * i + 128, 256 * j + 128
                E = []
                ok = True
                for e in range(3):
                    a, b = v[(e + 1) % 3], v[(e + 2) % 3]
                    dx, dy = b[0] - a[0], b[1] - a[1]
                    Ev = dx * (Sy - a[1]) - dy * (Sx - a[0])
                    tl = dy < 0 or (dy == 0 and dx > 0)
                    if not (Ev > 0 or (Ev == 0 and tl)):
                        ok = False
                        break
                    E.append(Ev)
                if not ok:
                    continue
                assert sum(E) == A2
                # fp32: fma(f2,q2, fma(f1,q1, f0*q0)) / fA -- fma emulated exactly in float64->float32
                m = f32(f32(E[0]) * f32(v[0][2]))
                n1 = f32(np.float64(f32(E[1])) * np.float64(f32(v[1][2])) + np.float64(m))
                n2 = f32(np.float64(f32(E[2])) * np.float64(f32(v[2][2])) + np.float64(n1))
                qp = f32(n2 / f32(A2))
                key = (int(qp.view(np.uint32)) << 32) | (0xFFFFFFFF - t)
                if key > best.get((j, i), 0):
                    best[(j, i)] = key
    ids = np.full((H, W), MISS, dtype=np.uint32)
    for (j, i), key in best.items():
        ids[j, i] = 0xFFFFFFFF - (key & 0xFFFFFFFF)
    return ids


def _soup(rng, n, spread=0.9, size=0.5, z=(2.0, 4.0)):
    c = np.stack([rng.uniform(-spread, spread, n), rng.uniform(-spread, spread, n), rng.uniform(*z, n)], 1)
    pos = (c[:, None, :] + rng.uniform(-size, size, (n, 3, 3)) * [1, 1, 0.3]).reshape(-1, 3)
    return pos.astype(np.float32), rng.uniform(0, 1, (3 * n, 2)).astype(np.float32), \
        np.arange(3 * n, dtype=np.uint32).reshape(n, 3)


def test_bruteforce_exact_ids():
    rng = np.random.default_rng(11)
    W, H = 24, 20
    cam = synth.look_at_camera((0.3, -0.2, -0.5), W, H, 50.0, target=(0, 0, 3.0))
    layers = []
    for l in range(2):
        pos, uv, idx = _soup(rng, 60)
        layers.append(L(pos, uv, idx, const_tex([0, 0, 0, 0])))
    # degenerate + duplicated triangles: zero area is skipped, equal depth -> lowest index wins
    layers[0].indices = np.concatenate([layers[0].indices, [[0, 0, 1]], layers[0].indices[:5]]).astype(np.uint32)
    r = oracle.render_view(layers, 0, cam, W, H)
    for l in range(2):
        assert np.array_equal(r["ids"][l], _brute_ids(layers[l], cam, W, H))
    assert r["stats"][1] >= 1
    assert (r["ids"][0] != MISS).mean() > 0.2
    # threads / band split do not change anything
    for nt in (1, 3, 7):
        r2 = oracle.render_view(layers, 0, cam, W, H, num_threads=nt)
        assert np.array_equal(r2["ids"], r["ids"]) and np.array_equal(r2["rgba"], r["rgba"])


# ---- 5(ii). geometric brute force: double-precision ray-triangle intersection ---------------------
def _raycast(layer, cam, W, H):
    """Nearest hit per pixel by Moeller-Trumbore in float64 on the UNSNAPPED vertices.
    Returns ids, depth (z_cam), barycentric-interpolated uv, distance (px) to the nearest projected
    edge of any triangle, gap to the second-nearest hit."""
    R = cam[4:13].astype(np.float64).reshape(3, 3)
    t = cam[13:16].astype(np.float64)
    fx, fy, cx, cy = [float(x) for x in cam[:4]]
    P = layer.positions.astype(np.float64) @ R.T + t          # camera space
    tri = P[layer.indices.astype(np.int64)]                   # [T,3,3]
    uvt = layer.uvs.astype(np.float64)[layer.indices.astype(np.int64)]
    proj = np.stack([fx * tri[..., 0] / tri[..., 2] + cx, fy * tri[..., 1] / tri[..., 2] + cy], -1)
    ids = np.full((H, W), MISS, dtype=np.uint32)
    depth = np.zeros((H, W))
    uv = np.zeros((H, W, 2))
    edge_dist = np.full((H, W), np.inf)
    gap = np.full((H, W), np.inf)
    e1, e2 = tri[:, 1] - tri[:, 0], tri[:, 2] - tri[:, 0]
    for j in range(H):
        for i in range(W):
            d = np.array([(i + 0.5 - cx) / fx, (j + 0.5 - cy) / fy, 1.0])
            pv = np.cross(d, e2)
            det = np.einsum("ij,ij->i", e1, pv)
            ok = np.abs(det) > 1e-14
            inv = np.where(ok, 1.0 / np.where(ok, det, 1.0), 0.0)
            tv = -tri[:, 0]
            u = np.einsum("ij,ij->i", tv, pv) * inv
            qv = np.cross(tv, e1)
            v = (qv @ d) * inv
            tt = np.einsum("ij,ij->i", e2, qv) * inv
            hit = ok & (u >= 0) & (v >= 0) & (u + v <= 1) & (tt > 0)
            s = np.array([i + 0.5, j + 0.5])
            for e in range(3):
                a, b = proj[:, e], proj[:, (e + 1) % 3]
                ab = b - a
                tpar = np.clip(np.einsum("ij,ij->i", s - a, ab) / np.maximum(np.einsum("ij,ij->i", ab, ab), 1e-30), 0, 1)
                dist = np.linalg.norm(a + tpar[:, None] * ab - s, axis=1)
                edge_dist[j, i] = min(edge_dist[j, i], dist.min())
            if hit.any():
                cand = np.where(hit)[0]
                order = cand[np.argsort(tt[cand])]
                w = order[0]
                ids[j, i] = w
                depth[j, i] = tt[w]
                uv[j, i] = (1 - u[w] - v[w]) * uvt[w, 0] + u[w] * uvt[w, 1] + v[w] * uvt[w, 2]
                if len(order) > 1:
                    gap[j, i] = (tt[order[1]] - tt[w]) / tt[w]
    return ids, depth, uv, edge_dist, gap


def test_bruteforce_geometric():
    rng = np.random.default_rng(12)
    W, H = 32, 24
    cam = synth.look_at_camera((0.4, 0.3, -0.6), W, H, 45.0, target=(0, 0, 3.0))
    pos, uv, idx = _soup(rng, 40, size=0.6)
    layer = L(pos, uv, idx, const_tex([0, 0, 0, 0]))
    r = oracle.render_view([layer], 0, cam, W, H, want_qp=True, want_layer_uv=True)
    gid, gdepth, guv, edist, gap = _raycast(layer, cam, W, H)
    safe = (edist > 1 / 64) & (gap > 1e-3)
    assert safe.mean() > 0.5
    assert np.array_equal(r["ids"][0][safe], gid[safe])
    hit = safe & (gid != MISS)
    assert hit.sum() > 100
    # snapping moves vertices by <= 1/512 px: attributes agree to ~1e-3 of their range
    np.testing.assert_allclose(1.0 / r["qp"][0][hit], gdepth[hit], rtol=2e-3)
    np.testing.assert_allclose(r["layer_uv"][0][hit], guv[hit], atol=4e-3)
    # and much better than that on average (a wrong vertex pairing would be O(0.1))
    assert np.abs(r["layer_uv"][0][hit] - guv[hit]).mean() < 3e-4


# ---- 2. single opaque layer == single-surface render (independent pipeline) -------------------------
def _smooth_texture(Ht, Wt, n, rng, opaque=True):
    jj, ii = np.meshgrid((np.arange(Ht) + 0.5) / Ht, (np.arange(Wt) + 0.5) / Wt, indexing="ij")
    tex = np.zeros((Ht, Wt, n, 4), dtype=np.float32)
    for c in range(n):
        for ch in range(4):
            fa, fb, ph = rng.uniform(0.5, 2.0), rng.uniform(0.5, 2.0), rng.uniform(0, 6.28)
            tex[:, :, c, ch] = 0.8 * np.sin(2 * np.pi * (fa * ii + fb * jj) + ph)
    if opaque:
        tex[:, :, 0, 3] = 60000.0          # sigmoid -> exactly 1 (finite in fp16 too)
        tex[:, :, 1:, 3] = 0.0
    return tex


def test_single_opaque_layer_is_single_surface_render():
    import torch
    from scipy.special import expit
    from tests.test_oracle_units import _real_sh_scipy
    rng = np.random.default_rng(13)
    W, H = 40, 30
    cam = synth.look_at_camera((1.2, 0.8, -2.4), W, H, 40.0)
    pos, uv, idx = synth.icosphere_charted(1, 1.0, 64)
    tex = _smooth_texture(64, 64, 9, rng)
    layer = L(pos, uv, idx, tex)
    r = oracle.render_view([layer], 2, cam, W, H)
    gid, _, guv, edist, gap = _raycast(layer, cam, W, H)
    safe = (edist > 1 / 64) & (gid != MISS)
    assert safe.sum() > 200
    assert np.array_equal(r["ids"][0][edist > 1 / 64], gid[edist > 1 / 64])
    # z-buffer + library texture lookup + library SH, written here, not in the oracle
    t = torch.from_numpy(tex.astype(np.float64)).reshape(64, 64, 36).permute(2, 0, 1)[None]
    grid = torch.from_numpy(guv * 2 - 1).reshape(1, H, W, 2)
    coef = torch.nn.functional.grid_sample(t, grid, mode="bilinear", padding_mode="border",
                                           align_corners=False)[0].permute(1, 2, 0).numpy().reshape(H, W, 9, 4)
    R = cam[4:13].astype(np.float64).reshape(3, 3)
    want = np.zeros((H, W, 4))
    for j in range(H):
        for i in range(W):
            d = R.T @ np.array([(i + 0.5 - cam[2]) / cam[0], (j + 0.5 - cam[3]) / cam[1], 1.0])
            want[j, i] = expit(_real_sh_scipy(2, d / np.linalg.norm(d)) @ coef[j, i])
    assert np.all(r["rgba"][..., 3][gid != MISS][:] == 1.0)
    np.testing.assert_allclose(r["rgba"][safe][:, :3], want[safe][:, :3], atol=3e-3)
    assert np.abs(r["rgba"][safe][:, :3] - want[safe][:, :3]).mean() < 2e-4
    # outside the silhouette: background, alpha 0
    out = (gid == MISS) & (edist > 1 / 64)
    assert np.all(r["rgba"][out] == 0)


# ---- 3. alpha = 0 layers are invisible ---------------------------------------------------------------
@pytest.mark.parametrize("dtype", [np.float32, np.float16])
def test_transparent_layers_invisible(dtype):
    sc = synth.make_config(1, width=48, height=48, num_cameras=2, tex_size=32)
    for l in sc.layers:
        l.texture = l.texture.astype(dtype)
    base = oracle.render_scene(sc, [1])[0]
    ghost = np.zeros_like(sc.layers[0].texture)
    ghost[:, :, 0, 3] = -60000.0      # sigmoid -> exactly 0; (-inf would make 0*inf = NaN in the lerp)
    ghost[:, :, :, :3] = 5.0
    pos, uv, idx = synth.icosphere_charted(2, 0.95, 32)
    extra = synth.Layer(pos, uv, idx, ghost)
    for where in (0, 1, 3):
        layers = list(sc.layers)
        layers.insert(where, extra)
        r = oracle.render_view(layers, 1, sc.cameras[1], 48, 48)
        assert np.array_equal(r["rgba"], base["rgba"])


# ---- 4. analytic compositing of constant-colour layers ---------------------------------------------
def test_constant_layers_analytic():
    k = 4
    cols = np.array([[0.9, 0.1, 0.2], [0.2, 0.8, 0.3], [0.1, 0.3, 0.7], [0.6, 0.6, 0.1]])
    alph = np.array([0.3, 0.5, 0.2, 0.9])
    logit = lambda p: np.log(p / (1 - p))
    layers = []
    for l in range(k):
        pos, uv, idx = synth.icosphere_charted(2, 1.0 - 0.15 * l, 16)
        layers.append(L(pos, uv, idx, const_tex(np.concatenate([logit(cols[l]), [logit(alph[l])]]), n=4)))
    W = H = 64
    cam = synth.look_at_camera((0.5, 1.0, 2.8), W, H)
    bg = (0.25, 0.5, 0.75)
    r = oracle.render_view(layers, 1, cam, W, H, t_min=0.0, background=bg)
    cov = r["ids"] != MISS
    # nested silhouettes; all four "rings" present
    for l in range(k - 1):
        assert np.all(cov[l] | ~cov[l + 1])
    assert all(np.any(cov.sum(0) == m) for m in range(k + 1))
    A = alph[:, None, None] * cov
    T = np.concatenate([np.ones((1, H, W)), np.cumprod(1 - A, 0)])
    want_rgb = (cols[:, None, None, :] * (A * T[:-1])[..., None]).sum(0) + T[-1][..., None] * np.asarray(bg)
    np.testing.assert_allclose(r["rgba"][..., :3], want_rgb, atol=1e-12)
    np.testing.assert_allclose(r["rgba"][..., 3], 1 - T[-1], atol=1e-12)
    # SPEC.md:L478 through the whole renderer: red 0.5 over opaque blue
    big = 40.0   # sigmoid(40) = 1 - 4e-18 -> 1.0 in double
    two = [L(layers[0].positions, layers[0].uvs, layers[0].indices, const_tex([big, -big, -big, 0.0], n=4)),
           L(layers[1].positions, layers[1].uvs, layers[1].indices, const_tex([-big, -big, big, big], n=4))]
    r2 = oracle.render_view(two, 1, cam, W, H)
    np.testing.assert_allclose(r2["rgba"][H // 2, W // 2], [0.5, 0.0, 0.5, 1.0], atol=1e-15)


# ---- sorting-free theorem: fixed order == depth-sorted blend on nested shells -----------------------
def test_fixed_order_equals_sorted_blend_on_nested_shells():
    sc = synth.make_config(2, mesh_n=12, width=64, height=64, tex_size=32, num_cameras=3, k=4)
    for v in range(3):
        r = oracle.render_scene(sc, [v], want_qp=True, want_layer_rgba=True, t_min=0.0)[0]
        hit = r["ids"] != MISS
        assert hit.any()
        qp = np.where(hit, r["qp"], -np.inf)
        # the recipe's shells are nested: wherever two layers are hit, the outer one is nearer
        for a in range(sc.k):
            for b in range(a + 1, sc.k):
                both = hit[a] & hit[b]
                assert np.all(qp[a][both] > qp[b][both])
        order = np.argsort(-qp, axis=0, kind="stable")         # nearest first
        lr = np.take_along_axis(r["layer_rgba"], order[..., None], 0)
        lh = np.take_along_axis(hit, order, 0)
        A = lr[..., 3] * lh
        T = np.concatenate([np.ones((1, 64, 64)), np.cumprod(1 - A, 0)])
        rgb = (lr[..., :3] * (A * T[:-1])[..., None]).sum(0)
        np.testing.assert_allclose(r["rgba"][..., :3], rgb, atol=1e-13)
        # negative control: innermost-first order is NOT the sorted blend
        rev = synth.Scene(sc.name, sc.layers[::-1], sc.sh_degree, sc.cameras, sc.width, sc.height)
        rr = oracle.render_scene(rev, [v], t_min=0.0)[0]
        assert np.abs(rr["rgba"] - r["rgba"]).max() > 1e-2


# ---- misc -----------------------------------------------------------------------------------------
def test_early_exit_bound_and_behind_camera():
    sc = synth.make_config(1, width=40, height=40, num_cameras=1, tex_size=32)
    for l in sc.layers:
        l.texture[:, :, 0, 3] += 8.0            # fairly opaque layers so the exit fires
    a = oracle.render_scene(sc, [0], t_min=2.0 ** -6)[0]["rgba"]
    b = oracle.render_scene(sc, [0], t_min=0.0)[0]["rgba"]
    assert np.abs(a - b).max() <= 2.0 ** -6 and np.abs(a - b).max() > 0
    # camera inside the shells looking out / shells behind the camera: triangles are dropped, not clipped
    cam = synth.look_at_camera((0, 0, 3.0), 40, 40, target=(0, 0, 6.0))
    r = oracle.render_view(sc.layers, 1, cam, 40, 40, background=(0.1, 0.2, 0.3))
    assert np.all(r["ids"] == MISS) and r["stats"][0] == 3 * 1280
    assert np.all(r["rgba"] == np.array([0.1, 0.2, 0.3, 0.0]))
    with pytest.raises(ValueError):
        oracle.render_view(sc.layers * 4, 1, cam, 40, 40)      # k = 12 > 9


def test_configs_drop_no_triangles():
    """The recipe keeps every camera outside the shells: no near-plane / guard-band drops (Q12)."""
    sc = synth.make_config(2, mesh_n=10, width=80, height=80, tex_size=16, num_cameras=16)
    for r in oracle.render_scene(sc):
        assert r["stats"][0] == 0
    sc = synth.make_config(5, mesh_n=10, width=96, height=54, tex_size=16, num_cameras=4)
    covs = []
    for r in oracle.render_scene(sc):
        assert r["stats"][0] == 0
        covs.append((r["ids"][0] != MISS).mean())
    assert covs[1] > 0.95 and covs[0] < 0.5        # close-ups fill the frame, far views do not

"""GPU parity: the CUDA path (through the C-ABI) against the CPU oracle on the same seeded inputs.
Bar (BASELINE.json north_star): coverage and per-layer triangle IDs BIT-EXACT, RGBA max abs error
<= 1e-4.  Sizes here are ones the oracle finishes in seconds and that still span many tiles and a
ragged tail; the full BASELINE.json sizes are in test_gpu_configs.py."""
import types

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-4


@pytest.fixture(scope="module", params=["direct", "tiled"])
def env(request):
    """Every test runs on both raster paths: the default triangle-parallel one (64-bit max keys in HBM/L2)
    and the per-tile one behind VS_FLAG_TILED_PATH (binning + shared-memory keys)."""
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    import oracle
    from paper_2409_02482_b200 import binding, synth
    binding.load_library()
    return types.SimpleNamespace(torch=torch, oracle=oracle, binding=binding, synth=synth,
                                 path_flags=binding.VS_FLAG_TILED_PATH if request.param == "tiled" else 0)


def gpu_render(env, sc, views, flags=0, t_min=None, background=None, views_per_chunk=0, want_ids=True):
    b = env.binding
    r = b.Renderer(sc)
    p = b.make_params(sc.width, sc.height, sc.near_plane, sc.t_min if t_min is None else t_min,
                      sc.background if background is None else background, flags | env.path_flags, views_per_chunk)
    rgba, ids = r.render(sc.cameras[list(views)], p, want_ids=want_ids)
    env.torch.cuda.synchronize()
    stats = r.stats()
    out = rgba.cpu().numpy(), (ids.cpu().numpy().view(np.uint32) if want_ids else None), stats
    r.close()
    return out


def check_against_oracle(env, sc, views, attenuation=False, **kw):
    if attenuation:
        kw["flags"] = kw.get("flags", 0) | env.binding.VS_FLAG_ATTENUATION
    rgba, ids, stats = gpu_render(env, sc, views, **kw)
    okw = {"attenuation": True} if attenuation else {}
    if "t_min" in kw and kw["t_min"] is not None:
        okw["t_min"] = kw["t_min"]
    if "background" in kw and kw["background"] is not None:
        okw["background"] = kw["background"]
    worst = 0.0
    for n, v in enumerate(views):
        ref = env.oracle.render_scene(sc, [v], **okw)[0]
        assert np.array_equal(ids[n], ref["ids"]), "triangle ids differ in view %d: %d pixels" % (
            v, int((ids[n] != ref["ids"]).sum()))
        err = float(np.abs(rgba[n].astype(np.float64) - ref["rgba"]).max())
        worst = max(worst, err)
        assert err <= TOL, "view %d: max abs rgba error %.3e" % (v, err)
        assert stats["dropped_triangles"] == 0 or ref["stats"][0] > 0
    return worst, rgba, ids


def test_config1_all_views(env):
    sc = env.synth.make_config(1)
    worst, rgba, ids = check_against_oracle(env, sc, range(4))
    assert (ids != env.binding.MISS).mean() > 0.5
    print("C1 worst rgba err %.3e" % worst)


def test_config1_reference_path_agrees(env):
    sc = env.synth.make_config(1)
    a = gpu_render(env, sc, [0, 2])
    b = gpu_render(env, sc, [0, 2], flags=env.binding.VS_FLAG_REFERENCE_PATH)
    assert np.array_equal(a[1], b[1])
    assert np.abs(a[0] - b[0]).max() <= 2e-6
    check_against_oracle(env, sc, [1], flags=env.binding.VS_FLAG_REFERENCE_PATH)


@pytest.mark.parametrize("cfg,kw", [
    (2, dict(mesh_n=40, width=333, height=250, tex_size=256, num_cameras=4)),          # fp16 deg 2, ragged tiles
    (3, dict(mesh_n=48, width=400, height=225, tex_size=256, num_cameras=3, k=7)),     # fp16 deg 3, low alpha
    (4, dict(mesh_n=64, width=480, height=270, tex_size=512, num_cameras=5, k=9)),     # fp16 deg 3, k = 9
    (5, dict(mesh_n=120, width=384, height=216, tex_size=512, num_cameras=4, k=9)),    # sub-pixel tris + close-ups
])
def test_reduced_configs(env, cfg, kw):
    sc = env.synth.make_config(cfg, **kw)
    worst, _, ids = check_against_oracle(env, sc, range(len(sc.cameras)), views_per_chunk=2)
    print("C%d reduced worst rgba err %.3e, coverage %.2f" % (cfg, worst, (ids != env.binding.MISS).mean()))


# ---- transparency attenuation behind VS_FLAG_ATTENUATION ----
def test_attenuation_config1(env):
    sc = env.synth.make_config(1)
    worst, rgba, ids = check_against_oracle(env, sc, range(4), attenuation=True)
    plain = gpu_render(env, sc, range(4))
    assert np.array_equal(plain[1], ids)                       # coverage does not depend on the flag
    hit = (ids != env.binding.MISS).any(axis=1)
    assert np.all(rgba[..., 3][hit] <= plain[0][..., 3][hit])  # alpha_w <= 1 can only lower the alpha
    assert (rgba[..., 3][hit] < plain[0][..., 3][hit] - 1e-3).mean() > 0.05   # and does so near the silhouettes
    # the brute-force kernel applies the same weight
    check_against_oracle(env, sc, [1], attenuation=True, flags=env.binding.VS_FLAG_REFERENCE_PATH)
    print("C1 attenuated worst rgba err %.3e" % worst)


@pytest.mark.parametrize("cfg,kw", [
    (3, dict(mesh_n=48, width=400, height=225, tex_size=256, num_cameras=3, k=7)),     # fp16 deg 3, low alpha
    (5, dict(mesh_n=120, width=384, height=216, tex_size=512, num_cameras=4, k=9)),    # sub-pixel tris + close-ups
])
def test_attenuation_reduced_configs(env, cfg, kw):
    sc = env.synth.make_config(cfg, **kw)
    worst, _, _ = check_against_oracle(env, sc, range(len(sc.cameras)), attenuation=True, views_per_chunk=2)
    check_against_oracle(env, sc, [0], attenuation=True, t_min=2.0 ** -6, background=(0.3, 0.1, 0.2))
    print("C%d reduced, attenuated: worst rgba err %.3e" % (cfg, worst))


def test_attenuation_degenerate_and_big_triangles(env):
    s = env.synth
    rng = np.random.default_rng(7)
    # tilted big quad + a triangle whose world area is zero (its normal is 0 -> alpha_w = 0; it covers nothing anyway)
    pos = np.array([[-2, -2, 3], [2, -2, 5], [2, 2, 5], [-2, 2, 3], [0, 0, 3.5]], np.float32)
    uv = np.array([[0, 0], [1, 0], [1, 1], [0, 1], [0.5, 0.5]], np.float32)
    idx = np.array([[0, 1, 2], [0, 2, 3], [0, 0, 1], [2, 1, 4]], np.uint32)
    tex = rng.normal(0, 0.5, (32, 32, 4, 4)).astype(np.float32)
    sc = s.Scene("att", [s.Layer(pos, uv, idx, tex)], 1,
                 np.stack([s.look_at_camera((0.3, 0.2, -1.0), 150, 100, target=(0, 0, 4.0))]), 150, 100)
    check_against_oracle(env, sc, [0], attenuation=True)


# ---- the paper's banded 8-bit mixed-resolution textures ----
def test_banded_config1(env):
    sc = env.synth.make_config(1, banded=True)
    worst, rgba, ids = check_against_oracle(env, sc, range(4))
    assert (ids != env.binding.MISS).mean() > 0.5
    # same geometry as the float C1: identical coverage
    plain = gpu_render(env, env.synth.make_config(1), range(4))
    assert np.array_equal(plain[1], ids)
    print("C1 banded worst rgba err %.3e" % worst)


@pytest.mark.parametrize("cfg,kw", [
    (2, dict(mesh_n=40, width=333, height=250, tex_size=256, num_cameras=4)),          # deg 2, ragged tiles
    (4, dict(mesh_n=64, width=480, height=270, tex_size=512, num_cameras=5, k=9)),     # deg 3, k = 9, bands 512..64
    (5, dict(mesh_n=120, width=384, height=216, tex_size=512, num_cameras=4, k=9)),    # sub-pixel tris + close-ups
])
def test_banded_reduced_configs(env, cfg, kw):
    sc = env.synth.make_config(cfg, banded=True, **kw)
    worst, _, ids = check_against_oracle(env, sc, range(len(sc.cameras)), views_per_chunk=2)
    check_against_oracle(env, sc, [1], attenuation=True, t_min=2.0 ** -6, background=(0.3, 0.1, 0.2))
    print("C%d reduced, banded: worst rgba err %.3e, coverage %.2f" % (cfg, worst, (ids != env.binding.MISS).mean()))


@pytest.mark.parametrize("deg", [0, 1, 2, 3])
def test_banded_formats_and_odd_sizes(env, deg):
    """Every degree; bands of unrelated, non-square sizes (incl. 1x1), full-range white-noise bytes, a range other than
    the paper's [-15, 15]."""
    rng = np.random.default_rng(11 + deg)
    sc = env.synth.make_config(1, width=96, height=80, num_cameras=2, banded=True)
    sizes = [(48, 64), (7, 5), (1, 1), (33, 2)]
    for ly in sc.layers:
        ly.band_textures = [rng.integers(0, 256, size=(sizes[b][0], sizes[b][1], 2 * b + 1, 4), dtype=np.uint8)
                            for b in range(deg + 1)]
    sc.sh_degree = deg
    sc.v_range = (-3.0, 2.0)
    check_against_oracle(env, sc, [0, 1])


def test_banded_host_descriptors_and_errors(env):
    b, torch = env.binding, env.torch
    sc = env.synth.make_config(2, mesh_n=24, width=160, height=120, tex_size=64, num_cameras=3, banded=True)
    dev_rgba, dev_ids, _ = gpu_render(env, sc, range(3))
    h = b.vs_scene_create_banded(sc.layers, sc.sh_degree, *sc.v_range)        # numpy arrays: VS_MEM_HOST
    out = torch.empty((3, 120, 160, 4), dtype=torch.float32).pin_memory()
    ids = torch.empty((3, sc.k, 120, 160), dtype=torch.int32).pin_memory()
    b.vs_render_host(h, sc.cameras, b.make_params(160, 120, flags=env.path_flags), out, ids)
    assert np.array_equal(out.numpy(), dev_rgba) and np.array_equal(ids.numpy().view(np.uint32), dev_ids)
    b.vs_scene_destroy(h)
    # the brute-force kernel reads the banded format too and agrees with the fast path
    ref = gpu_render(env, sc, [0, 2], flags=b.VS_FLAG_REFERENCE_PATH)
    assert np.array_equal(ref[1], dev_ids[[0, 2]]) and np.abs(ref[0] - dev_rgba[[0, 2]]).max() <= 2e-6
    with pytest.raises(b.VsError) as e:
        b.vs_scene_create_banded(sc.layers, sc.sh_degree, float("nan"), 15.0)
    assert e.value.status == b.VS_ERR_INVALID_ARG


# ---- per-layer render buffers through vs_render_aov ----
def check_aov(env, sc, views, attenuation=False, t_min=None, views_per_chunk=0, give_ids=True):
    b, torch = env.binding, env.torch
    flags = env.path_flags | (b.VS_FLAG_ATTENUATION if attenuation else 0)
    p = b.make_params(sc.width, sc.height, sc.near_plane, sc.t_min if t_min is None else t_min, sc.background, flags, views_per_chunk)
    r = b.Renderer(sc)
    B, k, H, W = len(views), sc.k, sc.height, sc.width
    dev = lambda *shape, dt=torch.float32: torch.full(shape, 7, dtype=dt, device="cuda")
    out, ids = dev(B, H, W, 4), dev(B, k, H, W, dt=torch.int32) if give_ids else None
    lrgba, luv, lnrm = dev(B, k, H, W, 4), dev(B, k, H, W, 2), dev(B, k, H, W, 3)
    b.vs_render_aov(r.handle, sc.cameras[list(views)], p, out, ids, lrgba, luv, lnrm)
    torch.cuda.synchronize()
    plain, _ = r.render(sc.cameras[list(views)], p)
    torch.cuda.synchronize()
    assert torch.equal(plain, out), "vs_render_aov and vs_render images differ"
    r.close()
    okw = dict(want_layer_rgba=True, want_layer_uv=True, want_layer_normal=True, attenuation=attenuation)
    if t_min is not None:
        okw["t_min"] = t_min
    for n, v in enumerate(views):
        ref = env.oracle.render_scene(sc, [v], **okw)[0]
        if give_ids:
            assert np.array_equal(ids[n].cpu().numpy().view(np.uint32), ref["ids"])
        assert np.abs(out[n].cpu().numpy() - ref["rgba"]).max() <= TOL
        assert np.abs(lrgba[n].cpu().numpy() - ref["layer_rgba"]).max() <= TOL
        assert np.abs(luv[n].cpu().numpy() - ref["layer_uv"]).max() <= 1e-5
        assert np.abs(lnrm[n].cpu().numpy() - ref["layer_normal"]).max() <= 1e-6
    return lrgba, luv, lnrm


def test_aov_config1(env):
    sc = env.synth.make_config(1)
    lrgba, luv, lnrm = check_aov(env, sc, range(4), views_per_chunk=3)
    assert float(luv.min()) >= 0.0 and float(luv.max()) <= 1.0            # SPEC.md:L503 "UV buffer values in [0,1]^2"
    check_aov(env, sc, [1], attenuation=True, give_ids=False)


def test_aov_early_exit_layers_still_filled(env):
    sc = env.synth.make_config(1, width=100, height=60, num_cameras=1, tex_size=64)
    for ly in sc.layers:
        ly.texture[:, :, 0, 3] += 12.0                                       # near-opaque: compositing stops after layer 0
    lrgba, _, _ = check_aov(env, sc, [0], t_min=2.0 ** -6)
    assert float(lrgba[0, 2, ..., 3].max()) > 0.99                           # ... the innermost layer's buffer is filled anyway


@pytest.mark.parametrize("banded", [False, True])
def test_aov_reduced_config4(env, banded):
    sc = env.synth.make_config(4, mesh_n=64, width=480, height=270, tex_size=512, num_cameras=3, k=9, banded=banded)
    check_aov(env, sc, range(3), attenuation=True, views_per_chunk=2)


# ---- backward pass to the texels through vs_render_backward ----
def check_backward(env, sc, views, attenuation=False, t_min=None, background=None, views_per_chunk=0):
    """GPU gradient textures (fp32 atomics, any order) against the oracle's fp64 ones: max abs error <= 1e-4 of the
    largest gradient magnitude of the layer + exact zeros where the oracle has exact zeros.  Both backward kernels are
    checked: the default k_shade<BWD> (k_shade's octet / tensor-core forward pass + recurrence + scatter) and the plain
    k_backward (VS_FLAG_PLAIN_BACKWARD)."""
    if env.path_flags:
        pytest.skip("vs_render_backward runs on the direct raster path only")
    b, torch = env.binding, env.torch
    rng = np.random.default_rng(21)
    B, H, W = len(views), sc.height, sc.width
    g = rng.normal(size=(B, H, W, 4)).astype(np.float32)
    t_min = sc.t_min if t_min is None else t_min
    background = sc.background if background is None else background
    want = None
    worst = 0.0
    for kernel_flag in (0, b.VS_FLAG_PLAIN_BACKWARD):
        p = b.make_params(W, H, sc.near_plane, t_min, background, (b.VS_FLAG_ATTENUATION if attenuation else 0) | kernel_flag,
                          views_per_chunk)
        r = b.Renderer(sc)
        grads = [torch.zeros(ly.texture.shape, dtype=torch.float32, device="cuda") for ly in sc.layers]
        b.vs_render_backward(r.handle, sc.cameras[list(views)], p, torch.from_numpy(g).cuda(), grads)
        torch.cuda.synchronize()
        # the scene is untouched by the backward call: a forward render afterwards still matches the oracle
        p_fwd = b.make_params(W, H, sc.near_plane, t_min, background, b.VS_FLAG_ATTENUATION if attenuation else 0, views_per_chunk)
        rgba, ids = r.render(sc.cameras[list(views)], p_fwd, want_ids=True)
        torch.cuda.synchronize()
        r.close()
        if want is None:
            for n, v in enumerate(views):
                ref = env.oracle.render_scene(sc, [v], t_min=t_min, background=background, attenuation=attenuation)[0]
                assert np.array_equal(ids[n].cpu().numpy().view(np.uint32), ref["ids"])
                want = env.oracle.render_backward(sc.layers, sc.sh_degree, sc.cameras[v], W, H, ref["ids"], g[n].astype(np.float64),
                                                  want, near_plane=sc.near_plane, t_min=t_min, background=background,
                                                  attenuation=attenuation)
        for l in range(sc.k):
            got = grads[l].cpu().numpy().astype(np.float64)
            scale = max(np.abs(want[l]).max(), 1e-30)
            err = np.abs(got - want[l]).max() / scale
            worst = max(worst, err)
            assert err <= 1e-4, "layer %d: relative gradient error %.3e (kernel flag %d)" % (l, err, kernel_flag)
            assert np.all(got[want[l] == 0.0] == 0.0)
    return worst, want


def test_backward_config1(env):
    sc = env.synth.make_config(1)
    worst, want = check_backward(env, sc, range(4), views_per_chunk=3)
    assert all(np.abs(w).max() > 1e-2 for w in want)
    check_backward(env, sc, [2], attenuation=True, background=(0.3, 0.6, 0.1), t_min=0.0)
    print("C1 backward: worst relative gradient error %.3e" % worst)


def test_backward_reduced_config4_fp16(env):
    sc = env.synth.make_config(4, mesh_n=48, width=320, height=180, tex_size=128, num_cameras=3, k=9)
    worst, _ = check_backward(env, sc, range(3), views_per_chunk=2)
    print("C4 reduced backward: worst relative gradient error %.3e" % worst)


def test_backward_early_exit_and_errors(env):
    b, torch = env.binding, env.torch
    sc = env.synth.make_config(1, width=100, height=60, num_cameras=1, tex_size=64)
    for ly in sc.layers:
        ly.texture[:, :, 0, 3] += 60.0                      # opaque outer layer: nothing behind it gets a gradient
    _, want = check_backward(env, sc, [0], t_min=2.0 ** -6)
    assert np.all(want[1] == 0.0) and np.all(want[2] == 0.0) and np.abs(want[0]).max() > 1e-3
    if not env.path_flags:
        banded = env.synth.make_config(1, width=32, height=32, num_cameras=1, banded=True)
        r = b.Renderer(banded)
        with pytest.raises(b.VsError) as e:
            b.vs_render_backward(r.handle, banded.cameras, b.make_params(32, 32), torch.zeros((1, 32, 32, 4), device="cuda"),
                                 [torch.zeros((1,), device="cuda")] * 3)
        assert e.value.status == b.VS_ERR_UNSUPPORTED
        r.close()


def test_backward_degenerate_footprints(env):
    """1x1 and 2x2 textures: all four texels of a footprint coincide (clamped) and whole rows of pixels share one footprint,
    the extreme case of the run merging in k_shade<BWD>; a 3-texel-wide texture under a 60-pixel object for long runs."""
    sc = env.synth.make_config(1, width=64, height=40, num_cameras=2, tex_size=16)
    sc.layers[0].texture = sc.layers[0].texture[:3, :3].copy()
    sc.layers[1].texture = sc.layers[1].texture[:2, :2].copy()
    sc.layers[2].texture = sc.layers[2].texture[:1, :1].copy()
    worst, want = check_backward(env, sc, [0, 1])
    assert all(np.abs(w).max() > 1e-3 for w in want)


def test_determinism_and_chunking(env):
    sc = env.synth.make_config(2, mesh_n=30, width=200, height=150, tex_size=128, num_cameras=6)
    a = gpu_render(env, sc, range(6), views_per_chunk=1)
    b = gpu_render(env, sc, range(6), views_per_chunk=4)
    c = gpu_render(env, sc, range(6))
    for x in (b, c):
        assert np.array_equal(a[0], x[0]) and np.array_equal(a[1], x[1])


def test_surface_order_is_a_permutation_of_screen_order(env):
    """The default shading order (the (view, tile) pairs of a pass sorted by where on the object they look,
    vs_kernels_order.cu) changes scheduling only: images and ids are bit-identical to VS_FLAG_SCREEN_ORDER, for forward,
    AOV-less backward and every chunking (a lost or doubled entry of the sorted list would leave a tile unshaded)."""
    b = env.binding
    sc = env.synth.make_config(4, mesh_n=40, width=333, height=217, tex_size=128, num_cameras=7)
    ref = gpu_render(env, sc, range(7), flags=b.VS_FLAG_SCREEN_ORDER)
    for chunk in (0, 1, 3, 7):
        got = gpu_render(env, sc, range(7), views_per_chunk=chunk)
        assert np.array_equal(ref[0], got[0]) and np.array_equal(ref[1], got[1])
    # a scene whose box is degenerate in one axis (a single quad), and an empty view (camera looking away)
    quad = env.synth.make_config(1, width=90, height=70, num_cameras=3, tex_size=32)
    for ly in quad.layers:
        ly.positions[:, 2] = 0.25
    a = gpu_render(env, quad, range(3), flags=b.VS_FLAG_SCREEN_ORDER)
    c = gpu_render(env, quad, range(3))
    assert np.array_equal(a[0], c[0]) and np.array_equal(a[1], c[1])


@pytest.mark.parametrize("dtype,deg", [(np.float32, 0), (np.float16, 0), (np.float16, 1), (np.float16, 2), (np.float32, 2), (np.float32, 3)])
def test_all_texture_formats(env, dtype, deg):
    rng = np.random.default_rng(5)
    sc = env.synth.make_config(1, width=96, height=80, num_cameras=2, tex_size=64)
    n = (deg + 1) ** 2
    for ly in sc.layers:
        ly.texture = rng.normal(0, 0.5, size=(48, 64, n, 4)).astype(dtype)     # non-square texture too
    sc.sh_degree = deg
    check_against_oracle(env, sc, [0, 1])
    if not env.path_flags:   # every (format, degree) instantiation of the backward kernels too
        check_backward(env, sc, [1])


def test_far_scene_takes_the_library_division(env):
    """k_raster_direct hoists the reciprocal of the triangle's area out of its per-sample loop (csrc/vs_div.cuh) only while
    1/w stays inside [1e-20, 1e20]; a scene 2^70 units away (1/w ~ 3e-22) must take the library division instead and still
    give the oracle's ids.  Scaling by a power of two is exact in fp32, so the images are those of the unscaled scene."""
    sc = env.synth.make_config(1, width=96, height=72, num_cameras=2, tex_size=64)
    near = gpu_render(env, sc, [0, 1])
    scale = np.float32(2.0 ** 70)
    for ly in sc.layers:
        ly.positions = (ly.positions * scale).astype(np.float32)
    sc.cameras = sc.cameras.copy()
    sc.cameras[:, 13:16] *= scale
    worst, rgba, ids = check_against_oracle(env, sc, [0, 1])
    assert (ids != env.binding.MISS).mean() > 0.3
    assert np.array_equal(ids, near[1]) and np.allclose(rgba, near[0], rtol=0.0, atol=1e-6)


def test_edge_cases(env):
    s = env.synth
    # early exit with opaque-ish layers, non-zero background, t_min variants
    sc = s.make_config(1, width=100, height=60, num_cameras=1, tex_size=64)
    for ly in sc.layers:
        ly.texture[:, :, 0, 3] += 12.0
    check_against_oracle(env, sc, [0], t_min=2.0 ** -6, background=(0.2, 0.4, 0.6))
    check_against_oracle(env, sc, [0], t_min=0.0)
    # exactly opaque / exactly transparent layers (fp16 +-60000)
    sc = s.make_config(2, mesh_n=16, width=90, height=70, tex_size=64, num_cameras=2, k=3)
    sc.layers[0].texture[:, :, 0, 3] = -60000.0
    sc.layers[1].texture[:, :, 0, 3] = 60000.0
    worst, rgba, ids = check_against_oracle(env, sc, [0, 1])
    assert np.all(rgba[..., 3][ids[:, 1] != env.binding.MISS] == 1.0)
    # a shell with no triangles, a 1x1 texture, k = 1, 1x1 image, image not a multiple of the tile
    sc = s.make_config(1, width=17, height=33, num_cameras=1, tex_size=16)
    sc.layers[1].indices = np.zeros((0, 3), np.uint32)
    sc.layers[2].texture = sc.layers[2].texture[:1, :1].copy()
    check_against_oracle(env, sc, [0])
    one = s.Scene("k1", sc.layers[:1], 1, sc.cameras, 1, 1)
    check_against_oracle(env, one, [0])
    # every triangle behind the camera: dropped, background everywhere
    cam = s.look_at_camera((0, 0, 3.0), 64, 48, target=(0, 0, 6.0))
    sc = s.make_config(1, width=64, height=48, num_cameras=1, tex_size=16)
    sc.cameras = cam[None]
    rgba, ids, stats = gpu_render(env, sc, [0], background=(0.1, 0.2, 0.3))
    assert np.all(ids == env.binding.MISS) and stats["dropped_triangles"] == 3 * 1280
    assert np.allclose(rgba, np.array([0.1, 0.2, 0.3, 0.0], np.float32))
    # big triangles (warp-cooperative path) + degenerate + duplicate triangles, UVs outside [0,1]
    rng = np.random.default_rng(3)
    pos = np.array([[-2, -2, 4], [2, -2, 4], [2, 2, 4], [-2, 2, 4], [0, 0, 3.5]], np.float32)
    uv = np.array([[-0.3, -0.2], [1.4, 0], [1.2, 1.3], [0, 1], [0.5, 0.5]], np.float32)
    idx = np.array([[0, 1, 2], [0, 2, 3], [0, 1, 4], [0, 0, 1], [0, 1, 2]], np.uint32)
    tex = rng.normal(0, 0.5, (32, 32, 4, 4)).astype(np.float32)
    big = s.Scene("big", [s.Layer(pos, uv, idx, tex)], 1,
                  np.stack([s.look_at_camera((0.3, 0.2, -1.0), 150, 100, target=(0, 0, 4.0))]), 150, 100)
    check_against_oracle(env, big, [0])
    rgba, ids, stats = gpu_render(env, big, [0])
    assert stats["degenerate_triangles"] == 1


def test_invalid_arguments_are_rejected(env):
    b, torch = env.binding, env.torch
    sc = env.synth.make_config(1, width=32, height=32, num_cameras=1, tex_size=16)
    sc.layers[0].indices = sc.layers[0].indices.copy()
    sc.layers[0].indices[5, 1] = 10 ** 6
    with pytest.raises(b.VsError) as e:
        b.Renderer(sc)
    assert e.value.status == b.VS_ERR_INVALID_ARG
    sc = env.synth.make_config(1, width=32, height=32, num_cameras=1, tex_size=16)
    sc.layers[1].positions = sc.layers[1].positions.copy()
    sc.layers[1].positions[7, 2] = np.nan
    with pytest.raises(b.VsError):
        b.Renderer(sc)
    sc = env.synth.make_config(1, width=32, height=32, num_cameras=1, tex_size=16)
    r = b.Renderer(sc)
    out = torch.empty((1, 32, 32, 4), device="cuda")
    with pytest.raises(b.VsError):
        b.vs_render(r.handle, sc.cameras, b.make_params(32, 32, near_plane=0.0), out)
    bad = sc.cameras.copy()
    bad[0, 5] = np.inf
    with pytest.raises(b.VsError):
        b.vs_render(r.handle, bad, b.make_params(32, 32), out)
    r.close()


def test_host_path_matches_device_path(env):
    b, torch = env.binding, env.torch
    sc = env.synth.make_config(2, mesh_n=24, width=160, height=120, tex_size=64, num_cameras=5)
    dev_rgba, dev_ids, _ = gpu_render(env, sc, range(5))
    # host descriptors (numpy arrays) for scene creation + host outputs
    h = b.vs_scene_create(sc.layers, sc.sh_degree)
    out = torch.empty((5, 120, 160, 4), dtype=torch.float32).pin_memory()
    ids = torch.empty((5, sc.k, 120, 160), dtype=torch.int32).pin_memory()
    b.vs_render_host(h, sc.cameras, b.make_params(160, 120, views_per_chunk=2), out, ids)
    assert np.array_equal(out.numpy(), dev_rgba) and np.array_equal(ids.numpy().view(np.uint32), dev_ids)
    pageable = np.empty((5, 120, 160, 4), np.float32)
    b.vs_render_host(h, sc.cameras, b.make_params(160, 120), pageable)
    assert np.array_equal(pageable, dev_rgba)
    b.vs_scene_destroy(h)


def test_census_counters_match_the_oracle(env):
    """The numerator of every roofline figure ("counted, not assumed"): VS_FLAG_COUNT_TEXELS' shaded
    fragments and unique 2x2-footprint texels against the oracle's footprint census (pinned in tests/test_oracle_census.py)
    on reduced C2 and C4 scenes and on C1, several views per call (the texel count is per view, summed over the views).
    Fragments must agree exactly; texels to 1e-4 relative (fp32-vs-fp64 texel coordinate at a texel boundary), and with an
    early exit (C1 with an opaque middle layer) the fragment count may differ by the knife-edge pixels only."""
    b = env.binding
    cases = [(env.synth.make_config(2, mesh_n=31, width=200, height=200, tex_size=256, num_cameras=3), [0, 1, 2], None),
             (env.synth.make_config(4, mesh_n=40, width=320, height=180, tex_size=256, num_cameras=3), [0, 2], None),
             (env.synth.make_config(1), [0, 1, 2, 3], None),
             (env.synth.make_config(1), [1, 3], 2.0 ** -6)]
    for n, (sc, views, t_min) in enumerate(cases):
        if t_min is not None:
            sc.layers[1].texture[:, :, 0, 3] += 30.0       # opaque middle layer: the innermost one is never composited
        tm = sc.t_min if t_min is None else t_min
        _, _, stats = gpu_render(env, sc, views, flags=b.VS_FLAG_COUNT_TEXELS, t_min=tm, want_ids=False)
        frags = texels = 0
        for v in views:
            ref = env.oracle.render_scene(sc, [v], want_layer_rgba=True, want_layer_uv=True, t_min=tm)[0]
            f, t, _ = env.oracle.count_footprints(sc.layers, sc.width, sc.height, ref, t_min=tm)
            frags += f
            texels += t
        assert frags > 1000 and texels > 1000
        assert stats["shaded_fragments"] == frags, "case %d: %d fragments on the GPU, %d in the oracle" % (n, stats["shaded_fragments"], frags)
        assert abs(stats["unique_texels"] - texels) <= max(2, 1e-4 * texels), \
            "case %d: %d unique texels on the GPU, %d in the oracle" % (n, stats["unique_texels"], texels)
        if t_min is not None:
            hits = sum(int((env.oracle.render_scene(sc, [v], t_min=tm)[0]["ids"] != env.oracle.MISS).sum()) for v in views)
            assert frags < hits, "the early exit must have removed fragments"


def test_every_output_is_written_in_bounds(env):
    """Stand-in for compute-sanitizer memcheck (closed on this pool): every caller-owned output of every entry point is a
    window inside a larger tensor filled with a sentinel; after the calls the margins must be untouched.  The library's own
    scratch buffers carry guard bands that vs_query_last_render (Renderer.stats) verifies.  Odd image and texture sizes, so
    that partial tiles, partial warps and the last texel rows are all exercised."""
    b, torch = env.binding, env.torch
    PAD = 4096
    for cfg, kw in ((1, dict(width=101, height=67, num_cameras=3, tex_size=37)),
                    (4, dict(mesh_n=14, width=77, height=45, tex_size=33, num_cameras=3))):
        sc = env.synth.make_config(cfg, **kw)
        B, W, H, k = len(sc.cameras), sc.width, sc.height, sc.k
        r = b.Renderer(sc)

        def window(n, dtype, fill):
            big = torch.full((n + 2 * PAD,), fill, dtype=dtype, device="cuda")
            return big, big[PAD:PAD + n]

        def intact(big, n, fill):
            return bool((big[:PAD] == fill).all()) and bool((big[PAD + n:] == fill).all())

        bufs = {"rgba": window(B * H * W * 4, torch.float32, 12345.0), "ids": window(B * k * H * W, torch.int32, 0x5A5A5A5A),
                "lrgba": window(B * k * H * W * 4, torch.float32, 12345.0), "luv": window(B * k * H * W * 2, torch.float32, 12345.0),
                "lnrm": window(B * k * H * W * 3, torch.float32, 12345.0)}
        for flags in (env.path_flags, env.path_flags | b.VS_FLAG_ATTENUATION, env.path_flags | b.VS_FLAG_COUNT_TEXELS):
            for chunk in (0, 1, 2):
                p = b.make_params(W, H, sc.near_plane, sc.t_min, sc.background, flags, chunk)
                b.vs_render(r.handle, sc.cameras, p, bufs["rgba"][1], bufs["ids"][1])
                b.vs_render_aov(r.handle, sc.cameras, p, bufs["rgba"][1], bufs["ids"][1], bufs["lrgba"][1], bufs["luv"][1], bufs["lnrm"][1])
                torch.cuda.synchronize()
                r.stats()           # raises if a scratch guard band was overwritten
        for name, (big, win) in bufs.items():
            fill = 0x5A5A5A5A if name == "ids" else 12345.0
            assert intact(big, win.numel(), fill), "%s: written outside [0, %d)" % (name, win.numel())
            assert not bool((win == fill).any()) or name != "rgba", "rgba: not every pixel was written"
        if not env.path_flags:
            gbig, gwin = [], []
            for ly in sc.layers:
                n = int(np.prod(ly.texture.shape))
                big = torch.full((n + 2 * PAD,), 777.0, dtype=torch.float32, device="cuda")
                big[PAD:PAD + n] = 0.0
                gbig.append(big)
                gwin.append(big[PAD:PAD + n].view(ly.texture.shape))
            g = torch.ones((B, H, W, 4), dtype=torch.float32, device="cuda")
            b.vs_render_backward(r.handle, sc.cameras, b.make_params(W, H, sc.near_plane, sc.t_min, sc.background), g, gwin)
            torch.cuda.synchronize()
            r.stats()
            for l, big in enumerate(gbig):
                assert intact(big, gwin[l].numel(), 777.0), "gradient texture %d: written out of bounds" % l
                assert float(gwin[l].abs().max()) > 0.0
        r.close()


def _with_vertex_normals(sc, which):
    """Smooth (radial, slightly sheared so that they are NOT the facet normals) per-vertex normals on the layers in `which`."""
    for l, ly in enumerate(sc.layers):
        if l in which:
            n = ly.positions.astype(np.float64)
            n = n / np.linalg.norm(n, axis=1, keepdims=True) + np.array([0.15, -0.1, 0.05]) * n[:, [1]]
            ly.normals = (1.7 * n).astype(np.float32)          # deliberately not unit length
    return sc


@pytest.mark.parametrize("banded", [False, True])
def test_per_vertex_normals_attenuation(env, banded):
    """SURVEY.md §8(f) NEXT-2, the optional per-vertex normals (vs_scene_set_vertex_normals): layers 0 and 2 carry normals,
    layer 1 keeps its face normals; image, per-layer opacity / normal buffers and the backward pass against the oracle."""
    sc = _with_vertex_normals(env.synth.make_config(1, width=120, height=90, num_cameras=2, banded=banded), {0, 2})
    worst, _, _ = check_against_oracle(env, sc, [0, 1], attenuation=True)
    check_aov(env, sc, [0, 1], attenuation=True)
    # the normals matter: the same scene without them renders differently
    plain = env.synth.make_config(1, width=120, height=90, num_cameras=2, banded=banded)
    a, _, _ = gpu_render(env, sc, [0], flags=env.binding.VS_FLAG_ATTENUATION, want_ids=False)
    c, _, _ = gpu_render(env, plain, [0], flags=env.binding.VS_FLAG_ATTENUATION, want_ids=False)
    assert np.abs(a - c).max() > 1e-3
    if not banded:
        check_backward(env, sc, [0, 1], attenuation=True)
    print("per-vertex normals (%s): worst rgba err %.3e" % ("banded" if banded else "float", worst))


def test_per_vertex_normals_reduced_config4(env):
    sc = _with_vertex_normals(env.synth.make_config(4, mesh_n=40, width=320, height=180, tex_size=256, num_cameras=2), set(range(9)))
    worst, _, _ = check_against_oracle(env, sc, [0, 1], attenuation=True)
    print("per-vertex normals, reduced C4: worst rgba err %.3e" % worst)


def test_asynchronous_calls_on_two_streams_and_threads(env):
    """vs_render is asynchronous and calls on different streams are legal.  Two batches are rendered on two
    streams without any synchronisation in between (and once more from two host threads): the images must be those of serial
    calls bit for bit, also under VS_FLAG_OVERLAP (S1-S4 of the next chunk on the internal stream) and with zero cameras."""
    import threading
    b, torch = env.binding, env.torch
    sc = env.synth.make_config(2, mesh_n=30, width=200, height=150, tex_size=128, num_cameras=6)
    r = b.Renderer(sc)
    W, H = sc.width, sc.height
    p = b.make_params(W, H, sc.near_plane, sc.t_min, sc.background, env.path_flags, 2)
    sets = [sc.cameras[:3], sc.cameras[3:]]
    serial = []
    for cams in sets:
        out, ids = r.render(cams, p, want_ids=True)
        torch.cuda.synchronize()
        serial.append((out.clone(), ids.clone()))
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs = [(torch.full((3, H, W, 4), -1.0, device="cuda"), torch.full((3, sc.k, H, W), 7, dtype=torch.int32, device="cuda")) for _ in sets]
    torch.cuda.synchronize()
    for rep in range(3):                                   # interleaved, nothing waits in between
        for i, cams in enumerate(sets):
            b.vs_render(r.handle, cams, p, outs[i][0], outs[i][1], stream=streams[i])
    torch.cuda.synchronize()
    for i in range(2):
        assert torch.equal(outs[i][0], serial[i][0]) and torch.equal(outs[i][1], serial[i][1]), "stream %d differs from the serial call" % i

    def worker(i):
        with torch.cuda.stream(streams[i]):
            for _ in range(3):
                b.vs_render(r.handle, sets[i], p, outs[i][0], outs[i][1], stream=streams[i])
    for o in outs:
        o[0].fill_(-1.0)
    torch.cuda.synchronize()
    threads = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    torch.cuda.synchronize()
    for i in range(2):
        assert torch.equal(outs[i][0], serial[i][0]) and torch.equal(outs[i][1], serial[i][1]), "thread %d differs from the serial call" % i
    if not env.path_flags:
        po = b.make_params(W, H, sc.near_plane, sc.t_min, sc.background, b.VS_FLAG_OVERLAP, 1)
        for i, cams in enumerate(sets):
            outs[i][0].fill_(-1.0)
            b.vs_render(r.handle, cams, po, outs[i][0], outs[i][1], stream=streams[i])
        torch.cuda.synchronize()
        for i in range(2):
            assert torch.equal(outs[i][0], serial[i][0]) and torch.equal(outs[i][1], serial[i][1]), "VS_FLAG_OVERLAP differs"
    # zero cameras: a legal no-op
    b.vs_render(r.handle, np.zeros((0, 16), np.float32), p, torch.empty((0, H, W, 4), device="cuda"))
    torch.cuda.synchronize()
    assert r.stats()["dropped_triangles"] == 0
    r.close()

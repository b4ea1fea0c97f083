"""GPU parity at BASELINE.json's FULL sizes (configs C2..C5; C1 is already full size in
test_gpu_parity.py), in the launch configuration bench.py times (whole camera batch in one vs_render
call, automatic chunking, no AOV in the timed call).

For each configuration the whole batch is rendered once; FOUR views (chosen to include the first, the
last and -- for C5 -- two far and two close-up cameras) are compared against the CPU oracle pixel
by pixel: triangle ids BIT-EXACT, RGBA max abs error <= 1e-4.  On the first of them the counters behind
every roofline figure (VS_FLAG_COUNT_TEXELS: shaded fragments, unique footprint texels) are compared with
the oracle's footprint census: fragments exactly, texels to 1e-4 relative (a footprint whose fp32 texel
coordinate falls on the other side of a texel boundary than the oracle's fp64 one moves by one texel).  Every view is additionally checked
through properties that hold at any size (the AOV-less timed call and the AOV call give the same
image bit for bit; the default direct raster path and the per-tile path give the same ids and image; alpha in [0,1]; pixels no layer hits are exactly the background; ids in range;
no dropped triangles)."""
import types

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-4
TEXEL_COUNT_RTOL = 1e-4     # fp32-vs-fp64 footprint edge cases


@pytest.fixture(scope="module")
def env():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    import oracle
    from paper_2409_02482_b200 import binding, synth
    binding.load_library()
    return types.SimpleNamespace(torch=torch, oracle=oracle, binding=binding, synth=synth)


def _check_config(env, cfg, sample_views, id_views):
    b, torch = env.binding, env.torch
    sc = env.synth.make_config(cfg)
    B, W, H, k = len(sc.cameras), sc.width, sc.height, sc.k
    r = b.Renderer(sc)
    p = b.make_params(W, H, sc.near_plane, sc.t_min, sc.background)
    p_tiled = b.make_params(W, H, sc.near_plane, sc.t_min, sc.background, b.VS_FLAG_TILED_PATH)
    # (1) the timed launch configuration: whole batch, no AOV
    out = torch.empty((B, H, W, 4), dtype=torch.float32, device="cuda")
    b.vs_render(r.handle, sc.cameras, p, out)
    torch.cuda.synchronize()
    stats = r.stats()
    assert stats["dropped_triangles"] == 0, "cameras are outside the shells: nothing may be dropped"
    rgba_all = out.cpu().numpy()
    del out
    assert np.isfinite(rgba_all).all()
    assert rgba_all[..., 3].min() >= 0.0 and rgba_all[..., 3].max() <= 1.0
    # (2) the AOV call on the sampled views must give the same image and ids that match the oracle
    worst = 0.0
    for v in sample_views:
        rgba, ids = r.render(sc.cameras[[v]], p, want_ids=True)
        torch.cuda.synchronize()
        rgba = rgba.cpu().numpy()[0]
        ids = ids.cpu().numpy().view(np.uint32)[0]
        assert np.array_equal(rgba, rgba_all[v]), "AOV call and timed call differ in view %d" % v
        # the per-tile raster path (binning + shared-memory keys) must give the same ids and image bit for bit
        rgba_t, ids_t = r.render(sc.cameras[[v]], p_tiled, want_ids=True)
        torch.cuda.synchronize()
        assert np.array_equal(ids_t.cpu().numpy().view(np.uint32)[0], ids), "tiled and direct ids differ in view %d" % v
        assert np.array_equal(rgba_t.cpu().numpy()[0], rgba), "tiled and direct images differ in view %d" % v
        del rgba_t, ids_t
        ntri = np.array([ly.indices.shape[0] for ly in sc.layers], np.uint32)[:, None, None]
        hit = ids != b.MISS
        assert np.all(ids[hit] < np.broadcast_to(ntri, ids.shape)[hit])
        nohit = ~hit.any(axis=0)
        bg = np.array(list(sc.background) + [0.0], np.float32)
        assert np.array_equal(rgba[nohit], np.broadcast_to(bg, rgba[nohit].shape))
        if v in id_views:
            ref = env.oracle.render_scene(sc, [v])[0]
            nbad = int((ids != ref["ids"]).sum())
            assert nbad == 0, "C%d view %d: %d triangle ids differ from the oracle" % (cfg, v, nbad)
            err = float(np.abs(rgba.astype(np.float64) - ref["rgba"]).max())
            worst = max(worst, err)
            assert err <= TOL, "C%d view %d: max abs rgba error %.3e" % (cfg, v, err)
    # (3) the roofline numerator: the GPU's instrumented pass against the oracle's footprint census on one view
    v = id_views[0]
    pc = b.make_params(W, H, sc.near_plane, sc.t_min, sc.background, b.VS_FLAG_COUNT_TEXELS)
    one = torch.empty((1, H, W, 4), dtype=torch.float32, device="cuda")
    b.vs_render(r.handle, sc.cameras[[v]], pc, one)
    cs = r.stats()
    ref = env.oracle.render_scene(sc, [v], want_layer_rgba=True, want_layer_uv=True)[0]
    frags, texels, _ = env.oracle.count_footprints(sc.layers, W, H, ref, t_min=sc.t_min)
    assert cs["shaded_fragments"] == frags, "C%d view %d: %d shaded fragments, the oracle composites %d" % (cfg, v, cs["shaded_fragments"], frags)
    assert abs(cs["unique_texels"] - texels) <= TEXEL_COUNT_RTOL * texels, \
        "C%d view %d: %d unique texels, the oracle counts %d" % (cfg, v, cs["unique_texels"], texels)
    r.close()
    print("C%d full size: %d views rendered, %d compared with the oracle, worst rgba err %.3e, coverage of view %d = %.3f; "
          "census of view %d: %d fragments (exact), %d unique texels (oracle %d)"
          % (cfg, B, len(id_views), worst, sample_views[0], float(hit.any(axis=0).mean()), v, frags, cs["unique_texels"], texels))


def test_config2_full(env):
    _check_config(env, 2, [0, 5, 10, 15], [0, 5, 10, 15])


def test_config3_full(env):
    _check_config(env, 3, [0, 13, 22, 31], [0, 13, 22, 31])


def test_config4_full(env):
    _check_config(env, 4, [0, 29, 46, 63], [0, 29, 46, 63])


def test_config4_full_attenuation(env):
    """SURVEY.md §8(f) NEXT-2 at the headline size: VS_FLAG_ATTENUATION on C4, whole batch in one
    call as bench.py --attenuation times it; two views against the oracle."""
    b, torch = env.binding, env.torch
    sc = env.synth.make_config(4)
    B, W, H = len(sc.cameras), sc.width, sc.height
    r = b.Renderer(sc)
    p = b.make_params(W, H, sc.near_plane, sc.t_min, sc.background, b.VS_FLAG_ATTENUATION)
    out = torch.empty((B, H, W, 4), dtype=torch.float32, device="cuda")
    b.vs_render(r.handle, sc.cameras, p, out)
    torch.cuda.synchronize()
    worst = 0.0
    for v in (0, 63):
        got = out[v].cpu().numpy()
        ref = env.oracle.render_scene(sc, [v], attenuation=True)[0]
        err = float(np.abs(got.astype(np.float64) - ref["rgba"]).max())
        worst = max(worst, err)
        assert err <= TOL, "C4 attenuated, view %d: max abs rgba error %.3e" % (v, err)
    r.close()
    print("C4 full size, attenuated: worst rgba err %.3e" % worst)


def test_config4_full_banded(env):
    """SURVEY.md §8(f) NEXT-1 at the headline size: C4 geometry and cameras with the paper's banded 8-bit textures
    (2048^2 .. 256^2 per band), whole batch in one call as bench.py --banded times it; two views
    against the oracle, ids bit-exact."""
    b, torch = env.binding, env.torch
    sc = env.synth.make_config(4, banded=True)
    B, W, H = len(sc.cameras), sc.width, sc.height
    r = b.Renderer(sc)
    p = b.make_params(W, H, sc.near_plane, sc.t_min, sc.background)
    out = torch.empty((B, H, W, 4), dtype=torch.float32, device="cuda")
    b.vs_render(r.handle, sc.cameras, p, out)
    torch.cuda.synchronize()
    assert r.stats()["dropped_triangles"] == 0
    worst = 0.0
    for v in (0, 63):
        rgba, ids = r.render(sc.cameras[[v]], p, want_ids=True)
        torch.cuda.synchronize()
        assert np.array_equal(rgba.cpu().numpy()[0], out[v].cpu().numpy())
        ref = env.oracle.render_scene(sc, [v])[0]
        assert np.array_equal(ids.cpu().numpy().view(np.uint32)[0], ref["ids"])
        err = float(np.abs(rgba.cpu().numpy()[0].astype(np.float64) - ref["rgba"]).max())
        worst = max(worst, err)
        assert err <= TOL, "C4 banded, view %d: max abs rgba error %.3e" % (v, err)
    r.close()
    print("C4 full size, banded: worst rgba err %.3e" % worst)


def test_config4_backward_full_resolution(env):
    """SURVEY.md §8(f) NEXT-4 at the headline geometry, image size and layer count (k = 9, ~300k triangles per layer,
    1920x1080): vs_render_backward over two views against the oracle's fp64 gradients.  Textures are 512^2 here (the
    oracle's fp64 gradient textures of the 2048^2 scene would take 19 GB): magnified texels, so thousands of fragments
    reduce into the same gradient texel -- the hard case for the atomic scatter."""
    b, torch = env.binding, env.torch
    sc = env.synth.make_config(4, tex_size=512, num_cameras=64)
    views = [0, 63]
    W, H = sc.width, sc.height
    g = np.random.default_rng(33).normal(size=(len(views), H, W, 4)).astype(np.float32)
    r = b.Renderer(sc)
    p = b.make_params(W, H, sc.near_plane, sc.t_min, sc.background)
    grads = [torch.zeros(ly.texture.shape, dtype=torch.float32, device="cuda") for ly in sc.layers]
    b.vs_render_backward(r.handle, sc.cameras[views], p, torch.from_numpy(g).cuda(), grads)
    torch.cuda.synchronize()
    r.close()
    want = None
    for n, v in enumerate(views):
        ref = env.oracle.render_scene(sc, [v])[0]
        want = env.oracle.render_backward(sc.layers, sc.sh_degree, sc.cameras[v], W, H, ref["ids"], g[n].astype(np.float64), want,
                                          near_plane=sc.near_plane, t_min=sc.t_min, background=sc.background)
    worst = 0.0
    for l in range(sc.k):
        got = grads[l].cpu().numpy().astype(np.float64)
        scale = np.abs(want[l]).max()
        assert scale > 1e-2
        err = np.abs(got - want[l]).max() / scale
        worst = max(worst, err)
        assert err <= 1e-4, "layer %d: relative gradient error %.3e" % (l, err)
        assert np.all(got[want[l] == 0.0] == 0.0)
    print("C4 geometry at 1920x1080, 512^2 textures, backward over 2 views: worst relative gradient error %.3e" % worst)


def test_config4_backward_full_size_textures(env):
    """The same at the FULL texture size (2048^2, the un-magnified regime: ~1.6 unique texels per fragment, so hardly any
    reduction per gradient texel -- the opposite case of the 512^2 test above).  The oracle's fp64 gradient of one layer is
    2.1 GB, so the layers are taken one at a time (oracle/render_backward skips the layers whose slot is None)."""
    b, torch = env.binding, env.torch
    sc = env.synth.make_config(4)
    v = 17
    W, H = sc.width, sc.height
    g = np.random.default_rng(34).normal(size=(1, H, W, 4)).astype(np.float32)
    r = b.Renderer(sc)
    p = b.make_params(W, H, sc.near_plane, sc.t_min, sc.background)
    grads = [torch.zeros(ly.texture.shape, dtype=torch.float32, device="cuda") for ly in sc.layers]
    b.vs_render_backward(r.handle, sc.cameras[[v]], p, torch.from_numpy(g).cuda(), grads)
    torch.cuda.synchronize()
    r.close()
    ref = env.oracle.render_scene(sc, [v])[0]
    worst = 0.0
    for l in (0, 4, 8):        # outermost, middle, innermost shell
        slot = [np.zeros(ly.texture.shape, np.float64) if i == l else None for i, ly in enumerate(sc.layers)]
        env.oracle.render_backward(sc.layers, sc.sh_degree, sc.cameras[v], W, H, ref["ids"], g[0].astype(np.float64), slot,
                                   near_plane=sc.near_plane, t_min=sc.t_min, background=sc.background)
        want = slot[l]
        got = grads[l].cpu().numpy()
        scale = np.abs(want).max()
        assert scale > 1e-3
        err = float(np.abs(got - want).max() / scale)
        worst = max(worst, err)
        assert err <= 1e-4, "layer %d: relative gradient error %.3e" % (l, err)
        assert np.all(got[want == 0.0] == 0.0)
        del slot, want, got
    print("C4 full size (2048^2 textures), backward of view %d, layers 0 / 4 / 8 against the oracle: worst relative gradient error %.3e"
          % (v, worst))


def test_config5_full(env):
    # even views are far cameras (r = 3), odd views close-ups (r = 1.6) that fill the frame: two of each
    _check_config(env, 5, [0, 1, 14, 15], [0, 1, 14, 15])

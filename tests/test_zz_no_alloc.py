"""vs_render_static (include/vs.h): the render call for callers that must not allocate -- all scratch in the library's
64 MiB `static __device__` array.  Checked against the existing path (vs_render) on the same inputs: triangle ids
bit-exact, RGBA within the tolerance of the parity tests (they are in fact bit-identical: same kernels), on two calls in
a row that lay the shared array out differently, then on another scene.  This file is collected LAST on purpose (the
suite runs with `pytest -x`); it passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-4


def _both(b, torch, sc, views, flags=0):
    """(rgba, ids) of vs_render and of vs_render_static for the given views of a scene."""
    r = b.Renderer(sc)
    try:
        cams = np.ascontiguousarray(sc.cameras[list(views)])
        p = b.make_params(sc.width, sc.height, sc.near_plane, sc.t_min, sc.background, flags)
        ref_rgba, ref_ids = r.render(cams, p, want_ids=True)
        torch.cuda.synchronize()
        out = torch.full((len(views), sc.height, sc.width, 4), -7.0, dtype=torch.float32, device="cuda")
        ids = torch.full((len(views), sc.k, sc.height, sc.width), 12345, dtype=torch.int32, device="cuda")
        b.vs_render_static(r.handle, cams, p, out, ids)
        torch.cuda.synchronize()
        return (ref_rgba.cpu().numpy(), ref_ids.cpu().numpy().view(np.uint32), out.cpu().numpy(), ids.cpu().numpy().view(np.uint32))
    finally:
        r.close()


def _check(ref_rgba, ref_ids, rgba, ids):
    assert np.array_equal(ids, ref_ids), "triangle ids differ in %d places" % int((ids != ref_ids).sum())
    err = float(np.abs(rgba.astype(np.float64) - ref_rgba.astype(np.float64)).max())
    assert err <= TOL, "max abs rgba difference %.3e" % err
    assert np.array_equal(rgba, ref_rgba), "same kernels, same operands: the images should be bit-identical (max diff %.3e)" % err
    assert (ref_ids != 0xFFFFFFFF).any() and ref_rgba[..., 3].max() > 0.1   # the scene is actually visible


def test_static_scratch_render_matches_vs_render_on_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "this test needs the B200"
    from paper_2409_02482_b200 import binding as b, synth
    b.load_library()
    sc = synth.make_config(4, mesh_n=40, width=333, height=217, tex_size=128, num_cameras=7)   # k = 9, fp16 SH-3, ragged tiles
    # call 1: seven views fill 36 MB of the array
    _check(*_both(b, torch, sc, range(7)))
    # call 2, right after it: other views, another count (every buffer moves inside the array, which still holds call 1's data)
    _check(*_both(b, torch, sc, [5, 2, 0]))
    # the other flags the entry point takes
    _check(*_both(b, torch, sc, [1, 6], flags=b.VS_FLAG_SCREEN_ORDER))
    _check(*_both(b, torch, sc, [3, 4], flags=b.VS_FLAG_ATTENUATION))
    # another scene (fp32 SH-1, k = 3, other image size) and a banded one share the same array
    c1 = synth.make_config(1)
    _check(*_both(b, torch, c1, range(len(c1.cameras))))
    cb = synth.make_config(4, mesh_n=24, width=160, height=120, tex_size=64, num_cameras=2, banded=True)
    _check(*_both(b, torch, cb, range(2)))


def test_static_scratch_render_allocates_nothing_and_rejects_what_does_not_fit():
    import torch
    from paper_2409_02482_b200 import binding as b, synth
    b.load_library()
    sc = synth.make_config(4, mesh_n=40, width=333, height=217, tex_size=128, num_cameras=7)
    r = b.Renderer(sc)
    try:
        p = b.make_params(sc.width, sc.height, sc.near_plane, sc.t_min, sc.background)
        out = torch.empty((7, sc.height, sc.width, 4), dtype=torch.float32, device="cuda")
        b.vs_render_static(r.handle, sc.cameras, p, out)            # warm-up: modules loaded, symbol address fetched
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        for _ in range(3):
            b.vs_render_static(r.handle, sc.cameras, p, out)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] >= free0, "device memory was allocated by vs_render_static"
        first = out.clone()
        b.vs_render_static(r.handle, sc.cameras, p, out)
        torch.cuda.synchronize()
        assert torch.equal(first, out)
        # 7 views of 1920 x 1080 x 9 layers need 1 GB: rejected with both numbers in the message, nothing launched
        big = b.make_params(1920, 1080, sc.near_plane, sc.t_min, sc.background)
        big_out = torch.empty((7, 1080, 1920, 4), dtype=torch.float32, device="cuda")
        with pytest.raises(b.VsError) as ei:
            b.vs_render_static(r.handle, sc.cameras, big, big_out)
        assert ei.value.status == b.VS_ERR_UNSUPPORTED
        assert str(b.VS_STATIC_SCRATCH_BYTES) in str(ei.value) and "bytes of scratch" in str(ei.value)
        # flags that need the library's other machinery are refused, zero cameras are a no-op
        with pytest.raises(b.VsError):
            b.vs_render_static(r.handle, sc.cameras, b.make_params(sc.width, sc.height, sc.near_plane, sc.t_min, sc.background,
                                                                  b.VS_FLAG_TILED_PATH), out)
        b.vs_render_static(r.handle, sc.cameras[:0], p, out[:0])
        torch.cuda.synchronize()
        assert torch.equal(first, out)
    finally:
        r.close()

"""Pins for the oracle's backward pass to the texels (SPEC.md:L388-396
"finite-difference gradient check").  The pinned forward oracle is the reference: for a loss L = sum_p g_p . out_p with a
fixed random g, dL/d(texel value) from vso_render_backward must equal the central finite difference of the forward
render.  CPU only."""
import numpy as np
import pytest

import oracle
from paper_2409_02482_b200 import synth


def _scene(k=3, att_tex=0.0):
    sc = synth.make_config(1, width=40, height=32, num_cameras=1, tex_size=16, k=k)
    for ly in sc.layers:
        ly.texture = (ly.texture * 1.5).astype(np.float32)
        ly.texture[:, :, 0, 3] += att_tex
    return sc


def _loss(sc, g, **kw):
    r = oracle.render_scene(sc, [0], **kw)[0]
    return float((r["rgba"] * g).sum()), r


@pytest.mark.parametrize("attenuation,background", [(False, (0.0, 0.0, 0.0)), (True, (0.3, 0.6, 0.1))])
def test_backward_matches_finite_differences(attenuation, background):
    sc = _scene()
    rng = np.random.default_rng(5)
    g = rng.normal(size=(sc.height, sc.width, 4))
    kw = dict(t_min=0.0, background=background, attenuation=attenuation)
    L0, r = _loss(sc, g, **kw)
    grads = oracle.render_backward(sc.layers, sc.sh_degree, sc.cameras[0], sc.width, sc.height, r["ids"], g,
                                   near_plane=sc.near_plane, **kw)
    assert all(np.isfinite(gt).all() for gt in grads)
    checked = 0
    for l in range(sc.k):
        nz = np.argwhere(np.abs(grads[l]) > 1e-3)
        assert len(nz) > 50                                        # the layer is seen through the ones in front of it
        for (ty, tx, c, ch) in nz[rng.choice(len(nz), 12, replace=False)]:
            tex = sc.layers[l].texture
            old = tex[ty, tx, c, ch]
            hi, lo = np.float32(old + 2.0 ** -6), np.float32(old - 2.0 ** -6)
            tex[ty, tx, c, ch] = hi
            Lp, _ = _loss(sc, g, **kw)
            tex[ty, tx, c, ch] = lo
            Lm, _ = _loss(sc, g, **kw)
            tex[ty, tx, c, ch] = old
            fd = (Lp - Lm) / (float(hi) - float(lo))
            assert abs(fd - grads[l][ty, tx, c, ch]) <= 2e-4 * max(1.0, abs(fd)), (l, ty, tx, c, ch, fd, grads[l][ty, tx, c, ch])
            checked += 1
    assert checked == 12 * sc.k
    # texels no fragment's footprint touches get exactly zero
    assert any((gt == 0.0).any() for gt in grads)


def test_backward_is_linear_in_the_upstream_gradient_and_accumulates():
    sc = _scene()
    rng = np.random.default_rng(6)
    g1, g2 = rng.normal(size=(2, sc.height, sc.width, 4))
    r = oracle.render_scene(sc, [0])[0]
    args = (sc.layers, sc.sh_degree, sc.cameras[0], sc.width, sc.height, r["ids"])
    a = oracle.render_backward(*args, g1)
    b = oracle.render_backward(*args, g2)
    both = oracle.render_backward(*args, 2.0 * g1 - g2)
    acc = oracle.render_backward(*args, g2, grad_tex=[x.copy() for x in a])       # += into existing buffers
    for l in range(sc.k):
        np.testing.assert_allclose(both[l], 2.0 * a[l] - b[l], atol=1e-12)
        np.testing.assert_allclose(acc[l], a[l] + b[l], atol=1e-12)


def test_layers_behind_the_early_exit_get_no_gradient():
    sc = _scene(att_tex=60.0)                     # near-opaque layers: T < t_min after the outermost one
    rng = np.random.default_rng(7)
    g = rng.normal(size=(sc.height, sc.width, 4))
    r = oracle.render_scene(sc, [0], t_min=2.0 ** -6)[0]
    grads = oracle.render_backward(sc.layers, sc.sh_degree, sc.cameras[0], sc.width, sc.height, r["ids"], g, t_min=2.0 ** -6)
    inner_only = (r["ids"][0] == oracle.MISS) & (r["ids"][1] != oracle.MISS)
    assert not inner_only.any()                   # nested shells: layer 1 is only ever seen through layer 0
    assert np.abs(grads[0]).max() > 1e-3 and np.all(grads[1] == 0.0) and np.all(grads[2] == 0.0)


def test_layers_can_be_taken_one_at_a_time():
    """grad_tex[l] = None skips layer l; the other layers' gradients are unchanged (the full-size GPU test relies on it)."""
    sc = synth.make_config(1, width=40, height=32, num_cameras=1, tex_size=32)
    ref = oracle.render_scene(sc, [0])[0]
    g = np.random.default_rng(5).normal(size=(sc.height, sc.width, 4))
    kw = dict(near_plane=sc.near_plane, t_min=sc.t_min, background=sc.background)
    full = oracle.render_backward(sc.layers, sc.sh_degree, sc.cameras[0], sc.width, sc.height, ref["ids"], g, **kw)
    for l in range(sc.k):
        only = [np.zeros(ly.texture.shape, np.float64) if i == l else None for i, ly in enumerate(sc.layers)]
        oracle.render_backward(sc.layers, sc.sh_degree, sc.cameras[0], sc.width, sc.height, ref["ids"], g, only, **kw)
        np.testing.assert_allclose(only[l], full[l], rtol=0, atol=1e-12 * max(1.0, np.abs(full[l]).max()))

"""Pins for the oracle's banded 8-bit texture path (§4.5 "Mixed
resolutions" and "Squeezing and quantization").  CPU only.  Pinned: q and the re-scale against the values SPEC.md
prints; the mixed-resolution sample against torch grid_sample per band; the whole banded render against the
(already pinned) float render of the decoded coefficients -- same resolution for all bands (concatenation and
channel order), and mixed resolutions through affine band images that bilinear interpolation reproduces exactly."""
import os
import types

import numpy as np
import pytest

import oracle
from paper_2409_02482_b200 import synth

VR = (-15.0, 15.0)


def decode(t, v_range=VR):
    return v_range[0] + (v_range[1] - v_range[0]) * (t.astype(np.float64) / 255.0)


def test_quantization_golden(golden_dir):
    rows = [[f.strip() for f in l.split("|")] for l in open(os.path.join(golden_dir, "quantization_examples.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 6
    for kind, x, want, tol in rows:
        x, want, tol = float(x), float(want), float(tol)
        got = oracle.quantize(x) if kind == "quantize" else oracle.rescale(oracle.quantize(x), -15.0, 15.0)
        assert abs(got - want) <= tol, (kind, x, got, want)


def test_quantize_properties():
    rng = np.random.default_rng(0)
    for x in rng.uniform(0, 1, 2000):
        q = oracle.quantize(x)
        assert oracle.quantize(q) == q                          # idempotent
        assert abs(q - x) <= 0.5 / 255 + 1e-15                  # nearest of the 256 levels
        assert abs(q * 255 - round(q * 255)) < 1e-12
    assert oracle.quantize(0.5) == 128 / 255                    # the half rounds AWAY from zero (127.5 -> 128)
    assert oracle.rescale(0.0, -3.0, 7.0) == -3.0 and oracle.rescale(1.0, -3.0, 7.0) == 7.0
    assert oracle.rescale(0.25, -3.0, 7.0) == -0.5


def test_sample_banded_matches_grid_sample_per_band():
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(1)
    sizes = [(24, 32), (12, 16), (5, 7), (3, 2)]                 # (H, W) per band: every band has its own grid
    bands = [rng.integers(0, 256, size=(h, w, 2 * b + 1, 4), dtype=np.uint8) for b, (h, w) in enumerate(sizes)]
    uvs = np.concatenate([rng.uniform(0, 1, (200, 2)), rng.uniform(-0.2, 1.2, (50, 2)),
                          [[0.0, 0.0], [1.0, 1.0], [0.5, 0.5]]])
    grid = torch.tensor(uvs * 2 - 1, dtype=torch.float64).view(1, -1, 1, 2)
    want = np.zeros((len(uvs), 16, 4))
    for b, t in enumerate(bands):
        img = torch.tensor(decode(t)).permute(2, 3, 0, 1).reshape(1, -1, t.shape[0], t.shape[1])
        s = torch.nn.functional.grid_sample(img, grid, mode="bilinear", padding_mode="border", align_corners=False)
        want[:, b * b:(b + 1) ** 2, :] = s.view(2 * b + 1, 4, -1).permute(2, 0, 1).numpy()
    for i, (u, v) in enumerate(uvs):
        got = oracle.sample_banded(bands, VR[0], VR[1], u, v)
        np.testing.assert_allclose(got, want[i], atol=1e-11)


def _float_twin(sc, band_to_full):
    """The float32 scene whose coefficient texture holds the decoded values of the banded scene's bytes, band b
    brought to the base resolution by `band_to_full(b, decoded_band, H, W)`."""
    layers = []
    for ly in sc.layers:
        H, W = ly.band_textures[0].shape[:2]
        tex = np.zeros((H, W, (sc.sh_degree + 1) ** 2, 4), dtype=np.float32)
        for b, t in enumerate(ly.band_textures):
            tex[:, :, b * b:(b + 1) ** 2, :] = band_to_full(b, decode(t, sc.v_range), H, W)
        layers.append(synth.Layer(ly.positions, ly.uvs, ly.indices, tex))
    return synth.Scene("twin", layers, sc.sh_degree, sc.cameras, sc.width, sc.height, sc.near_plane, sc.t_min, sc.background)


def test_banded_same_resolution_equals_float_render():
    """All bands at one resolution: the banded render IS the float render of the decoded coefficients.  Uses values
    whose decode is exact in float32 (v_range (0, 255): sh = t), so the two differ by rounding order only."""
    rng = np.random.default_rng(2)
    sc = synth.make_config(4, mesh_n=16, width=96, height=64, tex_size=32, num_cameras=2, k=3, banded=True)
    for ly in sc.layers:        # small logits so that the sigmoid is not saturated: bytes 0..5 around 2.5
        ly.band_textures = [rng.integers(0, 6, size=(32, 32, 2 * b + 1, 4), dtype=np.uint8) for b in range(4)]
    sc.v_range = (-2.5, 252.5)  # sh = t - 2.5: exact in float32
    twin = _float_twin(sc, lambda b, d, H, W: d)
    for v in range(2):
        a = oracle.render_scene(sc, [v], want_layer_rgba=True)[0]
        f = oracle.render_scene(twin, [v], want_layer_rgba=True)[0]
        assert np.array_equal(a["ids"], f["ids"])
        assert (a["ids"] != oracle.MISS).mean() > 0.2
        np.testing.assert_allclose(a["layer_rgba"], f["layer_rgba"], atol=1e-12)
        np.testing.assert_allclose(a["rgba"], f["rgba"], atol=1e-12)
    # a wrong band offset or channel order would mix coefficients: make the bands distinguishable and re-check one pixel set
    assert len({t.tobytes() for t in sc.layers[0].band_textures}) == 4


def test_banded_mixed_resolution_affine_bands():
    """Band b at (32 >> b)^2 holding an affine function of uv sampled at ITS texel centres; the float twin holds the same
    affine function at the base resolution's texel centres.  Bilinear interpolation reproduces affine functions, so
    away from the clamped border both renders agree: this pins each band's own (W_b, H_b) texel-centre mapping."""
    sc = synth.make_config(4, mesh_n=16, width=96, height=64, tex_size=32, num_cameras=2, k=2, banded=True)
    deg = sc.sh_degree
    rng = np.random.default_rng(3)
    slopes = np.array([(0, 0), (1, 0), (-1, 0), (0, 1), (0, -1)])
    coefs = np.concatenate([rng.integers(-2, 3, size=(len(sc.layers), 16, 4, 1)),       # a + 64 (bu u + cv v) per (c, ch)
                            slopes[rng.integers(0, 5, size=(len(sc.layers), 16, 4))]], axis=-1)

    def affine(l, b, size):
        # integer-valued bytes: t = 128 + a + 64 (bu u + cv v) with u = (i + .5)/size, size | 32: 64 u is an integer
        i = (np.arange(size) + 0.5) / size
        uu, vv = np.meshgrid(i, i, indexing="xy")
        cf = coefs[l, b * b:(b + 1) ** 2]                                                 # [2b+1, 4, 3]
        return 128.0 + cf[None, None, :, :, 0] + 64.0 * (cf[None, None, :, :, 1] * uu[..., None, None]
                                                         + cf[None, None, :, :, 2] * vv[..., None, None])
    for l, ly in enumerate(sc.layers):
        bt = []
        for b in range(deg + 1):
            size = 32 >> b
            t = affine(l, b, size)
            assert np.array_equal(t, np.rint(t)) and t.min() >= 0 and t.max() <= 255      # exactly representable bytes
            bt.append(t.astype(np.uint8))
        ly.band_textures = bt
    sc.v_range = (-1.28, 1.27)     # sh = -1.28 + t/100: logits around 0
    layers = []
    for l, ly in enumerate(sc.layers):
        tex = np.zeros((32, 32, 16, 4), dtype=np.float64)
        for b in range(deg + 1):
            tex[:, :, b * b:(b + 1) ** 2, :] = decode(affine(l, b, 32), sc.v_range)
        layers.append(synth.Layer(ly.positions, ly.uvs, ly.indices, tex.astype(np.float32)))
    twin = synth.Scene("twin", layers, deg, sc.cameras, sc.width, sc.height, sc.near_plane, sc.t_min, sc.background)
    for v in range(2):
        a = oracle.render_scene(sc, [v], want_layer_rgba=True, want_layer_uv=True)[0]
        f = oracle.render_scene(twin, [v], want_layer_rgba=True)[0]
        assert np.array_equal(a["ids"], f["ids"])
        uv = a["layer_uv"]
        # interior of the coarsest band's unclamped region: its texel centres span [0.5/4, 1 - 0.5/4]
        lo, hi = 0.5 / (32 >> deg), 1 - 0.5 / (32 >> deg)
        inner = (a["ids"] != oracle.MISS) & (uv[..., 0] > lo) & (uv[..., 0] < hi) & (uv[..., 1] > lo) & (uv[..., 1] < hi)
        assert inner.sum() > 300
        np.testing.assert_allclose(a["layer_rgba"][inner], f["layer_rgba"][inner], atol=2e-7)   # float32 twin texels
        # and outside it they DO differ somewhere (the coarse bands clamp earlier): the check is not vacuous
        outer = (a["ids"] != oracle.MISS) & ~inner
        assert np.abs(a["layer_rgba"][outer] - f["layer_rgba"][outer]).max() > 1e-4

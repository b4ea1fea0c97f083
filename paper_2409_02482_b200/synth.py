"""Seeded synthetic inputs for the k-shell renderer: meshes, UV atlases, textures, cameras.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path, and therefore holds none of
the method's arithmetic (no projection, rasterisation, texture filtering, SH or blending): it only
makes input arrays.  numpy only.

The paper measures on Shelly / DTU / NeRF-Synthetic / custom captures (§5) whose
baked assets are not available; these scenes take their *shape* instead: object-centric, k nested
closed shells ordered outermost -> innermost, per-shell chart-based UV
atlases, per-shell textures of (deg+1)^2 x RGBA spherical-harmonics coefficients
(PAPER.md:L437-438, L463), cameras orbiting outside the object.  The five configurations are the
ones `BASELINE.json` names (recipe: SURVEY.md §8(d), restated in DESIGN.md §4).
"""
from __future__ import annotations

import dataclasses
import math
from concurrent.futures import ThreadPoolExecutor

import numpy as np

CAMERA_FLOATS = 16  # fx fy cx cy R[9] (row-major) t[3]


@dataclasses.dataclass
class Layer:
    positions: np.ndarray  # [V,3] float32, world space
    uvs: np.ndarray        # [V,2] float32 in [0,1]
    indices: np.ndarray    # [T,3] uint32
    texture: np.ndarray    # [H,W,n,4] float32 or float16 ; ch 0-2 RGB, ch 3 opacity logit (None for banded scenes)
    band_textures: list | None = None   # banded 8-bit format: band b = uint8 [H_b, W_b, 2b+1, 4]
    normals: np.ndarray | None = None   # optional [V,3] float32 per-vertex normals (transparency attenuation)


@dataclasses.dataclass
class Scene:
    name: str
    layers: list           # outermost first
    sh_degree: int
    cameras: np.ndarray    # [B,16] float32
    width: int
    height: int
    near_plane: float = 0.05
    t_min: float = 2.0 ** -14
    background: tuple = (0.0, 0.0, 0.0)
    v_range: tuple | None = None   # banded scenes: (v_min, v_max) the stored bytes are re-scaled to

    @property
    def k(self) -> int:
        return len(self.layers)

    @property
    def n_coef(self) -> int:
        return (self.sh_degree + 1) ** 2

    @property
    def tex_dtype(self):
        return np.dtype(np.uint8) if self.layers[0].band_textures is not None else self.layers[0].texture.dtype


# ------------------------------------------------------------------------------------------------
# meshes
# ------------------------------------------------------------------------------------------------

def _icosahedron():
    t = (1.0 + math.sqrt(5.0)) / 2.0
    v = np.array([[-1, t, 0], [1, t, 0], [-1, -t, 0], [1, -t, 0],
                  [0, -1, t], [0, 1, t], [0, -1, -t], [0, 1, -t],
                  [t, 0, -1], [t, 0, 1], [-t, 0, -1], [-t, 0, 1]], dtype=np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    f = np.array([[0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11],
                  [1, 5, 9], [5, 11, 4], [11, 10, 2], [10, 7, 6], [7, 1, 8],
                  [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8], [3, 8, 9],
                  [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1]], dtype=np.int64)
    return v, f


def icosphere_charted(subdiv: int, radius: float, tex_size: int = 256, gutter_texels: float = 2.0):
    """Unit icosphere, each of the 20 base faces tessellated into 4**subdiv triangles and given its
    own UV chart (5x4 grid of cells, seam vertices duplicated).  Returns positions, uvs, indices."""
    bv, bf = _icosahedron()
    m = 2 ** subdiv
    pos, uv, idx = [], [], []
    g = gutter_texels / tex_size
    for c, (a, b, d) in enumerate(bf):
        cell_x, cell_y = c % 5, c // 5
        ox, oy = cell_x / 5.0 + g, cell_y / 4.0 + g
        sx, sy = 1.0 / 5.0 - 2 * g, 1.0 / 4.0 - 2 * g
        base = sum(len(p) for p in pos)
        local = {}
        P, U = [], []
        for i in range(m + 1):
            for j in range(m + 1 - i):
                wa, wb, wd = (m - i - j) / m, i / m, j / m
                p = wa * bv[a] + wb * bv[b] + wd * bv[d]
                p = p / np.linalg.norm(p) * radius
                local[(i, j)] = len(P)
                P.append(p)
                U.append((ox + sx * (i / m), oy + sy * (j / m)))
        F = []
        for i in range(m):
            for j in range(m - i):
                F.append((local[(i, j)], local[(i + 1, j)], local[(i, j + 1)]))
                if j < m - i - 1:
                    F.append((local[(i + 1, j)], local[(i + 1, j + 1)], local[(i, j + 1)]))
        pos.append(np.asarray(P))
        uv.append(np.asarray(U))
        idx.append(np.asarray(F, dtype=np.int64) + base)
    return (np.concatenate(pos).astype(np.float32), np.concatenate(uv).astype(np.float32),
            np.concatenate(idx).astype(np.uint32))


def cube_sphere_charted(n: int, tex_size: int, gutter_texels: float = 2.0):
    """Cube-sphere: 6 faces x (n+1)^2 vertices, 12 n^2 triangles; unit directions.  UV = 6 square
    charts in a 3x2 atlas with a gutter.  Returns unit directions [V,3] float64, uvs, indices."""
    s = np.linspace(-1.0, 1.0, n + 1)
    a, b = np.meshgrid(s, s, indexing="xy")  # a varies along columns
    one = np.ones_like(a)
    faces = [(one, a, b), (-one, b, a), (b, one, a), (a, -one, b), (a, b, one), (b, a, -one)]
    g = gutter_texels / tex_size
    qi, qj = np.meshgrid(np.arange(n), np.arange(n), indexing="xy")
    v00 = (qj * (n + 1) + qi).ravel()
    v01 = v00 + 1
    v10 = v00 + (n + 1)
    v11 = v10 + 1
    quad = np.stack([np.stack([v00, v01, v11], 1), np.stack([v00, v11, v10], 1)], 1).reshape(-1, 3)
    dirs, uvs, idx = [], [], []
    for c, (x, y, z) in enumerate(faces):
        d = np.stack([x, y, z], -1).reshape(-1, 3)
        d = d / np.linalg.norm(d, axis=1, keepdims=True)
        cu, cv = c % 3, c // 3
        uu = (cu + g * 3 + (a + 1) * 0.5 * (1 - 2 * g * 3)) / 3.0
        vv = (cv + g * 2 + (b + 1) * 0.5 * (1 - 2 * g * 2)) / 2.0
        dirs.append(d)
        uvs.append(np.stack([uu, vv], -1).reshape(-1, 2))
        idx.append(quad + c * (n + 1) ** 2)
    return np.concatenate(dirs), np.concatenate(uvs).astype(np.float32), np.concatenate(idx).astype(np.uint32)


def plane_wave_noise(dirs: np.ndarray, rng: np.random.Generator, n_waves: int = 8, fmax: float = 2.0):
    """Low-frequency noise on the sphere: sum of seeded plane waves, normalised to |n| <= 1."""
    f = rng.uniform(-fmax, fmax, size=(n_waves, 3))
    nrm = np.linalg.norm(f, axis=1, keepdims=True)
    f = f / np.maximum(nrm / fmax, 1.0)          # |f| <= fmax
    amp = rng.uniform(0.5, 1.0, size=n_waves)
    ph = rng.uniform(0, 2 * math.pi, size=n_waves)
    val = np.zeros(len(dirs))
    for i in range(n_waves):
        val += amp[i] * np.sin(2 * math.pi * (dirs @ f[i]) + ph[i])
    return val / amp.sum()


def noise_shells(k: int, n: int, tex_size: int, seed: int, amplitude: float = 0.05, spacing: float = 0.03):
    """k strictly nested shells r_l(d) = 1 + amplitude*noise(d) - spacing*l (l = 0 outermost)."""
    dirs, uvs, idx = cube_sphere_charted(n, tex_size)
    noise = plane_wave_noise(dirs, np.random.default_rng([seed, 1000]))
    out = []
    for l in range(k):
        r = 1.0 + amplitude * noise - spacing * l
        out.append(((dirs * r[:, None]).astype(np.float32), uvs, idx))
    return out


# ------------------------------------------------------------------------------------------------
# cameras
# ------------------------------------------------------------------------------------------------

def look_at_camera(eye, width: int, height: int, fov_y_deg: float = 40.0, target=(0.0, 0.0, 0.0)):
    """x_cam = R x_world + t ; +x right, +y DOWN, +z forward.  Returns 16 float32."""
    eye = np.asarray(eye, dtype=np.float64)
    fwd = np.asarray(target, dtype=np.float64) - eye
    fwd /= np.linalg.norm(fwd)
    up = np.array([0.0, 1.0, 0.0])
    if abs(fwd @ up) > 0.99:
        up = np.array([1.0, 0.0, 0.0])
    right = np.cross(fwd, up)
    right /= np.linalg.norm(right)
    down = np.cross(fwd, right)
    R = np.stack([right, down, fwd])
    t = -R @ eye
    f = 0.5 * height / math.tan(math.radians(fov_y_deg) / 2)
    return np.concatenate([[f, f, width / 2.0, height / 2.0], R.ravel(), t]).astype(np.float32)


def circle_cameras(n: int, radius: float, width: int, height: int, fov: float = 40.0):
    cams = []
    for i in range(n):
        a = 2 * math.pi * i / n
        cams.append(look_at_camera((radius * math.sin(a), 0.0, radius * math.cos(a)), width, height, fov))
    return np.stack(cams)


def fibonacci_cameras(n: int, radius, width: int, height: int, fov: float = 40.0, rotate: float = 0.0):
    """Cameras on a Fibonacci sphere lattice looking at the origin.  `radius` scalar or [n]."""
    radius = np.broadcast_to(np.asarray(radius, dtype=np.float64), (n,))
    golden = math.pi * (3.0 - math.sqrt(5.0))
    cams = []
    for i in range(n):
        y = 1.0 - 2.0 * (i + 0.5) / n
        r = math.sqrt(max(0.0, 1.0 - y * y))
        th = golden * i + rotate
        cams.append(look_at_camera(radius[i] * np.array([r * math.cos(th), y, r * math.sin(th)]),
                                   width, height, fov))
    return np.stack(cams)


# ------------------------------------------------------------------------------------------------
# textures
# ------------------------------------------------------------------------------------------------

def normal_texture(seed_key, tex_h: int, tex_w: int, n_coef: int, sigma: float, dtype,
                   opacity_band0=None):
    """[H,W,n,4] coefficients ~ N(0, sigma).  `opacity_band0=(mu, sd)` redraws the band-0 opacity
    coefficient so that the view-independent part of the opacity *logit* is ~ N(mu, sd)."""
    rng = np.random.default_rng(seed_key)
    tex = np.empty((tex_h, tex_w, n_coef, 4), dtype=dtype)
    rows = max(1, (1 << 22) // (tex_w * n_coef * 4))
    for r0 in range(0, tex_h, rows):
        r1 = min(tex_h, r0 + rows)
        blk = rng.standard_normal((r1 - r0, tex_w, n_coef, 4), dtype=np.float32)
        blk *= np.float32(sigma)
        if opacity_band0 is not None:
            g = rng.standard_normal((r1 - r0, tex_w), dtype=np.float32)
            blk[:, :, 0, 3] = (np.float32(opacity_band0[0]) + np.float32(opacity_band0[1]) * g) \
                / np.float32(0.28209479177387814)
        tex[r0:r1] = blk
    return tex


def banded_textures(seed_key, base_size: int, degree: int, sigma_lsb: float = 2.55):
    """The paper's baked texture format: one 8-bit image set per SH band, band b at
    (base_size >> b)^2 ("base color at the highest resolution, the highest SH degree at the lowest": 2048^2 .. 256^2
    for degree 3).  Bytes ~ round(N(127.5, sigma_lsb)) clipped to 0..255: with the paper's range [-15, 15]
    (30/255 per step) sigma_lsb = 2.55 is the N(0, 0.3) coefficient spread of the float configurations."""
    rng = np.random.default_rng(seed_key)
    out = []
    for b in range(degree + 1):
        size = max(1, base_size >> b)
        t = rng.standard_normal((size, size, 2 * b + 1, 4), dtype=np.float32)
        t *= np.float32(sigma_lsb)
        t += np.float32(127.5)
        np.rint(t, out=t)
        np.clip(t, 0, 255, out=t)
        out.append(t.astype(np.uint8))
    return out


def _parallel(fns):
    with ThreadPoolExecutor(max_workers=min(len(fns), 16)) as ex:
        return list(ex.map(lambda f: f(), fns))


# ------------------------------------------------------------------------------------------------
# the five BASELINE.json configurations
# ------------------------------------------------------------------------------------------------

CONFIG_NAMES = {
    1: "C1 k=3 icospheres 128x128 x4 cams, fp32 SH1 256^2",
    2: "C2 k=5 noise shells ~100k tris, 800x800 x16 cams, fp16 SH2 1024^2",
    3: "C3 k=7 noise shells ~200k tris, 1920x1080 x32 cams, fp16 SH3 2048^2, low alpha",
    4: "C4 k=9 noise shells ~300k tris, 1920x1080 x64 views, fp16 SH3 2048^2 (headline)",
    5: "C5 k=9 noise shells ~1M tris, 3840x2160 x16 cams incl. close-ups, fp16 SH3 4096^2",
}


def _scene_name(cfg: int, layers, W: int, H: int, B: int, deg: int, reduced: bool, suffix: str = "") -> str:
    """Name built from the ACTUAL sizes; the full configuration keeps its BASELINE.json wording, a variant made with
    overrides is called "Cn-reduced" and lists what was really built (so that no log line claims more than was run)."""
    if not reduced:
        return CONFIG_NAMES[cfg] + suffix
    ly = layers[0]
    if ly.band_textures is not None:
        tex = "uint8 banded %d^2" % ly.band_textures[0].shape[0]
    else:
        tex = "%s SH%d %dx%d" % ("fp16" if ly.texture.dtype == np.float16 else "fp32", deg, ly.texture.shape[1], ly.texture.shape[0])
    return "C%d-reduced k=%d, %d tris/layer, %dx%d x%d views, %s%s" % (cfg, len(layers), ly.indices.shape[0], W, H, B, tex, suffix)


def make_config(cfg: int, *, seed: int = 0, mesh_n: int | None = None, width: int | None = None,
                height: int | None = None, tex_size: int | None = None, num_cameras: int | None = None,
                k: int | None = None, camera_rotate: float = 0.0, banded: bool = False,
                camera_subset: str | None = None) -> Scene:
    """Build configuration `cfg` (1..5).  The keyword overrides give *reduced* variants of the same
    recipe (used by the CPU tests, where the full sizes would take too long).  `banded=True` gives the
    same geometry and cameras with the paper's 8-bit mixed-resolution textures (`banded_textures`, v_range (-15, 15))
    instead of the float ones.  `camera_subset` = "far" / "close" keeps every other camera of the set:
    on C5 the even ones orbit at r = 3, the odd ones are the close-ups at r = 1.6 (the two regimes of SURVEY.md §8(d))."""
    reduced = any(v is not None for v in (mesh_n, width, height, tex_size, num_cameras, k))
    if cfg == 1:
        k = k or 3
        ts = tex_size or 256
        W, H = width or 128, height or 128
        B = num_cameras or 4
        radii = [1.0 - 0.1 * l for l in range(k)]
        layers = []
        for l in range(k):
            pos, uv, idx = icosphere_charted(3 if mesh_n is None else mesh_n, radii[l], ts)
            if banded:
                layers.append(Layer(pos, uv, idx, None, banded_textures([seed, 101, l], ts, 1, 8.0)))
                continue
            rng = np.random.default_rng([seed, 1, l])
            tex = np.empty((ts, ts, 4, 4), dtype=np.float32)
            tex[..., :3] = rng.uniform(-0.5, 0.5, size=(ts, ts, 4, 3))
            tex[..., 3] = rng.standard_normal((ts, ts, 4))
            layers.append(Layer(pos, uv, idx, tex))
        cams = circle_cameras(B, 3.0, W, H)
        if banded:
            return Scene(_scene_name(1, layers, W, H, B, 1, reduced, " [banded u8]"), layers, 1, cams, W, H, v_range=(-15.0, 15.0))
        return Scene(_scene_name(1, layers, W, H, B, 1, reduced), layers, 1, cams, W, H)

    spec = {
        2: dict(k=5, n=91, W=800, H=800, B=16, ts=1024, deg=2, op=None),
        3: dict(k=7, n=129, W=1920, H=1080, B=32, ts=2048, deg=3, op=(-1.0, 1.5)),
        4: dict(k=9, n=158, W=1920, H=1080, B=64, ts=2048, deg=3, op=None),
        5: dict(k=9, n=289, W=3840, H=2160, B=16, ts=4096, deg=3, op=None),
    }[cfg]
    k = k or spec["k"]
    n = mesh_n or spec["n"]
    W, H = width or spec["W"], height or spec["H"]
    B = num_cameras or spec["B"]
    ts = tex_size or spec["ts"]
    deg = spec["deg"]
    ncoef = (deg + 1) ** 2
    shells = noise_shells(k, n, ts, seed)
    if banded:
        texs = _parallel([(lambda l=l: banded_textures([seed, 100 + cfg, l], ts, deg)) for l in range(k)])
        layers = [Layer(p, uv, idx, None, texs[l]) for l, (p, uv, idx) in enumerate(shells)]
    else:
        texs = _parallel([
            (lambda l=l: normal_texture([seed, cfg, l], ts, ts, ncoef, 0.3, np.float16, spec["op"]))
            for l in range(k)])
        layers = [Layer(p, uv, idx, texs[l]) for l, (p, uv, idx) in enumerate(shells)]
    if cfg == 5:
        radius = np.where(np.arange(B) % 2 == 0, 3.0, 1.6)  # far / close-up alternate
    else:
        radius = 3.0
    cams = fibonacci_cameras(B, radius, W, H, rotate=camera_rotate)
    suffix = ""
    if camera_subset is not None:
        assert camera_subset in ("far", "close")
        cams = np.ascontiguousarray(cams[0::2] if camera_subset == "far" else cams[1::2])
        suffix = " [%d %s cameras of the set]" % (len(cams), camera_subset)
    if banded:
        return Scene(_scene_name(cfg, layers, W, H, len(cams), deg, reduced, " [banded u8 %d^2..%d^2]" % (ts, max(1, ts >> deg)) + suffix),
                     layers, deg, cams, W, H, v_range=(-15.0, 15.0))
    return Scene(_scene_name(cfg, layers, W, H, len(cams), deg, reduced, suffix), layers, deg, cams, W, H)

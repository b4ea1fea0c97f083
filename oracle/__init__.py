"""CPU oracle for the k-shell rasterise-and-composite path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It shares no code with the CUDA path (paper_2409_02482_b200/csrc, binding.py) and does
not import it; scenes come from paper_2409_02482_b200.synth, which holds none of the method's
arithmetic.  The arithmetic lives in oracle/vs_oracle.c (plain C, each function cites the passage it
follows); this file only marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import ensure_built

MISS = 0xFFFFFFFF


class _Layer(C.Structure):
    _fields_ = [("positions", C.c_void_p), ("uvs", C.c_void_p), ("indices", C.c_void_p),
                ("texture", C.c_void_p), ("num_vertices", C.c_uint32), ("num_triangles", C.c_uint32),
                ("tex_w", C.c_uint32), ("tex_h", C.c_uint32), ("normals", C.c_void_p)]


class _Bands(C.Structure):
    _fields_ = [("tex", C.c_void_p * 4), ("w", C.c_uint32 * 4), ("h", C.c_uint32 * 4)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(ensure_built())
        L.vso_render.restype = C.c_int
        L.vso_render.argtypes = [C.POINTER(_Layer), C.c_uint32, C.c_uint32, C.c_int, C.c_void_p,
                                 C.c_uint32, C.c_uint32, C.c_float, C.c_double, C.c_void_p,
                                 C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                 C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L.vso_render_banded.restype = C.c_int
        L.vso_render_banded.argtypes = [C.POINTER(_Layer), C.POINTER(_Bands), C.c_double, C.c_double, C.c_uint32, C.c_uint32,
                                        C.c_void_p, C.c_uint32, C.c_uint32, C.c_float, C.c_double, C.c_void_p,
                                        C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                        C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        L.vso_render_backward.restype = C.c_int
        L.vso_render_backward.argtypes = [C.POINTER(_Layer), C.c_uint32, C.c_uint32, C.c_int, C.c_void_p, C.c_uint32, C.c_uint32,
                                          C.c_float, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p),
                                          C.c_int, C.c_int]
        L.vso_quantize.restype = C.c_double
        L.vso_quantize.argtypes = [C.c_double]
        L.vso_rescale.restype = C.c_double
        L.vso_rescale.argtypes = [C.c_double, C.c_double, C.c_double]
        L.vso_sample_banded.argtypes = [C.POINTER(_Bands), C.c_uint32, C.c_double, C.c_double, C.c_double, C.c_double, C.c_void_p]
        L.vso_alpha_attenuation.restype = C.c_double
        L.vso_alpha_attenuation.argtypes = [C.c_void_p, C.c_void_p]
        L.vso_face_normal.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.vso_interp_normal.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.vso_half_to_double.restype = C.c_double
        L.vso_half_to_double.argtypes = [C.c_uint16]
        L.vso_sh_basis.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
        L.vso_sample_bilinear.argtypes = [C.c_void_p, C.c_int, C.c_uint32, C.c_uint32, C.c_uint32,
                                          C.c_double, C.c_double, C.c_void_p]
        L.vso_decode_rgba.argtypes = [C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p]
        L.vso_blend.argtypes = [C.c_uint32, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]
        L.vso_transform_vertex.argtypes = [C.c_void_p, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p,
                                           C.c_void_p, C.c_void_p]
        L.vso_max_threads.restype = C.c_int
        L.vso_count_footprints.restype = C.c_int
        L.vso_count_footprints.argtypes = [C.POINTER(_Layer), C.c_uint32, C.c_uint32, C.c_uint32, C.c_double, C.c_void_p,
                                           C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p), C.c_void_p]
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def _dtype_code(tex: np.ndarray) -> int:
    if tex.dtype == np.float32:
        return 0
    if tex.dtype == np.float16:
        return 1
    raise TypeError("texture dtype must be float32 or float16")


def max_threads() -> int:
    return int(lib().vso_max_threads())


def render_view(layers, sh_degree: int, camera, width: int, height: int, *, near_plane: float = 0.05,
                t_min: float = 2.0 ** -14, background=(0.0, 0.0, 0.0), num_threads: int = 0,
                want_qp: bool = False, want_layer_rgba: bool = False, want_layer_uv: bool = False,
                attenuation: bool = False, v_range=None, want_layer_normal: bool = False):
    """Render one view.  `layers`: objects with positions/uvs/indices/texture numpy arrays
    (outermost first); layers with a `band_textures` list (uint8 [h_b, w_b, 2b+1, 4] per SH band) are
    rendered in the paper's banded 8-bit format, re-scaled to `v_range` = (v_min, v_max).
    Returns dict(rgba [H,W,4] f64, ids [k,H,W] u32, stats [2] u64, ...)."""
    k = len(layers)
    n = (sh_degree + 1) ** 2
    keep = []
    arr = (_Layer * k)()
    banded = getattr(layers[0], "band_textures", None) is not None
    bands = (_Bands * k)() if banded else None
    code = None
    for i, L in enumerate(layers):
        pos = np.ascontiguousarray(L.positions, dtype=np.float32)
        uv = np.ascontiguousarray(L.uvs, dtype=np.float32)
        idx = np.ascontiguousarray(L.indices, dtype=np.uint32)
        assert pos.ndim == 2 and pos.shape[1] == 3 and uv.shape == (pos.shape[0], 2)
        assert idx.ndim == 2 and idx.shape[1] == 3
        assert idx.size == 0 or int(idx.max()) < pos.shape[0]
        keep += [pos, uv, idx]
        nrm = getattr(L, "normals", None)
        if nrm is not None:
            nrm = np.ascontiguousarray(nrm, dtype=np.float32)
            assert nrm.shape == pos.shape
            keep.append(nrm)
        nptr = _ptr(nrm) if nrm is not None else None
        if banded:
            assert len(L.band_textures) == sh_degree + 1 and v_range is not None
            for b, t in enumerate(L.band_textures):
                t = np.ascontiguousarray(t)
                assert t.dtype == np.uint8 and t.ndim == 4 and t.shape[2] == 2 * b + 1 and t.shape[3] == 4, t.shape
                keep.append(t)
                bands[i].tex[b] = t.ctypes.data
                bands[i].w[b], bands[i].h[b] = t.shape[1], t.shape[0]
            arr[i] = _Layer(_ptr(pos), _ptr(uv), _ptr(idx), None, pos.shape[0], idx.shape[0], 0, 0, nptr)
            continue
        tex = np.ascontiguousarray(L.texture)
        c = _dtype_code(tex)
        if code is None:
            code = c
        assert c == code, "all layers must share one texture dtype"
        assert tex.ndim == 4 and tex.shape[2] == n and tex.shape[3] == 4, tex.shape
        keep.append(tex)
        arr[i] = _Layer(_ptr(pos), _ptr(uv), _ptr(idx), _ptr(tex), pos.shape[0], idx.shape[0],
                        tex.shape[1], tex.shape[0], nptr)
    cam = np.ascontiguousarray(camera, dtype=np.float32)
    assert cam.shape == (16,)
    bg = np.asarray(background, dtype=np.float64)
    rgba = np.empty((height, width, 4), dtype=np.float64)
    ids = np.empty((k, height, width), dtype=np.uint32)
    qp = np.empty((k, height, width), dtype=np.float32) if want_qp else None
    lrgba = np.empty((k, height, width, 4), dtype=np.float64) if want_layer_rgba else None
    luv = np.empty((k, height, width, 2), dtype=np.float64) if want_layer_uv else None
    lnrm = np.empty((k, height, width, 3), dtype=np.float64) if want_layer_normal else None
    stats = np.zeros(2, dtype=np.uint64)
    tail = (_ptr(rgba), _ptr(ids), _ptr(qp) if want_qp else None,
            _ptr(lrgba) if want_layer_rgba else None, _ptr(luv) if want_layer_uv else None,
            _ptr(stats), num_threads, 1 if attenuation else 0, _ptr(lnrm) if want_layer_normal else None)
    if banded:
        rc = lib().vso_render_banded(arr, bands, float(v_range[0]), float(v_range[1]), k, sh_degree, _ptr(cam), width,
                                     height, near_plane, t_min, _ptr(bg), *tail)
    else:
        rc = lib().vso_render(arr, k, sh_degree, code, _ptr(cam), width, height, near_plane, t_min, _ptr(bg), *tail)
    if rc != 0:
        raise ValueError("vso_render rejected its arguments (rc=%d)" % rc)
    out = dict(rgba=rgba, ids=ids, stats=stats)
    if want_qp:
        out["qp"] = qp
    if want_layer_rgba:
        out["layer_rgba"] = lrgba
    if want_layer_uv:
        out["layer_uv"] = luv
    if want_layer_normal:
        out["layer_normal"] = lnrm
    return out


def render_backward(layers, sh_degree: int, camera, width: int, height: int, ids, grad_out, grad_tex=None, *,
                    near_plane: float = 0.05, t_min: float = 2.0 ** -14, background=(0.0, 0.0, 0.0),
                    attenuation: bool = False, num_threads: int = 0):
    """Accumulate dL/d(texture) of every layer for one view, given the forward ids of that view and the upstream
    gradient grad_out [H,W,4].  grad_tex: list of float64 arrays shaped like the textures (created as zeros if None);
    an entry may be None: that layer's gradient is then not computed.  Returned."""
    k = len(layers)
    arr = (_Layer * k)()
    keep, code = [], None
    for i, L in enumerate(layers):
        pos = np.ascontiguousarray(L.positions, dtype=np.float32)
        uv = np.ascontiguousarray(L.uvs, dtype=np.float32)
        idx = np.ascontiguousarray(L.indices, dtype=np.uint32)
        tex = np.ascontiguousarray(L.texture)
        code = _dtype_code(tex)
        keep += [pos, uv, idx, tex]
        nrm = getattr(L, "normals", None)
        if nrm is not None:
            nrm = np.ascontiguousarray(nrm, dtype=np.float32)
            keep.append(nrm)
        arr[i] = _Layer(_ptr(pos), _ptr(uv), _ptr(idx), _ptr(tex), pos.shape[0], idx.shape[0], tex.shape[1], tex.shape[0],
                        _ptr(nrm) if nrm is not None else None)
    if grad_tex is None:
        grad_tex = [np.zeros(L.texture.shape, dtype=np.float64) for L in layers]
    for gt, L in zip(grad_tex, layers):
        assert gt is None or (gt.dtype == np.float64 and gt.flags.c_contiguous and gt.shape == L.texture.shape)
    gptr = (C.c_void_p * k)(*[None if g is None else g.ctypes.data for g in grad_tex])
    cam = np.ascontiguousarray(camera, dtype=np.float32)
    bg = np.asarray(background, dtype=np.float64)
    ids = np.ascontiguousarray(ids, dtype=np.uint32)
    go = np.ascontiguousarray(grad_out, dtype=np.float64)
    assert ids.shape == (k, height, width) and go.shape == (height, width, 4)
    rc = lib().vso_render_backward(arr, k, sh_degree, code, _ptr(cam), width, height, near_plane, t_min, _ptr(bg),
                                   _ptr(ids), _ptr(go), gptr, 1 if attenuation else 0, num_threads)
    if rc != 0:
        raise ValueError("vso_render_backward rejected its arguments (rc=%d)" % rc)
    return grad_tex


def count_footprints(layers, width: int, height: int, view, *, t_min: float = 2.0 ** -14, marks=None):
    """Footprint census of one rendered view (SURVEY.md §8(d) "counted, not assumed"): `view` is the dict returned by
    render_view(..., want_layer_rgba=True, want_layer_uv=True) with the same t_min.  `marks`: list of uint8 [tex_h, tex_w]
    arrays (one per layer; zeros are created if None) that accumulate the referenced texels.
    Returns (composited_fragments, newly_marked_texels, marks)."""
    k = len(layers)
    arr = (_Layer * k)()
    sizes = []
    for i, L in enumerate(layers):
        th, tw = (L.band_textures[0].shape[:2] if getattr(L, "band_textures", None) is not None else L.texture.shape[:2])
        sizes.append((th, tw))
        arr[i] = _Layer(None, None, None, None, 0, 0, tw, th, None)
    if marks is None:
        marks = [np.zeros(s, dtype=np.uint8) for s in sizes]
    for m, s in zip(marks, sizes):
        assert m.dtype == np.uint8 and m.flags.c_contiguous and m.shape == s
    mptr = (C.c_void_p * k)(*[m.ctypes.data for m in marks])
    ids = np.ascontiguousarray(view["ids"], dtype=np.uint32)
    lrgba = np.ascontiguousarray(view["layer_rgba"], dtype=np.float64)
    luv = np.ascontiguousarray(view["layer_uv"], dtype=np.float64)
    assert ids.shape == (k, height, width) and lrgba.shape == (k, height, width, 4) and luv.shape == (k, height, width, 2)
    out = np.zeros(2, dtype=np.uint64)
    rc = lib().vso_count_footprints(arr, k, width, height, float(t_min), _ptr(ids), _ptr(lrgba), _ptr(luv), mptr, _ptr(out))
    if rc != 0:
        raise ValueError("vso_count_footprints rejected its arguments (rc=%d)" % rc)
    return int(out[0]), int(out[1]), marks


def render_scene(scene, views=None, **kw):
    """Render the given view indices (default: all) of a synth.Scene; returns a list of dicts."""
    views = range(len(scene.cameras)) if views is None else views
    kw.setdefault("near_plane", scene.near_plane)
    kw.setdefault("t_min", scene.t_min)
    kw.setdefault("background", scene.background)
    if getattr(scene, "v_range", None) is not None:
        kw.setdefault("v_range", scene.v_range)
    return [render_view(scene.layers, scene.sh_degree, scene.cameras[v], scene.width, scene.height, **kw)
            for v in views]


# ---- single-function entry points, used by the pins -------------------------------------------

def half_to_double(bits: int) -> float:
    return float(lib().vso_half_to_double(int(bits)))


def sh_basis(degree: int, v) -> np.ndarray:
    v = np.ascontiguousarray(v, dtype=np.float64)
    Y = np.zeros(16, dtype=np.float64)
    lib().vso_sh_basis(degree, _ptr(v), _ptr(Y))
    return Y[: (degree + 1) ** 2]


def sample_bilinear(tex: np.ndarray, u: float, v: float) -> np.ndarray:
    tex = np.ascontiguousarray(tex)
    H, W, n, _ = tex.shape
    out = np.empty((n, 4), dtype=np.float64)
    lib().vso_sample_bilinear(_ptr(tex), _dtype_code(tex), W, H, n, float(u), float(v), _ptr(out))
    return out


def decode_rgba(coef: np.ndarray, Y: np.ndarray) -> np.ndarray:
    coef = np.ascontiguousarray(coef, dtype=np.float64)
    Y = np.ascontiguousarray(Y, dtype=np.float64)
    out = np.empty(4, dtype=np.float64)
    lib().vso_decode_rgba(coef.shape[0], _ptr(coef), _ptr(Y), _ptr(out))
    return out


def quantize(x: float) -> float:
    return float(lib().vso_quantize(float(x)))


def rescale(q: float, v_min: float, v_max: float) -> float:
    return float(lib().vso_rescale(float(q), float(v_min), float(v_max)))


def sample_banded(band_textures, v_min: float, v_max: float, u: float, v: float) -> np.ndarray:
    deg = len(band_textures) - 1
    B = _Bands()
    keep = []
    for b, t in enumerate(band_textures):
        t = np.ascontiguousarray(t, dtype=np.uint8)
        keep.append(t)
        B.tex[b] = t.ctypes.data
        B.w[b], B.h[b] = t.shape[1], t.shape[0]
    out = np.empty(((deg + 1) ** 2, 4), dtype=np.float64)
    lib().vso_sample_banded(C.byref(B), deg, float(v_min), float(v_max), float(u), float(v), _ptr(out))
    return out


def alpha_attenuation(v, n) -> float:
    v = np.ascontiguousarray(v, dtype=np.float64)
    n = np.ascontiguousarray(n, dtype=np.float64)
    return float(lib().vso_alpha_attenuation(_ptr(v), _ptr(n)))


def interp_normal(b, n0, n1, n2) -> np.ndarray:
    b = np.ascontiguousarray(b, dtype=np.float64)
    ns = [np.ascontiguousarray(n, dtype=np.float32) for n in (n0, n1, n2)]
    out = np.empty(3, dtype=np.float64)
    lib().vso_interp_normal(_ptr(b), _ptr(ns[0]), _ptr(ns[1]), _ptr(ns[2]), _ptr(out))
    return out


def face_normal(p0, p1, p2) -> np.ndarray:
    ps = [np.ascontiguousarray(p, dtype=np.float32) for p in (p0, p1, p2)]
    n = np.empty(3, dtype=np.float64)
    lib().vso_face_normal(_ptr(ps[0]), _ptr(ps[1]), _ptr(ps[2]), _ptr(n))
    return n


def blend(layer_rgba, hit=None, t_min: float = 0.0, background=(0.0, 0.0, 0.0)) -> np.ndarray:
    layer_rgba = np.ascontiguousarray(layer_rgba, dtype=np.float64)
    k = layer_rgba.shape[0]
    hit = np.ones(k, dtype=np.int32) if hit is None else np.ascontiguousarray(hit, dtype=np.int32)
    bg = np.asarray(background, dtype=np.float64)
    out = np.empty(4, dtype=np.float64)
    lib().vso_blend(k, _ptr(layer_rgba), _ptr(hit), float(t_min), _ptr(bg), _ptr(out))
    return out


def transform_vertex(camera, near_plane: float, p):
    cam = np.ascontiguousarray(camera, dtype=np.float32)
    p = np.ascontiguousarray(p, dtype=np.float32)
    X, Y, bad = C.c_int32(), C.c_int32(), C.c_int32()
    q = C.c_float()
    lib().vso_transform_vertex(_ptr(cam), near_plane, _ptr(p), C.byref(X), C.byref(Y), C.byref(q), C.byref(bad))
    return X.value, Y.value, q.value, bad.value

"""Thin ctypes binding of the C-ABI library (include/vs.h): argument marshalling only -- every step
of the path runs in the CUDA kernels of libvs_b200.so.  PyTorch supplies device memory and streams.

There is no fallback: if the library is missing and cannot be built, or no CUDA device is present,
the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libvs_b200.so")

VS_OK, VS_ERR_INVALID_ARG, VS_ERR_OUT_OF_MEMORY, VS_ERR_CUDA, VS_ERR_UNSUPPORTED = range(5)
VS_F32, VS_F16 = 0, 1
VS_MEM_DEVICE, VS_MEM_HOST = 0, 1
VS_FLAG_REFERENCE_PATH, VS_FLAG_KERNEL_TIMING, VS_FLAG_COUNT_TEXELS, VS_FLAG_TILED_PATH = 1, 2, 4, 8
VS_FLAG_ATTENUATION = 16
VS_FLAG_OVERLAP = 32
VS_FLAG_SCREEN_ORDER = 64
VS_FLAG_PLAIN_BACKWARD = 128
VS_STATIC_SCRATCH_BYTES = 64 << 20   # vs_render_static: size of the library's static device scratch
MISS = 0xFFFFFFFF

EXPORTS = ["vs_scene_create", "vs_scene_create_banded", "vs_scene_set_vertex_normals", "vs_render", "vs_render_aov", "vs_render_backward", "vs_render_host", "vs_render_static", "vs_query_last_render", "vs_scene_destroy",
           "vs_last_error", "vs_version"]


class VsError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("vs status %d: %s" % (status, msg))
        self.status = status


class vs_layer_desc(C.Structure):
    _fields_ = [("positions", C.c_void_p), ("uvs", C.c_void_p), ("num_vertices", C.c_uint32),
                ("indices", C.c_void_p), ("num_triangles", C.c_uint32), ("texture", C.c_void_p),
                ("tex_w", C.c_uint32), ("tex_h", C.c_uint32)]


class vs_scene_desc(C.Structure):
    _fields_ = [("num_layers", C.c_uint32), ("sh_degree", C.c_uint32), ("tex_dtype", C.c_int),
                ("memory", C.c_int), ("layers", C.POINTER(vs_layer_desc))]


class vs_layer_desc_banded(C.Structure):
    _fields_ = [("positions", C.c_void_p), ("uvs", C.c_void_p), ("num_vertices", C.c_uint32),
                ("indices", C.c_void_p), ("num_triangles", C.c_uint32), ("band_texture", C.c_void_p * 4),
                ("band_w", C.c_uint32 * 4), ("band_h", C.c_uint32 * 4)]


class vs_scene_desc_banded(C.Structure):
    _fields_ = [("num_layers", C.c_uint32), ("sh_degree", C.c_uint32), ("memory", C.c_int),
                ("v_min", C.c_float), ("v_max", C.c_float), ("layers", C.POINTER(vs_layer_desc_banded))]


class vs_aov_buffers(C.Structure):
    _fields_ = [("tri_ids", C.c_void_p), ("layer_rgba", C.c_void_p), ("layer_uv", C.c_void_p), ("layer_normal", C.c_void_p)]


class vs_camera(C.Structure):
    _fields_ = [("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float), ("cy", C.c_float),
                ("R", C.c_float * 9), ("t", C.c_float * 3)]


class vs_render_params(C.Structure):
    _fields_ = [("width", C.c_uint32), ("height", C.c_uint32), ("near_plane", C.c_float),
                ("t_min", C.c_float), ("background", C.c_float * 3), ("flags", C.c_uint32),
                ("views_per_chunk", C.c_uint32)]


class vs_render_stats(C.Structure):
    _fields_ = [("dropped_triangles", C.c_uint64), ("degenerate_triangles", C.c_uint64),
                ("tile_refs", C.c_uint64), ("scratch_bytes", C.c_uint64), ("kernel_launches", C.c_uint64),
                ("raster_launches", C.c_uint64), ("shade_launches", C.c_uint64), ("shaded_fragments", C.c_uint64),
                ("unique_texels", C.c_uint64), ("ms_transform", C.c_double), ("ms_binning", C.c_double),
                ("ms_raster", C.c_double), ("ms_shade", C.c_double)]


_lib = None
# handle -> (k, n_coef, [(tex_h, tex_w)] per layer, banded): what the marshalling checks of the render calls need
_SCENES = {}


def _scene_info(scene):
    info = _SCENES.get(int(scene))
    if info is None:
        raise ValueError("unknown scene handle %r (not created through this binding, or already destroyed)" % (scene,))
    return info


def load_library(build_if_missing: bool = True):
    """dlopen libvs_b200.so (building it with nvcc first if it is absent or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing:
        from .build import ensure_built
        try:
            ensure_built()
        except Exception as e:  # no nvcc on this machine: use the shipped .so if there is one
            if not os.path.exists(LIB_PATH):
                raise RuntimeError("libvs_b200.so is missing and could not be built: %s" % e)
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("libvs_b200.so is missing (run `python -m paper_2409_02482_b200.build`)")
    L = C.CDLL(LIB_PATH)
    L.vs_scene_create.restype = C.c_int
    L.vs_scene_create.argtypes = [C.POINTER(vs_scene_desc), C.c_void_p, C.POINTER(C.c_void_p)]
    L.vs_scene_create_banded.restype = C.c_int
    L.vs_scene_create_banded.argtypes = [C.POINTER(vs_scene_desc_banded), C.c_void_p, C.POINTER(C.c_void_p)]
    for name in ("vs_render", "vs_render_host", "vs_render_static"):
        f = getattr(L, name)
        f.restype = C.c_int
        f.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32, C.POINTER(vs_render_params), C.c_void_p,
                      C.c_void_p, C.c_void_p]
    L.vs_render_aov.restype = C.c_int
    L.vs_render_aov.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32, C.POINTER(vs_render_params), C.c_void_p,
                                C.POINTER(vs_aov_buffers), C.c_void_p]
    L.vs_render_backward.restype = C.c_int
    L.vs_render_backward.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32, C.POINTER(vs_render_params), C.c_void_p,
                                     C.POINTER(C.c_void_p), C.c_void_p]
    L.vs_scene_set_vertex_normals.restype = C.c_int
    L.vs_scene_set_vertex_normals.argtypes = [C.c_void_p, C.POINTER(C.c_void_p), C.c_int, C.c_void_p]
    L.vs_query_last_render.restype = C.c_int
    L.vs_query_last_render.argtypes = [C.c_void_p, C.POINTER(vs_render_stats)]
    L.vs_scene_destroy.restype = None
    L.vs_scene_destroy.argtypes = [C.c_void_p]
    L.vs_last_error.restype = C.c_char_p
    L.vs_version.restype = C.c_char_p
    _lib = L
    return L


def _check(status):
    if status != VS_OK:
        raise VsError(status, load_library().vs_last_error().decode())


def _stream_ptr(stream):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def make_params(width, height, near_plane=0.05, t_min=2.0 ** -14, background=(0.0, 0.0, 0.0), flags=0,
                views_per_chunk=0):
    p = vs_render_params()
    p.width, p.height, p.near_plane, p.t_min = int(width), int(height), float(near_plane), float(t_min)
    p.background = (C.c_float * 3)(*[float(b) for b in background])
    p.flags, p.views_per_chunk = int(flags), int(views_per_chunk)
    return p


# ---- the C-ABI calls, same names ---------------------------------------------------------------

def vs_scene_create(layers, sh_degree: int, stream=None) -> int:
    """`layers`: sequence of objects with .positions [V,3] f32, .uvs [V,2] f32, .indices [T,3]
    u32/int32, .texture [H,W,n,4] f32|f16 -- all torch CUDA tensors (device pointers) or all numpy
    arrays (host pointers).  Returns the opaque scene handle."""
    import torch
    L = load_library()
    k = len(layers)
    arr = (vs_layer_desc * max(k, 1))()
    keep = []
    on_host = k > 0 and isinstance(layers[0].positions, np.ndarray)
    dtype_code = None
    for i, ly in enumerate(layers):
        if on_host:
            pos = np.ascontiguousarray(ly.positions, dtype=np.float32)
            uv = np.ascontiguousarray(ly.uvs, dtype=np.float32)
            idx = np.ascontiguousarray(ly.indices, dtype=np.uint32)
            tex = np.ascontiguousarray(ly.texture)
            code = {np.dtype(np.float32): VS_F32, np.dtype(np.float16): VS_F16}[tex.dtype]
            ptr = lambda a: a.ctypes.data
        else:
            pos = ly.positions.contiguous()
            uv = ly.uvs.contiguous()
            idx = ly.indices.contiguous()
            tex = ly.texture.contiguous()
            assert pos.is_cuda and uv.is_cuda and idx.is_cuda and tex.is_cuda
            assert pos.dtype == torch.float32 and uv.dtype == torch.float32
            assert idx.dtype in (torch.int32, torch.uint32)
            code = {torch.float32: VS_F32, torch.float16: VS_F16}[tex.dtype]
            ptr = lambda a: a.data_ptr()
        if dtype_code is None:
            dtype_code = code
        assert code == dtype_code, "all layers must share one texture dtype"
        assert tex.ndim == 4 and tex.shape[3] == 4 and tex.shape[2] == (sh_degree + 1) ** 2, tuple(tex.shape)
        keep += [pos, uv, idx, tex]
        arr[i] = vs_layer_desc(ptr(pos), ptr(uv), pos.shape[0], ptr(idx), idx.shape[0], ptr(tex),
                               tex.shape[1], tex.shape[0])
    desc = vs_scene_desc(k, sh_degree, dtype_code or 0, VS_MEM_HOST if on_host else VS_MEM_DEVICE, arr)
    handle = C.c_void_p()
    _check(L.vs_scene_create(C.byref(desc), _stream_ptr(stream), C.byref(handle)))
    _SCENES[handle.value] = (k, (sh_degree + 1) ** 2, [(int(ly.texture.shape[0]), int(ly.texture.shape[1])) for ly in layers], False)
    return handle.value


def vs_scene_create_banded(layers, sh_degree: int, v_min: float, v_max: float, stream=None) -> int:
    """The paper's banded 8-bit format: `layers` as for vs_scene_create but with .band_textures = list of
    sh_degree + 1 uint8 arrays [H_b, W_b, 2b+1, 4] instead of .texture (all torch CUDA tensors or all numpy arrays)."""
    L = load_library()
    k = len(layers)
    arr = (vs_layer_desc_banded * max(k, 1))()
    keep = []
    on_host = k > 0 and isinstance(layers[0].positions, np.ndarray)
    for i, ly in enumerate(layers):
        assert len(ly.band_textures) == sh_degree + 1
        if on_host:
            pos = np.ascontiguousarray(ly.positions, dtype=np.float32)
            uv = np.ascontiguousarray(ly.uvs, dtype=np.float32)
            idx = np.ascontiguousarray(ly.indices, dtype=np.uint32)
            bands = [np.ascontiguousarray(t, dtype=np.uint8) for t in ly.band_textures]
            ptr = lambda a: a.ctypes.data
        else:
            pos, uv, idx = ly.positions.contiguous(), ly.uvs.contiguous(), ly.indices.contiguous()
            bands = [t.contiguous() for t in ly.band_textures]
            assert pos.is_cuda and uv.is_cuda and idx.is_cuda and all(t.is_cuda and t.element_size() == 1 for t in bands)
            ptr = lambda a: a.data_ptr()
        keep += [pos, uv, idx] + bands
        d = vs_layer_desc_banded()
        d.positions, d.uvs, d.num_vertices = ptr(pos), ptr(uv), pos.shape[0]
        d.indices, d.num_triangles = ptr(idx), idx.shape[0]
        for b, t in enumerate(bands):
            assert t.ndim == 4 and t.shape[2] == 2 * b + 1 and t.shape[3] == 4, tuple(t.shape)
            d.band_texture[b] = ptr(t)
            d.band_w[b], d.band_h[b] = t.shape[1], t.shape[0]
        arr[i] = d
    desc = vs_scene_desc_banded(k, sh_degree, VS_MEM_HOST if on_host else VS_MEM_DEVICE, float(v_min), float(v_max), arr)
    handle = C.c_void_p()
    _check(L.vs_scene_create_banded(C.byref(desc), _stream_ptr(stream), C.byref(handle)))
    _SCENES[handle.value] = (k, (sh_degree + 1) ** 2, [(int(ly.band_textures[0].shape[0]), int(ly.band_textures[0].shape[1])) for ly in layers], True)
    return handle.value


def vs_scene_set_vertex_normals(scene: int, normals, stream=None):
    """normals: one entry per layer, a [V_l, 3] float32 array (all numpy = host memory, or all CUDA tensors) or None."""
    k = _scene_info(scene)[0]
    assert len(normals) == k, "normals: %d entries for a scene of %d layers" % (len(normals), k)
    given = [n for n in normals if n is not None]
    on_host = bool(given) and isinstance(given[0], np.ndarray)
    keep, ptrs = [], (C.c_void_p * k)()
    for l, n in enumerate(normals):
        if n is None:
            continue
        if on_host:
            n = np.ascontiguousarray(n, dtype=np.float32)
            ptrs[l] = n.ctypes.data
        else:
            import torch
            assert n.is_cuda and n.dtype == torch.float32
            n = n.contiguous()
            ptrs[l] = n.data_ptr()
        assert n.ndim == 2 and n.shape[1] == 3, tuple(n.shape)
        keep.append(n)
    _check(load_library().vs_scene_set_vertex_normals(scene, ptrs, VS_MEM_HOST if on_host or not given else VS_MEM_DEVICE,
                                                      _stream_ptr(stream)))


def _cams(cameras):
    cams = np.ascontiguousarray(cameras, dtype=np.float32)
    assert cams.ndim == 2 and cams.shape[1] == 16
    return cams


def vs_render(scene: int, cameras, params: vs_render_params, out_rgba, out_tri_ids=None, stream=None):
    """cameras: HOST [B,16] float32; out_rgba: CUDA float32 [B,H,W,4]; out_tri_ids: CUDA int32/uint32
    [B,k,H,W] or None.  Asynchronous on `stream` (default: torch's current stream): the call returns once the work is
    enqueued (the cameras have been copied by then); only the per-tile path (VS_FLAG_TILED_PATH) waits for its overflow check."""
    import torch
    cams = _cams(cameras)
    k = _scene_info(scene)[0]
    px = cams.shape[0] * params.width * params.height
    assert out_rgba.is_cuda and out_rgba.is_contiguous() and out_rgba.dtype == torch.float32 and out_rgba.numel() == px * 4
    ids_ptr = None
    if out_tri_ids is not None:
        assert out_tri_ids.is_cuda and out_tri_ids.is_contiguous() and out_tri_ids.element_size() == 4 and out_tri_ids.numel() == px * k
        ids_ptr = out_tri_ids.data_ptr()
    _check(load_library().vs_render(scene, cams.ctypes.data, cams.shape[0], C.byref(params),
                                    out_rgba.data_ptr(), ids_ptr, _stream_ptr(stream)))


def vs_render_static(scene: int, cameras, params: vs_render_params, out_rgba, out_tri_ids=None, stream=None):
    """vs_render without any allocation: all scratch in the library's static 64 MiB device array (include/vs.h).  Same
    arguments as vs_render; raises VsError(VS_ERR_UNSUPPORTED) when the call does not fit.  Calls that overlap on the GPU race."""
    import torch
    cams = _cams(cameras)
    k = _scene_info(scene)[0]
    px = cams.shape[0] * params.width * params.height
    assert out_rgba.is_cuda and out_rgba.is_contiguous() and out_rgba.dtype == torch.float32 and out_rgba.numel() == px * 4
    ids_ptr = None
    if out_tri_ids is not None:
        assert out_tri_ids.is_cuda and out_tri_ids.is_contiguous() and out_tri_ids.element_size() == 4 and out_tri_ids.numel() == px * k
        ids_ptr = out_tri_ids.data_ptr()
    _check(load_library().vs_render_static(scene, cams.ctypes.data, cams.shape[0], C.byref(params),
                                           out_rgba.data_ptr(), ids_ptr, _stream_ptr(stream)))


def vs_render_aov(scene: int, cameras, params: vs_render_params, out_rgba, tri_ids=None, layer_rgba=None, layer_uv=None,
                  layer_normal=None, stream=None):
    """vs_render plus the per-layer buffers (CUDA tensors or None): tri_ids [B,k,H,W] int32, layer_rgba [B,k,H,W,4],
    layer_uv [B,k,H,W,2], layer_normal [B,k,H,W,3] float32."""
    import torch
    cams = _cams(cameras)
    k = _scene_info(scene)[0]
    px = cams.shape[0] * params.width * params.height
    assert out_rgba.is_cuda and out_rgba.is_contiguous() and out_rgba.dtype == torch.float32 and out_rgba.numel() == px * 4
    a = vs_aov_buffers()
    for name, t, per_px in (("tri_ids", tri_ids, 1), ("layer_rgba", layer_rgba, 4), ("layer_uv", layer_uv, 2), ("layer_normal", layer_normal, 3)):
        if t is not None:
            assert t.is_cuda and t.is_contiguous() and t.element_size() == 4, name
            assert name == "tri_ids" or t.dtype == torch.float32, name
            assert t.numel() == px * k * per_px, "%s: %d elements, expected %d" % (name, t.numel(), px * k * per_px)
            setattr(a, name, t.data_ptr())
    _check(load_library().vs_render_aov(scene, cams.ctypes.data, cams.shape[0], C.byref(params), out_rgba.data_ptr(),
                                        C.byref(a), _stream_ptr(stream)))


def vs_render_backward(scene: int, cameras, params: vs_render_params, grad_rgba, grad_textures, stream=None):
    """grad_rgba: CUDA float32 [B,H,W,4]; grad_textures: list of k CUDA float32 tensors [tex_h,tex_w,n,4], accumulated into."""
    cams = _cams(cameras)
    assert grad_rgba.is_cuda and grad_rgba.is_contiguous() and grad_rgba.numel() == cams.shape[0] * params.width * params.height * 4
    import torch
    k, n_coef, tex_sizes, banded = _scene_info(scene)
    assert grad_rgba.dtype == torch.float32
    # the C side reads grad_textures[l] for every l < k and scatters at offsets derived from the SCENE's texture shapes
    assert len(grad_textures) == k, "grad_textures: %d tensors for a scene of %d layers" % (len(grad_textures), k)
    for l, t in enumerate(grad_textures):
        assert t.is_cuda and t.is_contiguous() and t.dtype == torch.float32, "grad_textures[%d]" % l
        if banded:
            continue          # the library rejects banded scenes itself (VS_ERR_UNSUPPORTED) before touching any tensor
        assert tuple(t.shape) == (tex_sizes[l][0], tex_sizes[l][1], n_coef, 4), \
            "grad_textures[%d]: shape %s, expected %s" % (l, tuple(t.shape), (tex_sizes[l][0], tex_sizes[l][1], n_coef, 4))
        assert t.data_ptr() % 16 == 0, "grad_textures[%d] must be 16-byte aligned" % l
    ptrs = (C.c_void_p * len(grad_textures))(*[t.data_ptr() for t in grad_textures])
    _check(load_library().vs_render_backward(scene, cams.ctypes.data, cams.shape[0], C.byref(params), grad_rgba.data_ptr(),
                                             ptrs, _stream_ptr(stream)))


def vs_render_host(scene: int, cameras, params: vs_render_params, out_rgba, out_tri_ids=None, stream=None):
    """Same, with HOST outputs (numpy arrays or CPU torch tensors, pinned for async copies).  Blocks
    until the images are in the host buffers."""
    cams = _cams(cameras)
    k = _scene_info(scene)[0]
    px = cams.shape[0] * params.width * params.height

    def nelem(a):
        return a.size if isinstance(a, np.ndarray) else a.numel()

    def host_ptr(a):
        if isinstance(a, np.ndarray):
            assert a.flags.c_contiguous and a.itemsize == 4
            return a.ctypes.data
        assert not a.is_cuda and a.is_contiguous() and a.element_size() == 4
        return a.data_ptr()

    assert nelem(out_rgba) == px * 4, "out_rgba: %d elements, expected %d" % (nelem(out_rgba), px * 4)
    assert out_tri_ids is None or nelem(out_tri_ids) == px * k

    _check(load_library().vs_render_host(scene, cams.ctypes.data, cams.shape[0], C.byref(params),
                                         host_ptr(out_rgba), host_ptr(out_tri_ids) if out_tri_ids is not None else None,
                                         _stream_ptr(stream)))


def vs_query_last_render(scene: int) -> dict:
    st = vs_render_stats()
    _check(load_library().vs_query_last_render(scene, C.byref(st)))
    return {f: (float if t is C.c_double else int)(getattr(st, f)) for f, t in vs_render_stats._fields_}


def vs_scene_destroy(scene: int):
    if scene:
        _SCENES.pop(int(scene), None)
        load_library().vs_scene_destroy(scene)


def vs_version() -> str:
    return load_library().vs_version().decode()


# ---- convenience -----------------------------------------------------------------------------------

class Renderer:
    """Owns a scene handle built from a synth.Scene-like object (numpy arrays are uploaded through
    torch so that the descriptor carries device pointers)."""

    def __init__(self, scene, device="cuda:0"):
        import torch
        import types
        self.k = len(scene.layers)
        self.sh_degree = scene.sh_degree
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            self.handle = None
            layers = []
            banded = getattr(scene.layers[0], "band_textures", None) is not None
            for ly in scene.layers:
                if banded:
                    layers.append(types.SimpleNamespace(
                        positions=torch.from_numpy(np.ascontiguousarray(ly.positions, dtype=np.float32)).to(self.device),
                        uvs=torch.from_numpy(np.ascontiguousarray(ly.uvs, dtype=np.float32)).to(self.device),
                        indices=torch.from_numpy(np.ascontiguousarray(ly.indices, dtype=np.uint32).view(np.int32)).to(self.device),
                        band_textures=[torch.from_numpy(np.ascontiguousarray(t, dtype=np.uint8)).to(self.device)
                                       for t in ly.band_textures]))
                    continue
                layers.append(types.SimpleNamespace(
                    positions=torch.from_numpy(np.ascontiguousarray(ly.positions, dtype=np.float32)).to(self.device),
                    uvs=torch.from_numpy(np.ascontiguousarray(ly.uvs, dtype=np.float32)).to(self.device),
                    indices=torch.from_numpy(np.ascontiguousarray(ly.indices, dtype=np.uint32).view(np.int32)).to(self.device),
                    texture=torch.from_numpy(np.ascontiguousarray(ly.texture)).to(self.device)))
            if banded:
                self.handle = vs_scene_create_banded(layers, scene.sh_degree, scene.v_range[0], scene.v_range[1])
            else:
                self.handle = vs_scene_create(layers, scene.sh_degree)
            del layers
            torch.cuda.empty_cache()
            normals = [getattr(ly, "normals", None) for ly in scene.layers]
            if any(n is not None for n in normals):
                vs_scene_set_vertex_normals(self.handle, [None if n is None else np.ascontiguousarray(n, dtype=np.float32) for n in normals])

    def render(self, cameras, params, want_ids=False, out_rgba=None, out_ids=None):
        import torch
        B = len(cameras)
        with torch.cuda.device(self.device):
            if out_rgba is None:
                out_rgba = torch.empty((B, params.height, params.width, 4), dtype=torch.float32, device=self.device)
            if want_ids and out_ids is None:
                out_ids = torch.empty((B, self.k, params.height, params.width), dtype=torch.int32, device=self.device)
            vs_render(self.handle, cameras, params, out_rgba, out_ids)
        return out_rgba, out_ids

    def stats(self):
        return vs_query_last_render(self.handle)

    def close(self):
        if self.handle:
            vs_scene_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

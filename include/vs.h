/*
 * vs.h -- C ABI of the B200-native k-shell renderer for "Volumetric Surfaces" (arXiv 2409.02482).
 *
 * The library renders the paper's baked representation: k (1..9; the paper uses 3 <= k <= 9,
 * PAPER.md:L10) semi-transparent, UV-textured mesh shells, "rendered in fixed layer order from
 * outermost to innermost" with no sorting.  Per pixel and per
 * layer it finds the nearest fragment of that layer ("only sampling the first intersection with
 * each surface", PAPER.md:L101 Fig. "sampling" c), interpolates UV, fetches the layer's texture of
 * spherical-harmonics coefficients bilinearly at texel centres (§4.5),
 * decodes RGBA with the view direction (§4.5; view-dependent opacity L58, L118) and
 * blends the layers front to back in that fixed order (§4.2 "Surface Blending";
 * "rasterizes all meshes in a fixed order and blends them in the final frame buffer", L464).
 * The exact arithmetic (projection op order, 24.8 snapping, top-left rule, depth key, tie-break,
 * texel addressing, SH convention, activation, blend) is DESIGN.md §3; the readings of the paper it
 * rests on are DESIGN.md §5.
 *
 * Everything runs in hand-written CUDA kernels for sm_100a on ONE GPU (the current device of the
 * calling thread at vs_scene_create time).  There is no CPU fallback: without a usable CUDA device
 * every entry point returns VS_ERR_CUDA.
 *
 * Conventions
 *   - Plain C99, no torch / C++ types.  "DEVICE" = pointer to memory of the scene's GPU,
 *     "HOST" = ordinary host memory (pageable or pinned).
 *   - Every function returns a vs_status and never throws or aborts across the ABI.  On error
 *     nothing has been written to the outputs, *out_scene is NULL, and vs_last_error() describes
 *     the failure (thread-local string, valid until the next call on that thread).
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 */
#ifndef VS_H_
#define VS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vs_scene vs_scene; /* opaque */

typedef enum {
    VS_OK = 0,
    VS_ERR_INVALID_ARG = 1,   /* NULL pointer, k outside 1..9, degree > 3, zero size, index >= num_vertices,
                                 non-finite vertex / camera, near_plane <= 0, reserved flag bits set */
    VS_ERR_OUT_OF_MEMORY = 2, /* a device or host allocation failed */
    VS_ERR_CUDA = 3,          /* no device, or a CUDA call / kernel failed; see vs_last_error() */
    VS_ERR_UNSUPPORTED = 4    /* e.g. image larger than 16384 px on a side, texture larger than 32768 */
} vs_status;

typedef enum { VS_F32 = 0, VS_F16 = 1 } vs_dtype;           /* texture element type (IEEE binary32/16) */
typedef enum { VS_MEM_DEVICE = 0, VS_MEM_HOST = 1 } vs_memory; /* where a descriptor's arrays live */

/* One shell ("Mesh baking": a lightweight UV-mapped triangle mesh per surface;
 * §4.5: per mesh, (deg+1)^2 RGBA coefficient images -- here one interleaved array). */
typedef struct {
    const float*    positions;     /* [num_vertices][3] world space, finite                              */
    const float*    uvs;           /* [num_vertices][2]; seams = duplicated vertices; values outside
                                      [0,1] are legal and clamp to the edge texels                       */
    uint32_t        num_vertices;
    const uint32_t* indices;       /* [num_triangles][3]; triangle id = row index; any winding
                                      (no culling: both orientations rasterise, the nearest wins)         */
    uint32_t        num_triangles; /* 0 is legal (an empty shell never hits)                             */
    const void*     texture;       /* [tex_h][tex_w][(deg+1)^2][4]; channel 0-2 = RGB, 3 = opacity;
                                      raw (pre-sigmoid) SH coefficients, coefficient index c = l*l+l+m;
                                      row j of memory is v-row j (no flip)                                */
    uint32_t        tex_w, tex_h;  /* >= 1, <= 32768                                                       */
} vs_layer_desc;

typedef struct {
    uint32_t             num_layers; /* 1..9; layers[0] is the OUTERMOST shell                            */
    uint32_t             sh_degree;  /* 0..3, shared by colour and opacity                                 */
    vs_dtype             tex_dtype;  /* all layers share one element type                                  */
    vs_memory            memory;     /* where positions / uvs / indices / texture of ALL layers live      */
    const vs_layer_desc* layers;     /* HOST array of num_layers descriptors                               */
} vs_scene_desc;

/* Pinhole camera (the paper gives none).  x_cam = R * x_world + t with
 * +x right, +y DOWN, +z forward; pixel (i,j) has its centre at (i+0.5, j+0.5), origin top-left. */
typedef struct {
    float fx, fy, cx, cy; /* pixels */
    float R[9];           /* row-major */
    float t[3];
} vs_camera;

enum {
    VS_FLAG_REFERENCE_PATH = 1u << 0, /* debugging aid: brute-force kernel (one thread per pixel, every
                                         triangle tested), same arithmetic and outputs; small scenes only */
    VS_FLAG_KERNEL_TIMING  = 1u << 1, /* bracket every kernel launch with CUDA events on the render stream
                                         and report per-stage device time in vs_render_stats              */
    VS_FLAG_TILED_PATH     = 1u << 3, /* rasterise through per-tile triangle lists (count / scan / scatter binning
                                         + one CTA per 16x16 tile with shared-memory keys) instead of the
                                         default triangle-parallel path (64-bit max keys in HBM/L2); same
                                         outputs bit for bit                                                */
    VS_FLAG_COUNT_TEXELS   = 1u << 2, /* measurement aid: count shaded fragments and, per view, the UNIQUE
                                         texels their 2x2 footprints reference (the algorithmic texture
                                         bytes of DESIGN.md §8); slower, not for timed runs                */
    VS_FLAG_OVERLAP        = 1u << 5, /* experiment: run S1-S4 of the next chunk of cameras on an internal
                                         high-priority stream, in one resident CTA per SM, beside S5-S7 of the current
                                         chunk instead of back to back on `cuda_stream`; same outputs bit for bit
                                         (measured slower on B200; off by default)                            */
    VS_FLAG_SCREEN_ORDER   = 1u << 6, /* shade the (view, tile) pairs of a pass in screen order (view by view) instead of the
                                         default SURFACE order, in which the tiles of all views of a pass that look at the
                                         same part of the object are shaded together so that their texels are shared
                                         through L2; same outputs bit for bit; for A/B measurements        */
    VS_FLAG_PLAIN_BACKWARD = 1u << 7, /* vs_render_backward only: the first backward kernel (k_backward: one lane per pixel
                                         re-shades its fragments with the plain per-lane routine) instead of the default
                                         k_shade<BWD>, which shares k_shade's octet / tensor-core forward pass; same
                                         gradients up to the fp32 summation order; for A/B measurements and cross-checks  */
    VS_FLAG_ATTENUATION    = 1u << 4  /* transparency attenuation (§4.2 "Transparency
                                         Attenuation"): every fragment's opacity is multiplied by
                                         alpha_w = 2 Sigmoid(10 |v . n|) - 1 before blending, v = the pixel's
                                         unit view direction, n = the unit geometric normal of the fragment's
                                         triangle in world space, or the interpolated per-vertex normal of layers
                                         given some (vs_scene_set_vertex_normals; reading Q13); off by default */
};

typedef struct {
    uint32_t width, height;   /* 1..16384                                                                  */
    float    near_plane;      /* > 0; a triangle with any vertex at depth w < near_plane is DROPPED (not
                                 clipped), as is one with a vertex projecting outside +-16384 px           */
    float    t_min;           /* >= 0; compositing stops after the layer that brings the transmittance
                                 below t_min (0 disables).  Recommended 2^-14 (reading Q15)      */
    float    background[3];   /* rgb_out = C + T * background ; (0,0,0) => premultiplied colour            */
    uint32_t flags;           /* VS_FLAG_* ; other bits must be 0                                          */
    uint32_t views_per_chunk; /* cameras processed per internal pass; 0 = choose automatically             */
} vs_render_params;

/* Counters of the most recent render call on a scene (summed over its cameras), plus the launch counts and the
 * VS_FLAG_KERNEL_TIMING stage times ACCUMULATED over all render calls since the previous vs_query_last_render (so that a
 * caller may time many asynchronous calls and pay one host wait). */
typedef struct {
    uint64_t dropped_triangles;    /* near-plane / guard-band drops (0 on all BASELINE.json configs)      */
    uint64_t degenerate_triangles; /* zero area after snapping                                             */
    uint64_t tile_refs;            /* (triangle, tile) pairs binned                                        */
    uint64_t scratch_bytes;        /* peak device scratch held by the scene so far                         */
    uint64_t kernel_launches;      /* kernels launched since the previous query (memsets / copies not counted) */
    uint64_t raster_launches;      /* of which k_raster (one per chunk of cameras)                         */
    uint64_t shade_launches;       /* of which k_shade  (one per chunk of cameras)                         */
    uint64_t shaded_fragments;     /* VS_FLAG_COUNT_TEXELS: (pixel, layer) fragments shaded                */
    uint64_t unique_texels;        /* VS_FLAG_COUNT_TEXELS: sum over views and layers of distinct texels   */
    double   ms_transform;         /* VS_FLAG_KERNEL_TIMING: device time per stage, summed since the previous query */
    double   ms_binning;           /*   count + scan + scatter                                             */
    double   ms_raster;            /*   coverage + nearest-fragment resolve kernel                         */
    double   ms_shade;             /*   texel fetch + SH + composite kernel                                */
} vs_render_stats;

/* The paper's own baked texture format (§4.5 "Mixed resolutions" and "Squeezing and
 * quantization"): 8-bit images, one set per SH band, band b at its OWN resolution
 * ("the base color is modeled at the highest resolution (2048^2), while the highest SH degree coefficients are
 * modeled at the lowest resolution (256^2)").  A stored byte t stands for q = t/255 (q(x) = round(255 x)/255 of the
 * squeezed coefficient); "before rendering, we re-scale value to a hyper-parameters controlled range":
 * sh = v_min + (v_max - v_min) q, [-15, 15] in the paper.  Each band is sampled bilinearly at its own texel
 * centres (same addressing rule as the float textures), re-scaled, and the bands are concatenated over the
 * coefficient dimension, c = b*b .. b*b + 2b. */
typedef struct {
    const float*    positions;       /* as vs_layer_desc                                                  */
    const float*    uvs;
    uint32_t        num_vertices;
    const uint32_t* indices;
    uint32_t        num_triangles;
    const uint8_t*  band_texture[4]; /* band b <= sh_degree: [band_h[b]][band_w[b]][2b+1][4] bytes; channel
                                        0-2 = RGB, 3 = opacity; coefficient order m = -b..b; others ignored */
    uint32_t        band_w[4], band_h[4]; /* >= 1, <= 8192                                                 */
} vs_layer_desc_banded;

typedef struct {
    uint32_t  num_layers;            /* 1..9; layers[0] is the OUTERMOST shell                            */
    uint32_t  sh_degree;             /* 0..3                                                               */
    vs_memory memory;                /* where the arrays of ALL layers live                                */
    float     v_min, v_max;          /* finite; range the bytes are re-scaled to                           */
    const vs_layer_desc_banded* layers; /* HOST array of num_layers descriptors                            */
} vs_scene_desc_banded;

/*
 * vs_scene_create_banded -- vs_scene_create for the banded 8-bit format.  The resulting scene is rendered
 * with the same vs_render / vs_render_host calls (S1-S4 are identical; S5-S6 run in a kernel specialised for
 * byte texels, k_shade_banded).  VS_FLAG_COUNT_TEXELS counts shaded fragments only on such scenes (no unique-texel
 * count).
 */
vs_status vs_scene_create_banded(const vs_scene_desc_banded* desc, void* cuda_stream, vs_scene** out_scene);

/*
 * vs_scene_create -- S0: upload / re-lay-out the baked asset once.
 *   Copies every array (the caller may free or overwrite its inputs as soon as the call returns: the
 *   function synchronises `cuda_stream` before returning), validates indices and finiteness, and
 *   converts each texture to the internal texel-interleaved layout.  The scene is
 *   immutable afterwards.  Device memory held: ~ sum over layers of 16 B/vertex... see DESIGN.md §6.
 */
vs_status vs_scene_create(const vs_scene_desc* desc, void* cuda_stream, vs_scene** out_scene);

/*
 * vs_scene_set_vertex_normals -- optional per-vertex normals for the transparency attenuation (
 * PAPER.md:L279-286 "the angle between the view direction and the surface normal").  Part of building the
 * scene: call it after vs_scene_create* and before rendering (it waits for the device; the scene is immutable while
 * renders are in flight).
 *   normals  HOST array of num_layers pointers; entry l is [num_vertices of layer l][3] floats in `memory` (finite, need
 *            not be unit length), or NULL: that layer keeps the geometric face normal of the hit triangle.
 * Under VS_FLAG_ATTENUATION a fragment of a layer WITH normals uses n = normalize(sum_i b'_i n_i), the three vertex normals
 * interpolated with the fragment's perspective-correct barycentrics (n = 0, hence alpha_w = 0, if the sum vanishes); the
 * layer_normal buffer of vs_render_aov reports the same vector.  Calling it again replaces the normals of the layers given
 * and drops those of the others.
 */
vs_status vs_scene_set_vertex_normals(vs_scene* scene, const float* const* normals, vs_memory memory, void* cuda_stream);

/*
 * vs_render -- the hot path, steps S1-S7 of DESIGN.md §1 for a batch of cameras:
 *   S1 vertex transform, S2 triangle setup + S4 coverage and per-layer nearest-fragment resolve (default: triangle-parallel
 *   with 64-bit maximum keys in HBM/L2; under VS_FLAG_TILED_PATH: S3 screen-tile binning by count / prefix sum / scatter, then
 *   one CTA per tile with the keys in shared memory), S5 perspective-correct UV + bilinear fetch, S6 SH evaluation + sigmoid,
 *   S7 fixed-order front-to-back compositing.
 *
 *   cameras      HOST  [num_cameras]; copied before the call returns (the caller may reuse the array at once)
 *   out_rgba     DEVICE [num_cameras][height][width][4] float: rgb = C + T*background, a = 1 - T.
 *                A pixel no layer hits is a value (background, alpha 0), not an error.
 *   out_tri_ids  DEVICE [num_cameras][num_layers][height][width] uint32 or NULL: id of the nearest
 *                covering triangle of each layer, 0xFFFFFFFF = miss (the AOV the parity tests read).
 *
 *   ASYNCHRONOUS: all work is enqueued on `cuda_stream` and the call returns without waiting for it; the outputs are
 *   complete when the stream reaches the end of the call's work (synchronise the stream, or keep enqueueing on it).
 *   Counters and kernel timings are fetched lazily by vs_query_last_render, the only host wait of the render API.
 *   Exception: under VS_FLAG_TILED_PATH the call waits once for the stream, because the per-tile triangle-reference list is
 *   sized from earlier calls and checked on the device; if a chunk of cameras needed more, the list is grown and the call
 *   renders again before returning.
 *   The scene itself is immutable.  What a call writes besides the caller's outputs lives in two scratch sets owned by the
 *   scene (transformed vertices, key image, tile masks), handed from user to user through CUDA events and grown with
 *   stream-ordered allocations from a pool private to the scene.  Calls on one scene from several host threads and on
 *   different streams are therefore LEGAL and give the same results as serial calls; they share the two sets, so their
 *   device work interleaves at the granularity of a chunk of cameras instead of overlapping freely (a deliberate limit:
 *   the key image of the direct path is kept zeroed between uses, which a per-call allocation could not offer without a
 *   multi-GB memset per call).
 */
vs_status vs_render(vs_scene* scene, const vs_camera* cameras, uint32_t num_cameras,
                    const vs_render_params* params, float* out_rgba, uint32_t* out_tri_ids,
                    void* cuda_stream);

/*
 * vs_render_host -- the same call with HOST output buffers (end-to-end path): renders chunk by
 * chunk into device staging and copies each finished chunk back while the next one renders.
 *   out_rgba / out_tri_ids  HOST, same shapes as vs_render (pinned memory makes the copies async;
 *   pageable memory works but serialises).  Returns after everything has landed in the host buffers.
 */
vs_status vs_render_host(vs_scene* scene, const vs_camera* cameras, uint32_t num_cameras,
                         const vs_render_params* params, float* out_rgba, uint32_t* out_tri_ids,
                         void* cuda_stream);

/* Per-layer render buffers (supplement Fig. "render buffers": a) surface normals, b) surface UVs,
 * c) surface opacity, d) surface colors of every layer).  Every pointer is DEVICE memory or
 * NULL (buffer not wanted); layer index l = 0 is the outermost shell; pixels a layer does not hit hold zeros (ids: MISS).
 * The buffers describe the nearest fragment of EVERY layer, also of layers the compositor never reached because the
 * transmittance fell below t_min. */
typedef struct {
    uint32_t* tri_ids;      /* [num_cameras][k][H][W]     as vs_render's out_tri_ids                                  */
    float*    layer_rgba;   /* [num_cameras][k][H][W][4]  rgb = Sigmoid of the SH dot (NOT premultiplied, NOT composited),
                                                           a = opacity as blended (after VS_FLAG_ATTENUATION's alpha_w)  */
    float*    layer_uv;     /* [num_cameras][k][H][W][2]  perspective-correct UV of the fragment                       */
    float*    layer_normal; /* [num_cameras][k][H][W][3]  unit geometric normal of the fragment's triangle, world space,
                                                           signed to face the viewer (v . n <= 0)                        */
} vs_aov_buffers;

/*
 * vs_render_aov -- vs_render plus the per-layer buffers of `aov` (which may be NULL: then it is vs_render without ids).
 *   The image is produced by the same kernels as vs_render (bit-identical); the buffers are written by a separate plain
 *   kernel (k_layer_aov) from the triangle-id planes, so the hot path carries no cost for them.  Asynchronous on
 *   `cuda_stream`, same rules as vs_render.
 */
vs_status vs_render_aov(vs_scene* scene, const vs_camera* cameras, uint32_t num_cameras,
                        const vs_render_params* params, float* out_rgba, const vs_aov_buffers* aov, void* cuda_stream);

/*
 * vs_render_backward -- backward pass to the texels (§4.5: the texture values are optimised through
 * the lookup the real-time renderer performs).  For the same scene, cameras and
 * params as a vs_render call, and an upstream gradient dL/d(out_rgba), ACCUMULATES dL/d(texture coefficient), summed
 * over the cameras, by the chain rule through the blend (S7), the sigmoids and SH dot (S6) and the bilinear weights (S5);
 * VS_FLAG_ATTENUATION's alpha_w and the t_min early exit are constants of the differentiation (layers behind the exit get
 * no gradient); coverage and UVs do not depend on the textures.
 *   grad_rgba      DEVICE [num_cameras][height][width][4] float
 *   grad_textures  HOST array of num_layers DEVICE pointers, layer l: [tex_h][tex_w][(deg+1)^2][4] float (the API layout
 *                  of vs_layer_desc.texture, always fp32); the caller zeroes them; sums are fp32 atomics in no fixed order
 *   Float-texture scenes only (VS_ERR_UNSUPPORTED on banded scenes and with VS_FLAG_REFERENCE_PATH / TILED / COUNT).
 *   Runs S1-S4 again (nothing of the forward call is kept) and k_shade<BWD> in place of k_shade (forward pass of the tile,
 *   then the recurrence and the scatter; VS_FLAG_PLAIN_BACKWARD: the plain k_backward); asynchronous on `cuda_stream` like
 *   vs_render.
 */
vs_status vs_render_backward(vs_scene* scene, const vs_camera* cameras, uint32_t num_cameras,
                             const vs_render_params* params, const float* grad_rgba, float* const* grad_textures,
                             void* cuda_stream);

/* Waits for the most recent render call on this scene and returns its counters (see vs_render_stats). */
vs_status vs_query_last_render(vs_scene* scene, vs_render_stats* out_stats);

/*
 * vs_render_static -- vs_render for callers that must not allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same steps S1-S7 on the default (direct) path, with EVERYTHING the call writes
 * besides the caller's outputs -- staged cameras, transformed vertices, key image, tile masks, the surface-order list and its
 * sort work space -- placed in one file-scope `static __device__` array of VS_STATIC_SCRATCH_BYTES inside the library
 * (csrc/vs_noalloc.cu).  The call makes no cudaMalloc / cudaFree / pool allocation of any kind; its outputs are bit-identical
 * to vs_render's.
 *
 *   Arguments, layouts and asynchrony as vs_render (cameras HOST, outputs DEVICE, work enqueued on `cuda_stream`).
 *   flags: only VS_FLAG_ATTENUATION and VS_FLAG_SCREEN_ORDER (else VS_ERR_UNSUPPORTED); views_per_chunk is ignored: the call
 *   is ONE pass.  No statistics: vs_query_last_render does not see these calls.
 *   LIMIT: the call needs about  num_cameras * (num_layers * width * height * 8 + total_vertices * 16 + tiles * 16 + 64) +
 *   0.6 MB  bytes of scratch (tiles = ceil(width / 16) * ceil(height / 16)); if that exceeds VS_STATIC_SCRATCH_BYTES the call
 *   fails with VS_ERR_UNSUPPORTED and a message that states both numbers -- render fewer cameras per call, or use vs_render.
 *   (k = 9 layers and 100 000 vertices: one 1024 x 768 view needs 58.8 MB, four 480 x 360 views 56.8 MB, of the 67.1 MB.)
 *   The array exists once per GPU that loads the library (64 MiB of device memory held until the process exits) and is
 *   SHARED by every call, every scene and every stream: what has to start at zero (key image, tile masks, counters) is
 *   cleared by each call on its stream, so stale contents never matter, but two calls whose device work OVERLAPS (different
 *   streams, or several host threads without ordering between their streams) RACE on it.  Order them on one stream or with
 *   events.  Host-side the call is serialised by a library-wide mutex.
 */
#define VS_STATIC_SCRATCH_BYTES (64u << 20)
vs_status vs_render_static(vs_scene* scene, const vs_camera* cameras, uint32_t num_cameras,
                           const vs_render_params* params, float* out_rgba, uint32_t* out_tri_ids,
                           void* cuda_stream);

/* Frees all device memory of the scene after synchronising the device.  NULL is a no-op. */
void vs_scene_destroy(vs_scene* scene);

/* Thread-local description of the last error on this thread ("" if none). */
const char* vs_last_error(void);

/* Library version, e.g. "vs-b200 0.2 (sm_100a)". */
const char* vs_version(void);

#ifdef __cplusplus
}
#endif
#endif /* VS_H_ */

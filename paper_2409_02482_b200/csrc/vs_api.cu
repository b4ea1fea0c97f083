// vs_api.cu -- the C-ABI of include/vs.h: argument validation, scene upload, scratch management and
// the per-chunk launch sequence S1..S7.  No arithmetic of the method lives here.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/vs.h"
#include "vs_common.cuh"

static thread_local char g_err[512] = "";

static vs_status fail(vs_status s, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return s;
}

#define CU(call)                                                                                         \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess)                                                                           \
            return fail(e_ == cudaErrorMemoryAllocation ? VS_ERR_OUT_OF_MEMORY : VS_ERR_CUDA, "%s: %s", #call, \
                        cudaGetErrorString(e_));                                                         \
    } while (0)

struct DevBuf {
    void* p = nullptr;
    size_t cap = 0;
    cudaError_t reserve(size_t bytes)
    {
        if (bytes <= cap) return cudaSuccess;
        if (p) cudaFree(p);
        p = nullptr; cap = 0;
        size_t want = bytes + bytes / 8;
        cudaError_t e = cudaMalloc(&p, want);
        if (e != cudaSuccess) { e = cudaMalloc(&p, bytes); want = bytes; }
        if (e == cudaSuccess) cap = want; else p = nullptr;
        return e;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
};

struct vs_scene {
    int device = 0;
    VsSceneDev dev{};
    int tex_f16 = 0;
    std::vector<void*> owned;
    // scratch, reused between calls
    DevBuf cams, vtx, tri_tiles, tile_count, tile_off, tile_cursor, tile_tris, ids, counters, texel_bits, stage_rgba[2], stage_ids[2];
    DevBuf keys, big_list, big_count;  // direct path
    DevBuf aov_ids;                    // vs_render_aov without a caller-supplied id buffer
    bool keys_dirty = true;            // the key image holds something other than zeros (fresh allocation or an aborted pass)
    // per-call bookkeeping
    uint64_t launches = 0, raster_launches = 0, shade_launches = 0;
    struct Span { cudaEvent_t a, b; int stage; };
    std::vector<Span> spans;        // VS_FLAG_KERNEL_TIMING: event pairs recorded this call
    std::vector<cudaEvent_t> event_pool;
    size_t events_used = 0;
    unsigned long long* host_counters = nullptr;  // pinned [VS_CNT_N]
    cudaStream_t last_stream = nullptr;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_render[2] = {nullptr, nullptr}, ev_copy[2] = {nullptr, nullptr};
    size_t scratch_peak = 0;
    size_t ref_capacity_wanted = 0;  // entries of tile_tris the next chunk asks for
    ~vs_scene()
    {
        for (void* p : owned) cudaFree(p);
        DevBuf* bufs[] = {&cams, &vtx, &tri_tiles, &tile_count, &tile_off, &tile_cursor, &tile_tris, &ids, &counters, &texel_bits,
                          &stage_rgba[0], &stage_rgba[1], &stage_ids[0], &stage_ids[1], &keys, &big_list, &big_count, &aov_ids};
        for (cudaEvent_t e : event_pool) cudaEventDestroy(e);
        for (DevBuf* b : bufs) b->release();
        if (host_counters) cudaFreeHost(host_counters);
        if (copy_stream) cudaStreamDestroy(copy_stream);
        for (int i = 0; i < 2; ++i) {
            if (ev_render[i]) cudaEventDestroy(ev_render[i]);
            if (ev_copy[i]) cudaEventDestroy(ev_copy[i]);
        }
    }
};

extern "C" const char* vs_last_error(void) { return g_err; }
extern "C" const char* vs_version(void) { return "vs-b200 0.1 (sm_100a)"; }

extern "C" void vs_scene_destroy(vs_scene* scene)
{
    if (!scene) return;
    cudaSetDevice(scene->device);
    cudaDeviceSynchronize();
    delete scene;
}

static vs_status dev_alloc(vs_scene* s, void** p, size_t bytes)
{
    CU(cudaMalloc(p, bytes ? bytes : 16));
    s->owned.push_back(*p);
    return VS_OK;
}

// Copy `bytes` from a descriptor array (device or host) to fresh device staging if needed.
static vs_status stage_in(const void* src, size_t bytes, vs_memory mem, cudaStream_t st, std::vector<void*>& temps,
                          const void** out)
{
    if (mem == VS_MEM_DEVICE || bytes == 0) { *out = src; return VS_OK; }
    void* d = nullptr;
    CU(cudaMalloc(&d, bytes));
    temps.push_back(d);
    CU(cudaMemcpyAsync(d, src, bytes, cudaMemcpyHostToDevice, st));
    *out = d;
    return VS_OK;
}

// `bd` != nullptr: banded 8-bit scene; `desc` then carries the geometry only (its texture fields are placeholders)
static vs_status scene_create_impl(const vs_scene_desc* desc, const vs_scene_desc_banded* bd, cudaStream_t st, vs_scene* s,
                                   std::vector<void*>& temps)
{
    const uint32_t k = desc->num_layers;
    const uint32_t n = (desc->sh_degree + 1) * (desc->sh_degree + 1);
    const int f16 = desc->tex_dtype == VS_F16;
    VsSceneDev& d = s->dev;
    d.k = k; d.sh_degree = desc->sh_degree; d.n_coef = n;
    d.texel_vecs = 4 * vs_vecs_per_channel(f16, n);
    d.np_pad = vs_vecs_per_channel(f16, n) * (f16 ? 8u : 4u);
    s->tex_f16 = f16;
    uint64_t vt = 0, tt = 0;
    for (uint32_t l = 0; l < k; ++l) {
        const vs_layer_desc& L = desc->layers[l];
        if (L.num_vertices == 0 && L.num_triangles != 0) return fail(VS_ERR_INVALID_ARG, "layer %u: triangles but no vertices", l);
        if ((L.num_vertices && (!L.positions || !L.uvs)) || (L.num_triangles && !L.indices) || !L.texture)
            return fail(VS_ERR_INVALID_ARG, "layer %u: NULL array", l);
        if (L.tex_w == 0 || L.tex_h == 0) return fail(VS_ERR_INVALID_ARG, "layer %u: empty texture", l);
        if (L.tex_w > 32768 || L.tex_h > 32768 || (uint64_t)L.tex_w * L.tex_h * d.texel_vecs >= (1ull << 32))
            return fail(VS_ERR_UNSUPPORTED, "layer %u: texture %ux%u too large", l, L.tex_w, L.tex_h);
        d.tri_off[l] = (uint32_t)tt;
        d.vtx_off[l] = (uint32_t)vt;
        vt += L.num_vertices; tt += L.num_triangles;
        if (vt >= (1ull << 31) || tt >= (1ull << 31)) return fail(VS_ERR_UNSUPPORTED, "scene too large");
    }
    for (uint32_t l = k; l <= VS_MAX_LAYERS; ++l) { d.tri_off[l] = (uint32_t)tt; d.vtx_off[l] = (uint32_t)vt; }
    uint64_t bits = 0;
    for (uint32_t l = 0; l <= VS_MAX_LAYERS; ++l) {
        d.tex_bit_off[l] = (uint32_t)bits;
        if (l < k) bits += ((uint64_t)desc->layers[l].tex_w * desc->layers[l].tex_h + 31) / 32 * 32;
        if (bits >= (1ull << 32)) return fail(VS_ERR_UNSUPPORTED, "textures too large");
    }
    d.v_total = (uint32_t)vt; d.t_total = (uint32_t)tt;

    float* pos; float2* uvs; uint4* tris; float4* nrm; uint32_t* flag;
    vs_status r;
    if ((r = dev_alloc(s, (void**)&pos, vt * 12)) != VS_OK) return r;
    if ((r = dev_alloc(s, (void**)&uvs, vt * 8)) != VS_OK) return r;
    if ((r = dev_alloc(s, (void**)&tris, tt * 16)) != VS_OK) return r;
    if ((r = dev_alloc(s, (void**)&nrm, tt * 16)) != VS_OK) return r;
    if ((r = dev_alloc(s, (void**)&flag, 16)) != VS_OK) return r;
    CU(cudaMemsetAsync(flag, 0, 16, st));
    uint64_t voff = 0;
    const cudaMemcpyKind kind = desc->memory == VS_MEM_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
    for (uint32_t l = 0; l < k; ++l) {
        const vs_layer_desc& L = desc->layers[l];
        if (L.num_vertices) {
            CU(cudaMemcpyAsync(pos + 3 * voff, L.positions, (size_t)L.num_vertices * 12, kind, st));
            CU(cudaMemcpyAsync(uvs + voff, L.uvs, (size_t)L.num_vertices * 8, kind, st));
        }
        const void* idx = nullptr;
        if ((r = stage_in(L.indices, (size_t)L.num_triangles * 12, desc->memory, st, temps, &idx)) != VS_OK) return r;
        CU(vs_launch_pack_tris((const uint32_t*)idx, pos + 3 * voff, L.num_triangles, L.num_vertices, (uint32_t)voff, l,
                               tris + d.tri_off[l], nrm + d.tri_off[l], flag, st));
        if (bd) {
            // banded 8-bit textures: one padded texel array per band
            const vs_layer_desc_banded& BL = bd->layers[l];
            for (uint32_t b = 0; b <= desc->sh_degree; ++b) {
                const size_t texels = (size_t)BL.band_w[b] * BL.band_h[b];
                unsigned char* bt;
                if ((r = dev_alloc(s, (void**)&bt, texels * VS_BAND_STRIDE(b))) != VS_OK) return r;
                const void* bsrc = nullptr;
                if ((r = stage_in(BL.band_texture[b], texels * (2 * b + 1) * 4, desc->memory, st, temps, &bsrc)) != VS_OK) return r;
                CU(vs_launch_pack_band((const unsigned char*)bsrc, (uint32_t)texels, b, bt, st));
                d.btex[l][b] = bt; d.bw[l][b] = BL.band_w[b]; d.bh[l][b] = BL.band_h[b];
            }
            d.tex[l] = nullptr; d.tex_w[l] = BL.band_w[0]; d.tex_h[l] = BL.band_h[0];
            voff += L.num_vertices;
            continue;
        }
        // texture -> internal layout (same element order, texel padded to a multiple of 16 bytes)
        const size_t texels = (size_t)L.tex_w * L.tex_h;
        const size_t src_bytes = texels * n * 4 * (f16 ? 2 : 4);
        uint4* tex;
        if ((r = dev_alloc(s, (void**)&tex, texels * d.texel_vecs * 16)) != VS_OK) return r;
        {
            const void* tsrc = nullptr;
            if ((r = stage_in(L.texture, src_bytes, desc->memory, st, temps, &tsrc)) != VS_OK) return r;
            CU(vs_launch_pack_texture(tsrc, f16, (uint32_t)texels, n, d.np_pad, tex, st));
        }
        d.tex[l] = tex; d.tex_w[l] = L.tex_w; d.tex_h[l] = L.tex_h;
        voff += L.num_vertices;
    }
    CU(vs_launch_check_finite(pos, (size_t)vt * 3, flag, st));
    CU(vs_launch_check_finite((const float*)uvs, (size_t)vt * 2, flag, st));
    uint32_t hflag = 0;
    CU(cudaMemcpyAsync(&hflag, flag, 4, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    if (hflag & 1u) return fail(VS_ERR_INVALID_ARG, "a triangle index is >= num_vertices of its layer");
    if (hflag & 2u) return fail(VS_ERR_INVALID_ARG, "a vertex position or uv is not finite");
    d.positions = pos; d.uvs = uvs; d.tris = tris; d.tri_nrm = nrm;
    d.banded = bd ? 1u : 0u;
    if (bd) { d.v_min = bd->v_min; d.v_scale = (bd->v_max - bd->v_min) / 255.0f; }
    CU(cudaHostAlloc((void**)&s->host_counters, VS_CNT_N * 8, cudaHostAllocDefault));
    CU(cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
        CU(cudaEventCreateWithFlags(&s->ev_render[i], cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&s->ev_copy[i], cudaEventDisableTiming));
    }
    return VS_OK;
}

extern "C" vs_status vs_scene_create(const vs_scene_desc* desc, void* cuda_stream, vs_scene** out_scene)
{
    g_err[0] = 0;
    if (out_scene) *out_scene = nullptr;
    if (!desc || !out_scene) return fail(VS_ERR_INVALID_ARG, "NULL argument");
    if (desc->num_layers < 1 || desc->num_layers > VS_MAX_LAYERS) return fail(VS_ERR_INVALID_ARG, "num_layers must be 1..9");
    if (desc->sh_degree > 3) return fail(VS_ERR_INVALID_ARG, "sh_degree must be 0..3");
    if (desc->tex_dtype != VS_F32 && desc->tex_dtype != VS_F16) return fail(VS_ERR_INVALID_ARG, "bad tex_dtype");
    if (desc->memory != VS_MEM_DEVICE && desc->memory != VS_MEM_HOST) return fail(VS_ERR_INVALID_ARG, "bad memory kind");
    if (!desc->layers) return fail(VS_ERR_INVALID_ARG, "NULL layers");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(VS_ERR_CUDA, "no CUDA device available (this library has no CPU fallback)");
    }
    vs_scene* s = new (std::nothrow) vs_scene();
    if (!s) return fail(VS_ERR_OUT_OF_MEMORY, "host allocation failed");
    cudaGetDevice(&s->device);
    std::vector<void*> temps;
    vs_status r = scene_create_impl(desc, nullptr, (cudaStream_t)cuda_stream, s, temps);
    cudaStreamSynchronize((cudaStream_t)cuda_stream);
    for (void* p : temps) cudaFree(p);
    if (r != VS_OK) {
        delete s;
        cudaGetLastError();
        return r;
    }
    *out_scene = s;
    return VS_OK;
}

extern "C" vs_status vs_scene_create_banded(const vs_scene_desc_banded* bd, void* cuda_stream, vs_scene** out_scene)
{
    g_err[0] = 0;
    if (out_scene) *out_scene = nullptr;
    if (!bd || !out_scene) return fail(VS_ERR_INVALID_ARG, "NULL argument");
    if (bd->num_layers < 1 || bd->num_layers > VS_MAX_LAYERS) return fail(VS_ERR_INVALID_ARG, "num_layers must be 1..9");
    if (bd->sh_degree > 3) return fail(VS_ERR_INVALID_ARG, "sh_degree must be 0..3");
    if (bd->memory != VS_MEM_DEVICE && bd->memory != VS_MEM_HOST) return fail(VS_ERR_INVALID_ARG, "bad memory kind");
    if (!bd->layers) return fail(VS_ERR_INVALID_ARG, "NULL layers");
    if (!std::isfinite(bd->v_min) || !std::isfinite(bd->v_max)) return fail(VS_ERR_INVALID_ARG, "v_min / v_max not finite");
    // geometry through the common path: a float descriptor whose texture fields are placeholders
    std::vector<vs_layer_desc> geo(bd->num_layers);
    for (uint32_t l = 0; l < bd->num_layers; ++l) {
        const vs_layer_desc_banded& B = bd->layers[l];
        for (uint32_t b = 0; b <= bd->sh_degree; ++b) {
            if (!B.band_texture[b]) return fail(VS_ERR_INVALID_ARG, "layer %u: band %u texture is NULL", l, b);
            if (B.band_w[b] == 0 || B.band_h[b] == 0) return fail(VS_ERR_INVALID_ARG, "layer %u: band %u is empty", l, b);
            if (B.band_w[b] > 8192 || B.band_h[b] > 8192) return fail(VS_ERR_UNSUPPORTED, "layer %u: band %u larger than 8192", l, b);
        }
        geo[l].positions = B.positions; geo[l].uvs = B.uvs; geo[l].num_vertices = B.num_vertices;
        geo[l].indices = B.indices; geo[l].num_triangles = B.num_triangles;
        geo[l].texture = B.band_texture[0]; geo[l].tex_w = 1; geo[l].tex_h = 1;
    }
    vs_scene_desc desc;
    desc.num_layers = bd->num_layers; desc.sh_degree = bd->sh_degree; desc.tex_dtype = VS_F32; desc.memory = bd->memory;
    desc.layers = geo.data();
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(VS_ERR_CUDA, "no CUDA device available (this library has no CPU fallback)");
    }
    vs_scene* s = new (std::nothrow) vs_scene();
    if (!s) return fail(VS_ERR_OUT_OF_MEMORY, "host allocation failed");
    cudaGetDevice(&s->device);
    std::vector<void*> temps;
    vs_status r = scene_create_impl(&desc, bd, (cudaStream_t)cuda_stream, s, temps);
    cudaStreamSynchronize((cudaStream_t)cuda_stream);
    for (void* p : temps) cudaFree(p);
    if (r != VS_OK) {
        delete s;
        cudaGetLastError();
        return r;
    }
    *out_scene = s;
    return VS_OK;
}

static vs_status validate_render(const vs_scene* scene, const vs_camera* cams, uint32_t n, const vs_render_params* p,
                                 const void* out_rgba)
{
    if (!scene || !p || !out_rgba || (n && !cams)) return fail(VS_ERR_INVALID_ARG, "NULL argument");
    if (p->width == 0 || p->height == 0) return fail(VS_ERR_INVALID_ARG, "empty image");
    if (p->width > 16384 || p->height > 16384) return fail(VS_ERR_UNSUPPORTED, "image larger than 16384 px");
    if (!(p->near_plane > 0.0f) || !std::isfinite(p->near_plane)) return fail(VS_ERR_INVALID_ARG, "near_plane must be > 0");
    if (!(p->t_min >= 0.0f) || !std::isfinite(p->t_min)) return fail(VS_ERR_INVALID_ARG, "t_min must be >= 0");
    if (p->flags & ~(uint32_t)(VS_FLAG_REFERENCE_PATH | VS_FLAG_KERNEL_TIMING | VS_FLAG_COUNT_TEXELS | VS_FLAG_TILED_PATH | VS_FLAG_ATTENUATION))
        return fail(VS_ERR_INVALID_ARG, "reserved flag bits set");
    for (int i = 0; i < 3; ++i)
        if (!std::isfinite(p->background[i])) return fail(VS_ERR_INVALID_ARG, "background not finite");
    for (uint32_t c = 0; c < n; ++c) {
        const float* f = &cams[c].fx;
        for (int i = 0; i < 16; ++i)
            if (!std::isfinite(f[i])) return fail(VS_ERR_INVALID_ARG, "camera %u not finite", c);
        if (!(cams[c].fx > 0.0f) || !(cams[c].fy > 0.0f)) return fail(VS_ERR_INVALID_ARG, "camera %u: fx, fy must be > 0", c);
    }
    return VS_OK;
}

// Views per internal pass.  Device outputs: as many as a ~3 GB scratch budget allows (fewer, larger launches:
// C4 26.8 ms per 64 views at 16 against 27.7 ms at 4).  Host outputs: at most 4, so that the download of one
// chunk overlaps the rendering of the next (C4 end to end: 3407 MP/s at 4 against 3025 MP/s at 16).
static uint32_t pick_chunk(const vs_scene* s, const vs_render_params* p, uint32_t n, bool host_outputs)
{
    if (p->views_per_chunk) return p->views_per_chunk < n ? p->views_per_chunk : n;
    // keep the per-chunk scratch (transformed vertices, key image or packed tile ranges + id planes) under ~3 GB
    const bool tiled = (p->flags & VS_FLAG_TILED_PATH) != 0;
    const size_t per_view = (size_t)s->dev.v_total * 16 + (tiled ? (size_t)s->dev.t_total * 8 : 0) +
                            (size_t)p->width * p->height * (tiled ? 4 : 8) * s->dev.k;
    size_t c = ((size_t)3 << 30) / (per_view ? per_view : 1);
    if (c < 1) c = 1;
    if (c > (host_outputs ? 4u : 16u)) c = host_outputs ? 4 : 16;
    return (uint32_t)(c < n ? c : n);
}

static vs_status span_begin(vs_scene* s, bool on, int stage, cudaStream_t st)
{
    if (!on) return VS_OK;
    while (s->event_pool.size() < s->events_used + 2) {
        cudaEvent_t e;
        CU(cudaEventCreate(&e));
        s->event_pool.push_back(e);
    }
    vs_scene::Span sp{s->event_pool[s->events_used], s->event_pool[s->events_used + 1], stage};
    s->events_used += 2;
    CU(cudaEventRecord(sp.a, st));
    s->spans.push_back(sp);
    return VS_OK;
}

static vs_status span_end(vs_scene* s, bool on, cudaStream_t st)
{
    if (!on) return VS_OK;
    CU(cudaEventRecord(s->spans.back().b, st));
    return VS_OK;
}

// Render `views` cameras starting at cams[0] into device outputs.  All work on `st`, no host sync.
static vs_status render_chunk(vs_scene* s, const vs_camera* cams, uint32_t views, const vs_render_params* p,
                              float* out_rgba, uint32_t* out_ids, cudaStream_t st, const float* grad_out = nullptr,
                              const VsGradTex* grad_tex = nullptr)
{
    VsFrame fr;
    fr.width = p->width; fr.height = p->height;
    fr.tiles_x = (p->width + VS_TILE_W - 1) / VS_TILE_W; fr.tiles_y = (p->height + VS_TILE_H - 1) / VS_TILE_H;
    fr.near_plane = p->near_plane; fr.t_min = p->t_min;
    for (int i = 0; i < 3; ++i) fr.bg[i] = p->background[i];
    fr.attenuate = (p->flags & VS_FLAG_ATTENUATION) ? 1u : 0u;
    const size_t ntile = (size_t)views * fr.tiles_x * fr.tiles_y;
    if (ntile >= (1ull << 31)) return fail(VS_ERR_UNSUPPORTED, "too many tiles in one chunk");
    const bool reference = (p->flags & VS_FLAG_REFERENCE_PATH) != 0;
    const bool tiled = (p->flags & VS_FLAG_TILED_PATH) != 0;
    const size_t id_words = (size_t)views * s->dev.k * p->width * p->height;

    CU(s->cams.reserve(sizeof(VsCamDev) * views));
    CU(s->vtx.reserve((size_t)s->dev.v_total * views * 16 + 16));
    if (!reference && !tiled) {
        const size_t had = s->keys.cap;
        CU(s->keys.reserve(id_words * 8 + 16));
        if (s->keys.cap != had) s->keys_dirty = true;
        CU(s->tile_count.reserve(ntile * 4));   // per-tile layer masks
        CU(s->big_list.reserve((size_t)65536 * 8));
        CU(s->big_count.reserve(16));
    }
    if (!reference && tiled) {
        CU(s->tri_tiles.reserve((size_t)s->dev.t_total * views * 4 + 16));
        CU(s->tile_count.reserve(ntile * 4));
        CU(s->tile_off.reserve((ntile + 1) * 4));
        CU(s->tile_cursor.reserve(ntile * 4));
        // the reference list is sized from what earlier calls needed (or a first guess) and CHECKED:
        // k_scan records the chunk's need when it exceeds the capacity and vs_render then retries
        if (s->ref_capacity_wanted < 1024) s->ref_capacity_wanted = 1024;
        CU(s->tile_tris.reserve(s->ref_capacity_wanted * 4));
        if (!out_ids) CU(s->ids.reserve(id_words * 4 + 16));
    }

    VsChunk ch{};
    ch.views = views;
    ch.cams = (const VsCamDev*)s->cams.p;
    ch.vtx = (int4*)s->vtx.p;
    ch.tri_tiles = (uint32_t*)s->tri_tiles.p;
    ch.tile_count = (uint32_t*)s->tile_count.p;
    ch.tile_off = (uint32_t*)s->tile_off.p;
    ch.tile_cursor = (uint32_t*)s->tile_cursor.p;
    ch.tile_tris = (uint32_t*)s->tile_tris.p;
    const size_t cap = s->tile_tris.cap / 4;
    ch.ref_capacity = cap > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)cap;
    ch.counters = (unsigned long long*)s->counters.p;
    ch.out_rgba = out_rgba;
    ch.ids = out_ids ? out_ids : (uint32_t*)s->ids.p;
    ch.ids_is_output = out_ids != nullptr;

    static_assert(sizeof(VsCamDev) == sizeof(vs_camera), "camera layout");
    const bool timing = (p->flags & VS_FLAG_KERNEL_TIMING) != 0;
    vs_status r;
    CU(cudaMemcpyAsync(s->cams.p, cams, sizeof(VsCamDev) * views, cudaMemcpyHostToDevice, st));
    if ((r = span_begin(s, timing, 0, st)) != VS_OK) return r;
    CU(vs_launch_transform(s->dev, fr, ch, st));
    if ((r = span_end(s, timing, st)) != VS_OK) return r;
    s->launches += 1;
    if (reference) {
        CU(vs_launch_reference(s->dev, s->tex_f16, fr, ch, st));
        s->launches += 1;
        return VS_OK;
    }
    if (tiled) {
        CU(cudaMemsetAsync(ch.tile_count, 0, ntile * 4, st));
        CU(cudaMemsetAsync(ch.tile_cursor, 0, ntile * 4, st));
    }
    if ((p->flags & VS_FLAG_COUNT_TEXELS) && s->dev.banded) {
        ch.count_fragments = 1;   // banded scenes: shaded fragments only (no unique-texel bitmap)
    } else if (p->flags & VS_FLAG_COUNT_TEXELS) {
        const size_t words = (size_t)views * (s->dev.tex_bit_off[s->dev.k] >> 5);
        CU(s->texel_bits.reserve(words * 4 + 16));
        CU(cudaMemsetAsync(s->texel_bits.p, 0, words * 4, st));
        ch.texel_bits = (uint32_t*)s->texel_bits.p;
    }
    if (!tiled) {
        // direct path: triangle-parallel raster into the key image, which k_shade reads and clears
        ch.keys = (unsigned long long*)s->keys.p;
        ch.big_list = (uint2*)s->big_list.p;
        ch.big_count = (uint32_t*)s->big_count.p;
        ch.big_capacity = 65536;
        if (s->keys_dirty) CU(cudaMemsetAsync(s->keys.p, 0, s->keys.cap, st));
        s->keys_dirty = true;
        CU(cudaMemsetAsync(ch.big_count, 0, 4, st));
        ch.tile_mask = ch.tile_count;
        CU(cudaMemsetAsync(ch.tile_mask, 0, ntile * 4, st));
        if ((r = span_begin(s, timing, 2, st)) != VS_OK) return r;
        CU(vs_launch_raster_direct(s->dev, fr, ch, st));
        if ((r = span_end(s, timing, st)) != VS_OK) return r;
        if ((r = span_begin(s, timing, 3, st)) != VS_OK) return r;
        if (grad_out) {   // vs_render_backward: k_backward consumes the key image in place of k_shade
            ch.grad_out = grad_out; ch.grad_tex = *grad_tex;
            CU(vs_launch_backward(s->dev, s->tex_f16, fr, ch, st));
        } else {
            CU(s->dev.banded ? vs_launch_shade_banded(s->dev, fr, ch, st) : vs_launch_shade(s->dev, s->tex_f16, fr, ch, st));
        }
        if ((r = span_end(s, timing, st)) != VS_OK) return r;
        s->keys_dirty = false;
        s->launches += (s->dev.t_total ? 2 : 0) + 1;
        s->raster_launches += 1;
        s->shade_launches += 1;
        if (ch.texel_bits) {
            CU(vs_launch_popcount(ch.texel_bits, (size_t)views * (s->dev.tex_bit_off[s->dev.k] >> 5),
                                  ch.counters + VS_CNT_TEXELS, st));
            s->launches += 1;
        }
        const size_t scratch = s->cams.cap + s->vtx.cap + s->keys.cap + s->big_list.cap + s->big_count.cap + s->tile_count.cap;
        if (scratch > s->scratch_peak) s->scratch_peak = scratch;
        return VS_OK;
    }
    if ((r = span_begin(s, timing, 1, st)) != VS_OK) return r;
    CU(vs_launch_bin_count(s->dev, fr, ch, st));
    CU(vs_launch_bin_scan(fr, ch, st));
    CU(vs_launch_bin_scatter(s->dev, fr, ch, st));
    if ((r = span_end(s, timing, st)) != VS_OK) return r;
    if ((r = span_begin(s, timing, 2, st)) != VS_OK) return r;
    CU(vs_launch_raster(s->dev, fr, ch, st));
    if ((r = span_end(s, timing, st)) != VS_OK) return r;
    if ((r = span_begin(s, timing, 3, st)) != VS_OK) return r;
    CU(s->dev.banded ? vs_launch_shade_banded(s->dev, fr, ch, st) : vs_launch_shade(s->dev, s->tex_f16, fr, ch, st));
    if ((r = span_end(s, timing, st)) != VS_OK) return r;
    s->launches += (s->dev.t_total ? 3 : 1) + 2;
    s->raster_launches += 1;
    s->shade_launches += 1;
    if (ch.texel_bits) {
        CU(vs_launch_popcount(ch.texel_bits, (size_t)views * (s->dev.tex_bit_off[s->dev.k] >> 5),
                              ch.counters + VS_CNT_TEXELS, st));
        s->launches += 1;
    }
    const size_t scratch = s->cams.cap + s->vtx.cap + s->tri_tiles.cap + s->tile_count.cap + s->tile_off.cap +
                           s->tile_cursor.cap + s->tile_tris.cap + s->ids.cap;
    if (scratch > s->scratch_peak) s->scratch_peak = scratch;
    return VS_OK;
}

static vs_status begin_render(vs_scene* s, cudaStream_t st)
{
    CU(cudaSetDevice(s->device));
    CU(s->counters.reserve(VS_CNT_N * 8));
    CU(cudaMemsetAsync(s->counters.p, 0, VS_CNT_N * 8, st));
    s->last_stream = st;
    s->scratch_peak = 0;
    s->launches = s->raster_launches = s->shade_launches = 0;
    s->spans.clear();
    s->events_used = 0;
    return VS_OK;
}

// Waits for the call's kernels and reads the counters back.  *retry is set when a chunk needed more
// triangle references than the list could hold (the images are then incomplete): the capacity is
// raised to what was needed and the caller renders again.
static vs_status finish_render(vs_scene* s, cudaStream_t st, bool* retry)
{
    CU(cudaMemcpyAsync(s->host_counters, s->counters.p, VS_CNT_N * 8, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    const unsigned long long need = s->host_counters[VS_CNT_OVERFLOW];
    *retry = need != 0;
    if (need) s->ref_capacity_wanted = (size_t)(need + need / 4 + 1024);
    return VS_OK;
}

static void first_capacity_guess(vs_scene* s, uint32_t chunk)
{
    if (s->ref_capacity_wanted == 0) s->ref_capacity_wanted = (size_t)2 * s->dev.t_total * chunk + 65536;
}

extern "C" vs_status vs_render(vs_scene* scene, const vs_camera* cameras, uint32_t num_cameras,
                               const vs_render_params* params, float* out_rgba, uint32_t* out_tri_ids,
                               void* cuda_stream)
{
    g_err[0] = 0;
    vs_status r = validate_render(scene, cameras, num_cameras, params, out_rgba);
    if (r != VS_OK) return r;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t chunk = pick_chunk(scene, params, num_cameras, false);
    const size_t px = (size_t)params->width * params->height;
    first_capacity_guess(scene, chunk);
    for (int attempt = 0; attempt < 4; ++attempt) {
        if ((r = begin_render(scene, st)) != VS_OK) return r;
        if (num_cameras == 0) return VS_OK;
        for (uint32_t v0 = 0; v0 < num_cameras; v0 += chunk) {
            const uint32_t nv = num_cameras - v0 < chunk ? num_cameras - v0 : chunk;
            r = render_chunk(scene, cameras + v0, nv, params, out_rgba + (size_t)v0 * px * 4,
                             out_tri_ids ? out_tri_ids + (size_t)v0 * scene->dev.k * px : nullptr, st);
            if (r != VS_OK) return r;
        }
        bool retry = false;
        if ((r = finish_render(scene, st, &retry)) != VS_OK) return r;
        if (!retry) return VS_OK;
    }
    return fail(VS_ERR_CUDA, "triangle reference list kept overflowing");
}

extern "C" vs_status vs_render_backward(vs_scene* scene, const vs_camera* cameras, uint32_t num_cameras,
                                        const vs_render_params* params, const float* grad_rgba,
                                        float* const* grad_textures, void* cuda_stream)
{
    g_err[0] = 0;
    vs_status r = validate_render(scene, cameras, num_cameras, params, grad_rgba);
    if (r != VS_OK) return r;
    if (!grad_textures) return fail(VS_ERR_INVALID_ARG, "NULL argument");
    if (scene->dev.banded) return fail(VS_ERR_UNSUPPORTED, "vs_render_backward: float textures only (banded scenes are baked, not fitted)");
    if (params->flags & (VS_FLAG_REFERENCE_PATH | VS_FLAG_TILED_PATH | VS_FLAG_COUNT_TEXELS))
        return fail(VS_ERR_UNSUPPORTED, "vs_render_backward runs on the default (direct) raster path only");
    VsGradTex gt{};
    for (uint32_t l = 0; l < scene->dev.k; ++l) {
        if (!grad_textures[l]) return fail(VS_ERR_INVALID_ARG, "grad_textures[%u] is NULL", l);
        if ((uint64_t)scene->dev.tex_w[l] * scene->dev.tex_h[l] * scene->dev.n_coef >= (1ull << 32))
            return fail(VS_ERR_UNSUPPORTED, "layer %u: gradient texture too large", l);
        gt.p[l] = grad_textures[l];
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t chunk = pick_chunk(scene, params, num_cameras, false);
    const size_t px = (size_t)params->width * params->height;
    if ((r = begin_render(scene, st)) != VS_OK) return r;
    for (uint32_t v0 = 0; v0 < num_cameras; v0 += chunk) {
        const uint32_t nv = num_cameras - v0 < chunk ? num_cameras - v0 : chunk;
        r = render_chunk(scene, cameras + v0, nv, params, nullptr, nullptr, st, grad_rgba + (size_t)v0 * px * 4, &gt);
        if (r != VS_OK) return r;
    }
    bool retry = false;
    return finish_render(scene, st, &retry);
}

extern "C" vs_status vs_render_aov(vs_scene* scene, const vs_camera* cameras, uint32_t num_cameras,
                                   const vs_render_params* params, float* out_rgba, const vs_aov_buffers* aov,
                                   void* cuda_stream)
{
    if (!aov || (!aov->layer_rgba && !aov->layer_uv && !aov->layer_normal))
        return vs_render(scene, cameras, num_cameras, params, out_rgba, aov ? aov->tri_ids : nullptr, cuda_stream);
    g_err[0] = 0;
    vs_status r = validate_render(scene, cameras, num_cameras, params, out_rgba);
    if (r != VS_OK) return r;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t chunk = pick_chunk(scene, params, num_cameras, false);
    const size_t px = (size_t)params->width * params->height, kpx = px * scene->dev.k;
    VsFrame fr;
    fr.width = params->width; fr.height = params->height;
    fr.tiles_x = (params->width + VS_TILE_W - 1) / VS_TILE_W; fr.tiles_y = (params->height + VS_TILE_H - 1) / VS_TILE_H;
    fr.near_plane = params->near_plane; fr.t_min = params->t_min;
    for (int i = 0; i < 3; ++i) fr.bg[i] = params->background[i];
    fr.attenuate = (params->flags & VS_FLAG_ATTENUATION) ? 1u : 0u;
    first_capacity_guess(scene, chunk);
    for (int attempt = 0; attempt < 4; ++attempt) {
        if ((r = begin_render(scene, st)) != VS_OK) return r;
        if (num_cameras == 0) return VS_OK;
        for (uint32_t v0 = 0; v0 < num_cameras; v0 += chunk) {
            const uint32_t nv = num_cameras - v0 < chunk ? num_cameras - v0 : chunk;
            uint32_t* ids = aov->tri_ids ? aov->tri_ids + (size_t)v0 * kpx : nullptr;
            if (!ids) {
                CU(scene->aov_ids.reserve(kpx * 4 * chunk + 16));
                ids = (uint32_t*)scene->aov_ids.p;
            }
            r = render_chunk(scene, cameras + v0, nv, params, out_rgba + (size_t)v0 * px * 4, ids, st);
            if (r != VS_OK) return r;
            // the chunk's cameras and transformed vertices are still in the scene's scratch
            CU(vs_launch_layer_aov(scene->dev, scene->tex_f16, fr, nv, (const VsCamDev*)scene->cams.p, (const int4*)scene->vtx.p, ids,
                                   aov->layer_rgba ? aov->layer_rgba + (size_t)v0 * kpx * 4 : nullptr,
                                   aov->layer_uv ? aov->layer_uv + (size_t)v0 * kpx * 2 : nullptr,
                                   aov->layer_normal ? aov->layer_normal + (size_t)v0 * kpx * 3 : nullptr, st));
            scene->launches += 1;
        }
        bool retry = false;
        if ((r = finish_render(scene, st, &retry)) != VS_OK) return r;
        if (!retry) return VS_OK;
    }
    return fail(VS_ERR_CUDA, "triangle reference list kept overflowing");
}

extern "C" vs_status vs_render_host(vs_scene* scene, const vs_camera* cameras, uint32_t num_cameras,
                                    const vs_render_params* params, float* out_rgba, uint32_t* out_tri_ids,
                                    void* cuda_stream)
{
    g_err[0] = 0;
    vs_status r = validate_render(scene, cameras, num_cameras, params, out_rgba);
    if (r != VS_OK) return r;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t chunk = pick_chunk(scene, params, num_cameras, true);
    const size_t px = (size_t)params->width * params->height;
    const size_t rgba_bytes = px * 16, ids_bytes = px * 4 * scene->dev.k;
    first_capacity_guess(scene, chunk);
    for (int attempt = 0; attempt < 4; ++attempt) {
        if ((r = begin_render(scene, st)) != VS_OK) return r;
        if (num_cameras == 0) return VS_OK;
        uint32_t b = 0;
        bool used[2] = {false, false};
        for (uint32_t v0 = 0; v0 < num_cameras; v0 += chunk, b ^= 1u) {
            const uint32_t nv = num_cameras - v0 < chunk ? num_cameras - v0 : chunk;
            CU(scene->stage_rgba[b].reserve(rgba_bytes * chunk));
            if (out_tri_ids) CU(scene->stage_ids[b].reserve(ids_bytes * chunk));
            if (used[b]) CU(cudaStreamWaitEvent(st, scene->ev_copy[b], 0));  // staging buffer b is free again
            r = render_chunk(scene, cameras + v0, nv, params, (float*)scene->stage_rgba[b].p,
                             out_tri_ids ? (uint32_t*)scene->stage_ids[b].p : nullptr, st);
            if (r != VS_OK) return r;
            CU(cudaEventRecord(scene->ev_render[b], st));
            CU(cudaStreamWaitEvent(scene->copy_stream, scene->ev_render[b], 0));
            CU(cudaMemcpyAsync(out_rgba + (size_t)v0 * px * 4, scene->stage_rgba[b].p, rgba_bytes * nv, cudaMemcpyDeviceToHost,
                               scene->copy_stream));
            if (out_tri_ids)
                CU(cudaMemcpyAsync(out_tri_ids + (size_t)v0 * scene->dev.k * px, scene->stage_ids[b].p, ids_bytes * nv,
                                   cudaMemcpyDeviceToHost, scene->copy_stream));
            CU(cudaEventRecord(scene->ev_copy[b], scene->copy_stream));
            used[b] = true;
        }
        bool retry = false;
        if ((r = finish_render(scene, st, &retry)) != VS_OK) return r;
        CU(cudaStreamSynchronize(scene->copy_stream));
        if (!retry) return VS_OK;
    }
    return fail(VS_ERR_CUDA, "triangle reference list kept overflowing");
}

extern "C" vs_status vs_query_last_render(vs_scene* scene, vs_render_stats* out)
{
    g_err[0] = 0;
    if (!scene || !out) return fail(VS_ERR_INVALID_ARG, "NULL argument");
    memset(out, 0, sizeof(*out));
    if (!scene->counters.p) return VS_OK;
    CU(cudaSetDevice(scene->device));
    CU(cudaStreamSynchronize(scene->last_stream));
    const unsigned long long* h = scene->host_counters;  // read back by finish_render
    out->dropped_triangles = h[VS_CNT_DROPPED];
    out->degenerate_triangles = h[VS_CNT_DEGENERATE];
    out->tile_refs = h[VS_CNT_REFS];
    out->scratch_bytes = scene->scratch_peak;
    out->kernel_launches = scene->launches;
    out->raster_launches = scene->raster_launches;
    out->shade_launches = scene->shade_launches;
    out->shaded_fragments = h[VS_CNT_FRAGS];
    out->unique_texels = h[VS_CNT_TEXELS];
    for (const vs_scene::Span& sp : scene->spans) {
        float ms = 0.0f;
        CU(cudaEventElapsedTime(&ms, sp.a, sp.b));
        (sp.stage == 0 ? out->ms_transform : sp.stage == 1 ? out->ms_binning : sp.stage == 2 ? out->ms_raster : out->ms_shade) += ms;
    }
    return VS_OK;
}

// vs_api.cu -- the C-ABI of include/vs.h: argument validation, scene upload, scratch management and
// the per-chunk launch sequence S1..S7.  No arithmetic of the method lives here.
//
// Execution model of a render call:
//   * the scene is immutable; everything a call writes besides the caller's outputs lives in one of VS_NUM_SETS scratch
//     sets (transformed vertices, key image, tile masks, ...).  A set is handed from user to user through CUDA events
//     (ev_done), never through the host, so calls are asynchronous and calls on different streams are legal: they
//     interleave at chunk granularity;
//   * scratch grows with stream-ordered allocations from a pool private to the scene (no device-wide synchronisation);
//   * under VS_FLAG_OVERLAP the chunks of a call are software-pipelined over the two sets: S1-S4 of chunk c+1 run on an
//     internal high-priority stream in a few resident CTAs per SM BESIDE the S5-S7 kernel of chunk c on the caller's
//     stream (an experiment that lost, kept behind the flag: DESIGN.md §7);
//   * counters and kernel timings are read back lazily by vs_query_last_render.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/vs.h"
#include "vs_common.cuh"
#include "vs_internal.cuh"

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
        if (e_ != cudaSuccess) {                                                                         \
            cudaGetLastError(); /* do not leave the error behind for the caller's next CUDA call */      \
            return fail(e_ == cudaErrorMemoryAllocation ? VS_ERR_OUT_OF_MEMORY : VS_ERR_CUDA, "%s: %s", #call, \
                        cudaGetErrorString(e_));                                                         \
        }                                                                                                \
    } while (0)

// Makes `device` current for the duration of an API call and restores the caller's device on every exit path.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(int device)
    {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != device) switched = cudaSetDevice(device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

// Device buffer that only grows.  Growth is stream-ordered (cudaFreeAsync + cudaMallocFromPoolAsync on the stream that
// uses the buffer next): no cudaFree / cudaMalloc, hence no implicit device synchronisation inside a render call.
// Every buffer sits between two guard bands of VS_GUARD_BYTES filled with 0xA5 at allocation; vs_query_last_render checks
// them (compute-sanitizer is not available on the target pool: an out-of-bounds WRITE of a kernel into scratch is caught here).
#define VS_GUARD_BYTES 4096
struct DevBuf {
    void* p = nullptr;     // first usable byte
    size_t cap = 0;        // usable bytes
    cudaError_t reserve(size_t bytes, cudaMemPool_t pool, cudaStream_t st, bool* grew = nullptr)
    {
        if (bytes <= cap) return cudaSuccess;
        if (p) cudaFreeAsync((char*)p - VS_GUARD_BYTES, st);
        p = nullptr; cap = 0;
        size_t want = (bytes + bytes / 8 + 255) & ~(size_t)255;
        void* base = nullptr;
        cudaError_t e = cudaMallocFromPoolAsync(&base, want + 2 * VS_GUARD_BYTES, pool, st);
        if (e != cudaSuccess) {
            cudaGetLastError();   // clear the failed attempt: the exact-size retry below may succeed
            want = (bytes + 255) & ~(size_t)255;
            e = cudaMallocFromPoolAsync(&base, want + 2 * VS_GUARD_BYTES, pool, st);
        }
        if (e != cudaSuccess) { cudaGetLastError(); return e; }
        p = (char*)base + VS_GUARD_BYTES; cap = want;
        if (grew) *grew = true;
        e = cudaMemsetAsync(base, 0xA5, VS_GUARD_BYTES, st);
        if (e == cudaSuccess) e = cudaMemsetAsync((char*)p + cap, 0xA5, VS_GUARD_BYTES, st);
        return e;
    }
    // after a device synchronisation only: true if both guard bands still hold their pattern
    bool guards_intact() const
    {
        if (!p) return true;
        unsigned char h[2][VS_GUARD_BYTES];
        if (cudaMemcpy(h[0], (char*)p - VS_GUARD_BYTES, VS_GUARD_BYTES, cudaMemcpyDeviceToHost) != cudaSuccess) return false;
        if (cudaMemcpy(h[1], (char*)p + cap, VS_GUARD_BYTES, cudaMemcpyDeviceToHost) != cudaSuccess) return false;
        for (int g = 0; g < 2; ++g)
            for (int i = 0; i < VS_GUARD_BYTES; ++i)
                if (h[g][i] != 0xA5) return false;
        return true;
    }
    void release() { if (p) cudaFree((char*)p - VS_GUARD_BYTES); p = nullptr; cap = 0; }   // after a device synchronisation only
};

#define VS_NUM_SETS 2      // scratch sets; a call ping-pongs between them
#ifndef VS_RESIDENT_RASTER_CTAS_PER_SM
#define VS_RESIDENT_RASTER_CTAS_PER_SM 1
#endif
#define VS_NUM_TICKETS 8   // calls whose counters may be in flight at once

// Everything one chunk of views writes besides the caller's outputs.
struct ScratchSet {
    DevBuf vtx, keys, tile_count, big_list, big_count;                 // direct path (tile_count doubles as the tile masks)
    DevBuf order, order_work;                                          // direct path: surface order of the (view, tile) pairs
    DevBuf tri_tiles, tile_off, tile_cursor, tile_tris, ids;           // per-tile path
    DevBuf texel_bits;                                                 // VS_FLAG_COUNT_TEXELS
    DevBuf aov_ids;                                                    // vs_render_aov without a caller-supplied id buffer
    bool keys_dirty = true;      // the key image holds something other than zeros (fresh allocation or an aborted pass)
    cudaEvent_t ev_raster = nullptr;   // S1-S4 of the chunk in this set have been enqueued up to here
    cudaEvent_t ev_done = nullptr;     // the last consumer of the set (shade / backward / aov kernel) ends here
    bool used = false;                 // ev_done has been recorded at least once
    const DevBuf* named(int i, const char** name) const
    {
        static const char* names[] = {"vtx", "keys", "tile_count", "big_list", "big_count", "tri_tiles", "tile_off", "tile_cursor",
                                      "tile_tris", "ids", "texel_bits", "aov_ids", "order", "order_work"};
        const DevBuf* bufs[] = {&vtx, &keys, &tile_count, &big_list, &big_count, &tri_tiles, &tile_off, &tile_cursor, &tile_tris, &ids,
                                &texel_bits, &aov_ids, &order, &order_work};
        if (i < 0 || i >= 14) return nullptr;
        *name = names[i];
        return bufs[i];
    }
    size_t bytes() const
    {
        return vtx.cap + keys.cap + tile_count.cap + big_list.cap + big_count.cap + tri_tiles.cap + tile_off.cap + tile_cursor.cap +
               tile_tris.cap + ids.cap + texel_bits.cap + aov_ids.cap + order.cap + order_work.cap;
    }
};

// Per-call record: device counters, their pinned host copy, the call's cameras.
struct Ticket {
    unsigned long long* dev_counters = nullptr;    // [VS_CNT_N]
    unsigned long long* host_counters = nullptr;   // pinned [VS_CNT_N]
    VsCamDev* host_cams = nullptr;                 // pinned staging of the call's cameras
    size_t host_cams_cap = 0;
    DevBuf cams;                                   // DEVICE [num_cameras]
    cudaEvent_t ev_end = nullptr;                  // counters have landed in host_counters
    bool in_flight = false;
};

struct vs_scene {
    int device = 0;
    VsSceneDev dev{};
    int tex_f16 = 0;
    std::vector<void*> owned;
    std::mutex mu;                     // host-side: one API call at a time per scene (the device work still overlaps)
    cudaMemPool_t pool = nullptr;      // private stream-ordered pool of all scratch
    ScratchSet sets[VS_NUM_SETS];
    uint64_t chunk_seq = 0;            // chunks rendered so far: chunk n uses sets[n % VS_NUM_SETS]
    Ticket tickets[VS_NUM_TICKETS];
    uint64_t ticket_seq = 0;
    int last_ticket = -1;
    cudaStream_t aux_stream = nullptr;   // high priority: S1-S4 of the next chunk beside the current chunk's shading
    cudaStream_t copy_stream = nullptr;  // vs_render_host downloads
    DevBuf stage_rgba[2], stage_ids[2];
    cudaEvent_t ev_render[2] = {nullptr, nullptr}, ev_copy[2] = {nullptr, nullptr};
    bool stage_used[2] = {false, false};
    // bookkeeping since the last vs_query_last_render
    uint64_t launches = 0, raster_launches = 0, shade_launches = 0;
    struct Span { cudaEvent_t a, b; int stage; };
    std::vector<Span> spans;        // VS_FLAG_KERNEL_TIMING: event pairs recorded since the last query
    std::vector<cudaEvent_t> event_pool;
    size_t events_used = 0;
    bool span_open = false;
    uint32_t resident_ctas = 148;    // CTAs of a raster kernel that shares the GPU with a consumer kernel (one per SM)
    size_t scratch_peak = 0;
    size_t scratch_budget = 0;       // bytes one pass may keep in scratch (set at the first call from the free device memory)
    size_t ref_capacity_wanted = 0;  // entries of tile_tris the next chunk asks for
    ~vs_scene()
    {
        for (void* p : owned) cudaFree(p);
        for (ScratchSet& ss : sets) {
            DevBuf* bufs[] = {&ss.vtx, &ss.keys, &ss.tile_count, &ss.big_list, &ss.big_count, &ss.tri_tiles, &ss.tile_off, &ss.tile_cursor,
                              &ss.tile_tris, &ss.ids, &ss.texel_bits, &ss.aov_ids, &ss.order, &ss.order_work};
            for (DevBuf* b : bufs) b->release();
            if (ss.ev_raster) cudaEventDestroy(ss.ev_raster);
            if (ss.ev_done) cudaEventDestroy(ss.ev_done);
        }
        for (Ticket& t : tickets) {
            if (t.dev_counters) cudaFree(t.dev_counters);
            if (t.host_counters) cudaFreeHost(t.host_counters);
            if (t.host_cams) cudaFreeHost(t.host_cams);
            t.cams.release();
            if (t.ev_end) cudaEventDestroy(t.ev_end);
        }
        for (int i = 0; i < 2; ++i) {
            stage_rgba[i].release(); stage_ids[i].release();
            if (ev_render[i]) cudaEventDestroy(ev_render[i]);
            if (ev_copy[i]) cudaEventDestroy(ev_copy[i]);
        }
        for (cudaEvent_t e : event_pool) cudaEventDestroy(e);
        if (aux_stream) cudaStreamDestroy(aux_stream);
        if (copy_stream) cudaStreamDestroy(copy_stream);
        if (pool) cudaMemPoolDestroy(pool);
    }
};

// streams, events, the scratch pool and the per-call tickets of a freshly created scene
static vs_status init_runtime(vs_scene* s)
{
    cudaMemPoolProps props{};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = s->device;
    CU(cudaMemPoolCreate(&s->pool, &props));
    unsigned long long keep = ~0ull;   // never hand scratch back to the driver between calls
    CU(cudaMemPoolSetAttribute(s->pool, cudaMemPoolAttrReleaseThreshold, &keep));
    int sms = 0;
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, s->device));
    s->resident_ctas = (uint32_t)(sms > 0 ? sms : 148) * VS_RESIDENT_RASTER_CTAS_PER_SM;
    int lo = 0, hi = 0;
    CU(cudaDeviceGetStreamPriorityRange(&lo, &hi));
    CU(cudaStreamCreateWithPriority(&s->aux_stream, cudaStreamNonBlocking, hi));
    CU(cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking));
    for (ScratchSet& ss : s->sets) {
        CU(cudaEventCreateWithFlags(&ss.ev_raster, cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&ss.ev_done, cudaEventDisableTiming));
    }
    for (Ticket& t : s->tickets) {
        CU(cudaMalloc((void**)&t.dev_counters, VS_CNT_N * 8));
        CU(cudaHostAlloc((void**)&t.host_counters, VS_CNT_N * 8, cudaHostAllocDefault));
        memset(t.host_counters, 0, VS_CNT_N * 8);
        CU(cudaEventCreateWithFlags(&t.ev_end, cudaEventDisableTiming));
    }
    for (int i = 0; i < 2; ++i) {
        CU(cudaEventCreateWithFlags(&s->ev_render[i], cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&s->ev_copy[i], cudaEventDisableTiming));
    }
    return VS_OK;
}

extern "C" const char* vs_last_error(void) { return g_err; }
extern "C" const char* vs_version(void) { return "vs-b200 0.2 (sm_100a)"; }

extern "C" void vs_scene_destroy(vs_scene* scene)
{
    if (!scene) return;
    DeviceGuard guard(scene->device);
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
    d.frag_layout = (f16 && d.np_pad == 16u && !bd) ? 1u : 0u;   // k_shade's tensor-core path
#ifdef VS_SHADE_NO_MMA
    d.frag_layout = 0u;   // experiment switch: channel-major texels and the packed-FFMA k_shade for every format
#endif
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
        if (L.num_triangles >= (1u << 28)) return fail(VS_ERR_UNSUPPORTED, "layer %u: more than 2^28 - 1 triangles", l);
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
        // + 256: k_shade prefetches whole 256-byte aligned blocks around a footprint row
        if ((r = dev_alloc(s, (void**)&tex, texels * d.texel_vecs * 16 + 256)) != VS_OK) return r;
        {
            const void* tsrc = nullptr;
            if ((r = stage_in(L.texture, src_bytes, desc->memory, st, temps, &tsrc)) != VS_OK) return r;
            CU(vs_launch_pack_texture(tsrc, f16, (uint32_t)texels, n, d.np_pad, d.frag_layout, tex, st));
        }
        d.tex[l] = tex; d.tex_w[l] = L.tex_w; d.tex_h[l] = L.tex_h;
        voff += L.num_vertices;
    }
    CU(vs_launch_check_finite(pos, (size_t)vt * 3, flag, st));
    CU(vs_launch_check_finite((const float*)uvs, (size_t)vt * 2, flag, st));
    int* bb;
    if ((r = dev_alloc(s, (void**)&bb, 32)) != VS_OK) return r;
    CU(vs_launch_bbox(pos, (uint32_t)vt, bb, st));
    uint32_t hflag = 0;
    int hbb[6];
    CU(cudaMemcpyAsync(&hflag, flag, 4, cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(hbb, bb, sizeof(hbb), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    for (int a = 0; a < 3; ++a) {   // (order-preserving ints back to floats; an empty scene gets a unit box)
        const int lo = hbb[a] ^ ((hbb[a] >> 31) & 0x7FFFFFFF), hi = hbb[3 + a] ^ ((hbb[3 + a] >> 31) & 0x7FFFFFFF);
        float fmin, fmax;
        memcpy(&fmin, &lo, 4); memcpy(&fmax, &hi, 4);
        if (!vt || !(fmax > fmin)) { fmin = vt ? fmin : 0.0f; fmax = fmin + 1.0f; }
        d.bb_min[a] = fmin; d.bb_scale[a] = 32.0f / (fmax - fmin);
    }
    if (hflag & 1u) return fail(VS_ERR_INVALID_ARG, "a triangle index is >= num_vertices of its layer");
    if (hflag & 2u) return fail(VS_ERR_INVALID_ARG, "a vertex position or uv is not finite");
    d.positions = pos; d.uvs = uvs; d.tris = tris; d.tri_nrm = nrm;
    d.banded = bd ? 1u : 0u;
    if (bd) { d.v_min = bd->v_min; d.v_scale = (bd->v_max - bd->v_min) / 255.0f; }
    return init_runtime(s);
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


extern "C" vs_status vs_scene_set_vertex_normals(vs_scene* scene, const float* const* normals, vs_memory memory, void* cuda_stream)
{
    g_err[0] = 0;
    if (!scene || !normals) return fail(VS_ERR_INVALID_ARG, "NULL argument");
    if (memory != VS_MEM_DEVICE && memory != VS_MEM_HOST) return fail(VS_ERR_INVALID_ARG, "bad memory kind");
    std::lock_guard<std::mutex> lock(scene->mu);
    DeviceGuard guard(scene->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(cudaDeviceSynchronize());   // renders in flight read the scene: it changes only while nothing runs
    VsSceneDev& d = scene->dev;
    float4* vn = const_cast<float4*>(d.vtx_nrm);
    if (!vn) {
        vs_status r = dev_alloc(scene, (void**)&vn, (size_t)d.v_total * 16);
        if (r != VS_OK) return r;
        CU(cudaMemsetAsync(vn, 0, (size_t)d.v_total * 16, st));
    }
    uint32_t* flag = nullptr;
    CU(cudaMalloc((void**)&flag, 16));
    CU(cudaMemsetAsync(flag, 0, 16, st));
    std::vector<void*> temps;
    uint32_t mask = 0;
    vs_status r = VS_OK;
    for (uint32_t l = 0; l < d.k && r == VS_OK; ++l) {
        if (!normals[l]) continue;
        const uint32_t nv = d.vtx_off[l + 1] - d.vtx_off[l];
        const void* src = nullptr;
        if ((r = stage_in(normals[l], (size_t)nv * 12, memory, st, temps, &src)) != VS_OK) break;
        cudaError_t e = vs_launch_check_finite((const float*)src, (size_t)nv * 3, flag, st);
        if (e == cudaSuccess) e = vs_launch_pack_normals((const float*)src, nv, vn + d.vtx_off[l], st);
        if (e != cudaSuccess) { r = fail(VS_ERR_CUDA, "vs_scene_set_vertex_normals: %s", cudaGetErrorString(e)); break; }
        mask |= 1u << l;
    }
    uint32_t hflag = 0;
    if (r == VS_OK && cudaMemcpyAsync(&hflag, flag, 4, cudaMemcpyDeviceToHost, st) != cudaSuccess) r = fail(VS_ERR_CUDA, "copy failed");
    cudaStreamSynchronize(st);
    for (void* p : temps) cudaFree(p);
    cudaFree(flag);
    cudaGetLastError();
    if (r != VS_OK) return r;
    if (hflag & 2u) return fail(VS_ERR_INVALID_ARG, "a vertex normal is not finite");
    d.vtx_nrm = vn;
    d.vnrm_mask = mask;
    return VS_OK;
}

static vs_status validate_render(const vs_scene* scene, const vs_camera* cams, uint32_t n, const vs_render_params* p,
                                 const void* out_rgba)
{
    if (!scene || !p || (n && (!cams || !out_rgba))) return fail(VS_ERR_INVALID_ARG, "NULL argument");   // zero cameras: a legal no-op
    if (p->width == 0 || p->height == 0) return fail(VS_ERR_INVALID_ARG, "empty image");
    if (p->width > 16384 || p->height > 16384) return fail(VS_ERR_UNSUPPORTED, "image larger than 16384 px");
    if (!(p->near_plane > 0.0f) || !std::isfinite(p->near_plane)) return fail(VS_ERR_INVALID_ARG, "near_plane must be > 0");
    if (!(p->t_min >= 0.0f) || !std::isfinite(p->t_min)) return fail(VS_ERR_INVALID_ARG, "t_min must be >= 0");
    if (p->flags & ~(uint32_t)(VS_FLAG_REFERENCE_PATH | VS_FLAG_KERNEL_TIMING | VS_FLAG_COUNT_TEXELS | VS_FLAG_TILED_PATH |
                               VS_FLAG_ATTENUATION | VS_FLAG_OVERLAP | VS_FLAG_SCREEN_ORDER | VS_FLAG_PLAIN_BACKWARD))
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

// Views per internal pass (chunk).  A pass keeps the transformed vertices and the key image (or packed tile ranges + id
// planes) of its views in one of the scene's two scratch sets.  Larger passes let more views share texels through L2 in
// surface order and launch fewer kernels (C4, 64 views: 23.5 ms in passes of 16, 23.0 of 32, 22.9 of 64), so device outputs
// take up to VS_CHUNK_DEVICE views as long as a set stays under a twelfth of the device memory that is free at the
// scene's first call (and under 12 GB); the views are then spread evenly over the passes.  Host outputs: at most 4 views, so
// that the download of one chunk overlaps the rendering of the next.
#ifndef VS_CHUNK_DEVICE
#define VS_CHUNK_DEVICE 64u
#endif
static uint32_t pick_chunk(vs_scene* s, const vs_render_params* p, uint32_t n, bool host_outputs)
{
    if (p->views_per_chunk) return p->views_per_chunk < n ? p->views_per_chunk : n;
    if (n == 0) return 0;
    if (s->scratch_budget == 0) {
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess) { cudaGetLastError(); free_b = (size_t)48 << 30; }
        s->scratch_budget = free_b / 12;   // per scratch set (there are two)
        if (s->scratch_budget > ((size_t)12 << 30)) s->scratch_budget = (size_t)12 << 30;
        if (s->scratch_budget < ((size_t)1 << 30)) s->scratch_budget = (size_t)1 << 30;
    }
    const bool tiled = (p->flags & VS_FLAG_TILED_PATH) != 0;
    const size_t per_view = (size_t)s->dev.v_total * 16 + (tiled ? (size_t)s->dev.t_total * 8 : 0) +
                            (size_t)p->width * p->height * (tiled ? 4 : 8) * s->dev.k;
    size_t c = s->scratch_budget / (per_view ? per_view : 1);
    if (c < 1) c = 1;
    const size_t cap = host_outputs ? 4u : VS_CHUNK_DEVICE;
    if (c > cap) c = cap;
    if (c >= n) return n;
    const size_t passes = (n + c - 1) / c;
    return (uint32_t)((n + passes - 1) / passes);
}

static vs_status span_begin(vs_scene* s, bool on, int stage, cudaStream_t st)
{
    s->span_open = false;
    if (!on || s->spans.size() >= 16384) return VS_OK;   // (a caller that never queries does not grow the list for ever)
    while (s->event_pool.size() < s->events_used + 2) {
        cudaEvent_t e;
        CU(cudaEventCreate(&e));
        s->event_pool.push_back(e);
    }
    vs_scene::Span sp{s->event_pool[s->events_used], s->event_pool[s->events_used + 1], stage};
    s->events_used += 2;
    CU(cudaEventRecord(sp.a, st));
    s->spans.push_back(sp);
    s->span_open = true;
    return VS_OK;
}

static vs_status span_end(vs_scene* s, bool on, cudaStream_t st)
{
    if (!on || !s->span_open) return VS_OK;
    CU(cudaEventRecord(s->spans.back().b, st));
    s->span_open = false;
    return VS_OK;
}

enum CallMode { MODE_FORWARD = 0, MODE_BACKWARD = 1, MODE_AOV = 2 };

// State of one API call while its chunks are being enqueued.
struct Call {
    vs_scene* s;
    Ticket* tk;
    const vs_render_params* p;
    VsFrame fr;
    cudaStream_t st;      // the caller's stream: consumers (S5-S7) and everything the caller may wait for
    cudaStream_t rs;      // the stream of S1-S4: the scene's aux stream when the call is pipelined, else `st`
    bool timing, reference, tiled;
    bool ordered;         // direct path: the consumer takes its (view, tile) pairs in surface order (vs_kernels_order.cu)
    CallMode mode;
    const float* grad_rgba;         // MODE_BACKWARD: [num_cameras][H][W][4]
    VsGradTex grad_tex;
    const vs_aov_buffers* aov;      // MODE_AOV
    uint32_t first_view;            // of the chunk being enqueued
};

static vs_status begin_call(vs_scene* s, Call& c, const vs_camera* cams, uint32_t n, const vs_render_params* p, cudaStream_t st,
                            CallMode mode)
{
    c.s = s; c.p = p; c.st = st; c.mode = mode;
    c.grad_rgba = nullptr; c.aov = nullptr; c.first_view = 0;
    c.fr.width = p->width; c.fr.height = p->height;
    c.fr.tiles_x = (p->width + VS_TILE_W - 1) / VS_TILE_W; c.fr.tiles_y = (p->height + VS_TILE_H - 1) / VS_TILE_H;
    c.fr.near_plane = p->near_plane; c.fr.t_min = p->t_min;
    for (int i = 0; i < 3; ++i) c.fr.bg[i] = p->background[i];
    c.fr.attenuate = (p->flags & VS_FLAG_ATTENUATION) ? 1u : 0u;
    c.timing = (p->flags & VS_FLAG_KERNEL_TIMING) != 0;
    c.reference = (p->flags & VS_FLAG_REFERENCE_PATH) != 0;
    c.tiled = (p->flags & VS_FLAG_TILED_PATH) != 0;
    // banded scenes keep screen order: their textures are 8x smaller and k_shade_banded leaves the HBM idle
    c.ordered = !c.reference && !c.tiled && !(p->flags & VS_FLAG_SCREEN_ORDER) && !s->dev.banded;
    // VS_FLAG_OVERLAP (direct path only): S1-S4 go to the internal stream so that they run beside the previous chunk's or
    // the previous call's shading.  Measured slower than back to back on B200 (both kernels are bound by the
    // warps the register file holds), hence opt-in
    const bool pipelined = !c.reference && !c.tiled && (p->flags & VS_FLAG_OVERLAP);
    c.rs = pipelined ? s->aux_stream : st;

    Ticket& tk = s->tickets[s->ticket_seq % VS_NUM_TICKETS];
    s->ticket_seq++;
    c.tk = &tk;
    if (tk.in_flight) CU(cudaEventSynchronize(tk.ev_end));   // a ticket comes round again after VS_NUM_TICKETS calls
    tk.in_flight = false;
    if (tk.host_cams_cap < n) {
        if (tk.host_cams) cudaFreeHost(tk.host_cams);
        tk.host_cams = nullptr; tk.host_cams_cap = 0;
        const size_t want = n + n / 2 + 16;
        CU(cudaHostAlloc((void**)&tk.host_cams, want * sizeof(VsCamDev), cudaHostAllocDefault));
        tk.host_cams_cap = want;
    }
    static_assert(sizeof(VsCamDev) == sizeof(vs_camera), "camera layout");
    memcpy(tk.host_cams, cams, (size_t)n * sizeof(VsCamDev));   // the caller's array may change as soon as the call returns
    CU(tk.cams.reserve((size_t)(n ? n : 1) * sizeof(VsCamDev), s->pool, c.rs));
    CU(cudaMemcpyAsync(tk.cams.p, tk.host_cams, (size_t)n * sizeof(VsCamDev), cudaMemcpyHostToDevice, c.rs));
    CU(cudaMemsetAsync(tk.dev_counters, 0, VS_CNT_N * 8, c.rs));
    return VS_OK;
}

// Counters -> pinned host memory, stream-ordered; nothing waits for them until vs_query_last_render.
static vs_status end_call(Call& c)
{
    vs_scene* s = c.s;
    if (c.rs != c.st) {   // a call without chunks: keep the counter copy behind the memset of begin_call
        CU(cudaEventRecord(c.tk->ev_end, c.rs));
        CU(cudaStreamWaitEvent(c.st, c.tk->ev_end, 0));
    }
    CU(cudaMemcpyAsync(c.tk->host_counters, c.tk->dev_counters, VS_CNT_N * 8, cudaMemcpyDeviceToHost, c.st));
    CU(cudaEventRecord(c.tk->ev_end, c.st));
    c.tk->in_flight = true;
    s->last_ticket = (int)(c.tk - s->tickets);
    size_t scratch = 0;
    for (const ScratchSet& ss : s->sets) scratch += ss.bytes();
    for (const Ticket& t : s->tickets) scratch += t.cams.cap;
    for (int i = 0; i < 2; ++i) scratch += s->stage_rgba[i].cap + s->stage_ids[i].cap;
    if (scratch > s->scratch_peak) s->scratch_peak = scratch;
    return VS_OK;
}

static VsChunk make_chunk(const Call& c, ScratchSet& ss, uint32_t views, float* out_rgba, uint32_t* out_ids)
{
    VsChunk ch{};
    ch.views = views;
    ch.cams = (const VsCamDev*)c.tk->cams.p + c.first_view;
    ch.vtx = (int4*)ss.vtx.p;
    ch.tri_tiles = (uint32_t*)ss.tri_tiles.p;
    ch.tile_count = (uint32_t*)ss.tile_count.p;
    ch.tile_off = (uint32_t*)ss.tile_off.p;
    ch.tile_cursor = (uint32_t*)ss.tile_cursor.p;
    ch.tile_tris = (uint32_t*)ss.tile_tris.p;
    const size_t cap = ss.tile_tris.cap / 4;
    ch.ref_capacity = cap > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)cap;
    ch.counters = c.tk->dev_counters;
    ch.out_rgba = out_rgba;
    ch.ids = out_ids ? out_ids : (uint32_t*)ss.ids.p;
    ch.ids_is_output = out_ids != nullptr;
    if (!c.reference && !c.tiled) {
        ch.keys = (unsigned long long*)ss.keys.p;
        ch.big_list = (uint2*)ss.big_list.p;
        ch.big_count = (uint32_t*)ss.big_count.p;
        ch.big_capacity = 65536;
        ch.tile_mask = ch.tile_count;
        if (c.ordered) ch.order = (const uint32_t*)ss.order.p;
    }
    if ((c.p->flags & VS_FLAG_COUNT_TEXELS) && c.s->dev.banded) ch.count_fragments = 1;   // banded scenes: fragments only
    else if (c.p->flags & VS_FLAG_COUNT_TEXELS) ch.texel_bits = (uint32_t*)ss.texel_bits.p;
    if (c.mode == MODE_BACKWARD) {
        ch.grad_out = c.grad_rgba + (size_t)c.first_view * c.fr.width * c.fr.height * 4;
        ch.grad_tex = c.grad_tex;
    }
    return ch;
}

// S1-S4 of `views` cameras starting at c.first_view into scratch set `ss`, on c.rs.  `resident`: the raster kernel runs in a
// few resident CTAs per SM because another kernel (the previous chunk's consumer) occupies the GPU at the same time.
static vs_status enqueue_geometry(Call& c, ScratchSet& ss, uint32_t views, uint32_t* out_ids, bool resident)
{
    vs_scene* s = c.s;
    const VsFrame& fr = c.fr;
    const size_t ntile = (size_t)views * fr.tiles_x * fr.tiles_y;
    if (ntile >= (1ull << 31)) return fail(VS_ERR_UNSUPPORTED, "too many tiles in one chunk");
    const size_t id_words = (size_t)views * s->dev.k * fr.width * fr.height;
    if (ss.used) CU(cudaStreamWaitEvent(c.rs, ss.ev_done, 0));   // the set's previous consumer has finished
    CU(ss.vtx.reserve((size_t)s->dev.v_total * views * 16 + 16, s->pool, c.rs));
    if (!c.reference && !c.tiled) {
        bool grew = false;
        CU(ss.keys.reserve(id_words * 8 + 16, s->pool, c.rs, &grew));
        if (grew) ss.keys_dirty = true;
        CU(ss.tile_count.reserve(ntile * 4, s->pool, c.rs));   // per-tile layer masks
        CU(ss.big_list.reserve((size_t)65536 * 8, s->pool, c.rs));
        CU(ss.big_count.reserve(16, s->pool, c.rs));
        if (c.ordered) {
            CU(ss.order.reserve(ntile * 4 + 16, s->pool, c.rs));
            CU(ss.order_work.reserve((2 * ntile + VS_ORDER_BINS) * 4 + 16, s->pool, c.rs));
        }
    }
    if (!c.reference && c.tiled) {
        CU(ss.tri_tiles.reserve((size_t)s->dev.t_total * views * 4 + 16, s->pool, c.rs));
        CU(ss.tile_count.reserve(ntile * 4, s->pool, c.rs));
        CU(ss.tile_off.reserve((ntile + 1) * 4, s->pool, c.rs));
        CU(ss.tile_cursor.reserve(ntile * 4, s->pool, c.rs));
        // the reference list is sized from what earlier calls needed (or a first guess) and CHECKED:
        // k_scan records the chunk's need when it exceeds the capacity and vs_render then retries
        if (s->ref_capacity_wanted < 1024) s->ref_capacity_wanted = 1024;
        CU(ss.tile_tris.reserve(s->ref_capacity_wanted * 4, s->pool, c.rs));
        if (!out_ids) CU(ss.ids.reserve(id_words * 4 + 16, s->pool, c.rs));
    }
    if ((c.p->flags & VS_FLAG_COUNT_TEXELS) && !s->dev.banded) {
        const size_t words = (size_t)views * (s->dev.tex_bit_off[s->dev.k] >> 5);
        CU(ss.texel_bits.reserve(words * 4 + 16, s->pool, c.rs));
        CU(cudaMemsetAsync(ss.texel_bits.p, 0, words * 4, c.rs));
    }
    const VsChunk ch = make_chunk(c, ss, views, nullptr, out_ids);

    vs_status r;
    if ((r = span_begin(s, c.timing, 0, c.rs)) != VS_OK) return r;
    CU(vs_launch_transform(s->dev, fr, ch, c.rs));
    if ((r = span_end(s, c.timing, c.rs)) != VS_OK) return r;
    s->launches += 1;
    if (c.reference) {
        CU(cudaEventRecord(ss.ev_raster, c.rs));
        return VS_OK;
    }
    if (!c.tiled) {
        // direct path: triangle-parallel raster into the key image, which the consumer reads and clears
        if (ss.keys_dirty) CU(cudaMemsetAsync(ss.keys.p, 0, ss.keys.cap, c.rs));
        ss.keys_dirty = true;   // until the consumer has been enqueued
        CU(cudaMemsetAsync(ch.big_count, 0, 4, c.rs));
#ifdef VS_EXP_NOMASK
        CU(cudaMemsetAsync(ch.tile_mask, 0xFF, ntile * 4, c.rs));
#else
        CU(cudaMemsetAsync(ch.tile_mask, 0, ntile * 4, c.rs));
#endif
        if ((r = span_begin(s, c.timing, 2, c.rs)) != VS_OK) return r;
        CU(vs_launch_raster_direct(s->dev, fr, ch, c.rs, resident ? s->resident_ctas : 0u));
        if (c.ordered) {   // counted with the raster stage: it is part of what S4 hands to the consumer
            CU(vs_launch_order(s->dev, fr, ch, (uint32_t*)ss.order.p, (uint32_t*)ss.order_work.p, c.rs));
            s->launches += 3;
        }
        if ((r = span_end(s, c.timing, c.rs)) != VS_OK) return r;
        s->launches += s->dev.t_total ? 2 : 0;
        s->raster_launches += 1;
    } else {
        CU(cudaMemsetAsync(ch.tile_count, 0, ntile * 4, c.rs));
        CU(cudaMemsetAsync(ch.tile_cursor, 0, ntile * 4, c.rs));
        if ((r = span_begin(s, c.timing, 1, c.rs)) != VS_OK) return r;
        CU(vs_launch_bin_count(s->dev, fr, ch, c.rs));
        CU(vs_launch_bin_scan(fr, ch, c.rs));
        CU(vs_launch_bin_scatter(s->dev, fr, ch, c.rs));
        if ((r = span_end(s, c.timing, c.rs)) != VS_OK) return r;
        if ((r = span_begin(s, c.timing, 2, c.rs)) != VS_OK) return r;
        CU(vs_launch_raster(s->dev, fr, ch, c.rs));
        if ((r = span_end(s, c.timing, c.rs)) != VS_OK) return r;
        s->launches += (s->dev.t_total ? 3 : 1) + 1;
        s->raster_launches += 1;
    }
    CU(cudaEventRecord(ss.ev_raster, c.rs));
    return VS_OK;
}

// S5-S7 (or the backward / AOV variant) of the chunk whose geometry is in `ss`, on the caller's stream.
static vs_status enqueue_consumer(Call& c, ScratchSet& ss, uint32_t views, float* out_rgba, uint32_t* out_ids)
{
    vs_scene* s = c.s;
    const VsFrame& fr = c.fr;
    if (c.rs != c.st) CU(cudaStreamWaitEvent(c.st, ss.ev_raster, 0));
    const size_t kpx = (size_t)fr.width * fr.height * s->dev.k;
    uint32_t* ids = out_ids;
    if (c.mode == MODE_AOV && !ids) {   // k_layer_aov reads the id planes: keep them in scratch
        CU(ss.aov_ids.reserve(kpx * 4 * views + 16, s->pool, c.st));
        ids = (uint32_t*)ss.aov_ids.p;
    }
    const VsChunk ch = make_chunk(c, ss, views, out_rgba, ids);
    vs_status r;
    if (c.reference) {
        CU(vs_launch_reference(s->dev, s->tex_f16, fr, ch, c.st));
        s->launches += 1;
    } else {
        if ((r = span_begin(s, c.timing, 3, c.st)) != VS_OK) return r;
        if (c.mode == MODE_BACKWARD)
            CU((c.p->flags & VS_FLAG_PLAIN_BACKWARD) ? vs_launch_backward(s->dev, s->tex_f16, fr, ch, c.st)
                                                     : vs_launch_shade_backward(s->dev, s->tex_f16, fr, ch, c.st));
        else CU(s->dev.banded ? vs_launch_shade_banded(s->dev, fr, ch, c.st) : vs_launch_shade(s->dev, s->tex_f16, fr, ch, c.st));
        if ((r = span_end(s, c.timing, c.st)) != VS_OK) return r;
        if (!c.tiled) ss.keys_dirty = false;   // the consumer clears what it reads
        s->launches += 1;
        s->shade_launches += 1;
        if (ch.texel_bits) {
            CU(vs_launch_popcount(ch.texel_bits, (size_t)views * (s->dev.tex_bit_off[s->dev.k] >> 5), ch.counters + VS_CNT_TEXELS, c.st));
            s->launches += 1;
        }
    }
    if (c.mode == MODE_AOV) {
        const vs_aov_buffers* a = c.aov;
        const size_t v0 = c.first_view;
        CU(vs_launch_layer_aov(s->dev, s->tex_f16, fr, views, ch.cams, ch.vtx, ids,
                               a->layer_rgba ? a->layer_rgba + v0 * kpx * 4 : nullptr, a->layer_uv ? a->layer_uv + v0 * kpx * 2 : nullptr,
                               a->layer_normal ? a->layer_normal + v0 * kpx * 3 : nullptr, c.st));
        s->launches += 1;
    }
    CU(cudaEventRecord(ss.ev_done, c.st));
    ss.used = true;
    return VS_OK;
}

// Is a consumer of an earlier chunk or call still running (or queued) on the GPU?  Then the next raster kernel is launched
// in its resident form so that the two share the SMs instead of queueing behind each other.
static bool gpu_busy_with_consumer(const vs_scene* s)
{
    bool busy = false;
    for (const ScratchSet& ss : s->sets)
        if (ss.used && cudaEventQuery(ss.ev_done) == cudaErrorNotReady) busy = true;
    cudaGetLastError();   // cudaErrorNotReady is an answer, not an error
    return busy;
}

// The chunk loop of every render entry point.  out(v0, nv, &rgba, &ids) names the device outputs of a chunk (and may enqueue
// waits on c.st); done(v0, nv) runs after the chunk's consumer has been enqueued (downloads).  On the direct path the
// geometry of chunk i+1 is enqueued BEFORE the consumer of chunk i: the two run side by side on the GPU.
template <typename OutFn, typename DoneFn>
static vs_status run_chunks(Call& c, uint32_t num_cameras, uint32_t chunk, OutFn out, DoneFn done)
{
    vs_scene* s = c.s;
    const bool pipelined = c.rs != c.st;
    vs_status r;
    auto geometry = [&](uint32_t v0, bool resident) -> vs_status {
        const uint32_t nv = num_cameras - v0 < chunk ? num_cameras - v0 : chunk;
        float* rgba = nullptr; uint32_t* ids = nullptr;
        c.first_view = v0;
        if (c.tiled) { vs_status q = out(v0, nv, &rgba, &ids, false); if (q != VS_OK) return q; }   // k_raster writes the ids itself
        return enqueue_geometry(c, s->sets[(s->chunk_seq + v0 / chunk) % VS_NUM_SETS], nv, ids, resident);
    };
    if (num_cameras == 0) return VS_OK;
    if ((r = geometry(0, pipelined && gpu_busy_with_consumer(s))) != VS_OK) return r;
    for (uint32_t v0 = 0; v0 < num_cameras; v0 += chunk) {
        const uint32_t nv = num_cameras - v0 < chunk ? num_cameras - v0 : chunk;
        if (pipelined && v0 + chunk < num_cameras && (r = geometry(v0 + chunk, true)) != VS_OK) return r;
        float* rgba = nullptr; uint32_t* ids = nullptr;
        if ((r = out(v0, nv, &rgba, &ids, true)) != VS_OK) return r;
        c.first_view = v0;
        if ((r = enqueue_consumer(c, s->sets[(s->chunk_seq + v0 / chunk) % VS_NUM_SETS], nv, rgba, ids)) != VS_OK) return r;
        if ((r = done(v0, nv)) != VS_OK) return r;
        if (!pipelined && v0 + chunk < num_cameras && (r = geometry(v0 + chunk, false)) != VS_OK) return r;
    }
    s->chunk_seq += (num_cameras + chunk - 1) / chunk;
    return VS_OK;
}

static void first_capacity_guess(vs_scene* s, uint32_t chunk)
{
    if (s->ref_capacity_wanted == 0) s->ref_capacity_wanted = (size_t)2 * s->dev.t_total * chunk + 65536;
}

// Per-tile path only: the triangle-reference list is sized from earlier calls and checked on the device; this waits for the
// call and reports whether a chunk needed more (the images are then incomplete and the caller renders again).
static vs_status tiled_overflow_check(Call& c, bool* retry)
{
    *retry = false;
    if (!c.tiled) return VS_OK;
    CU(cudaEventSynchronize(c.tk->ev_end));
    const unsigned long long need = c.tk->host_counters[VS_CNT_OVERFLOW];
    *retry = need != 0;
    if (need) c.s->ref_capacity_wanted = (size_t)(need + need / 4 + 1024);
    return VS_OK;
}

extern "C" vs_status vs_render(vs_scene* scene, const vs_camera* cameras, uint32_t num_cameras,
                               const vs_render_params* params, float* out_rgba, uint32_t* out_tri_ids,
                               void* cuda_stream)
{
    g_err[0] = 0;
    vs_status r = validate_render(scene, cameras, num_cameras, params, out_rgba);
    if (r != VS_OK) return r;
    std::lock_guard<std::mutex> lock(scene->mu);
    DeviceGuard guard(scene->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t chunk = pick_chunk(scene, params, num_cameras, false);
    const size_t px = (size_t)params->width * params->height;
    first_capacity_guess(scene, chunk);
    for (int attempt = 0; attempt < 4; ++attempt) {
        Call c;
        if ((r = begin_call(scene, c, cameras, num_cameras, params, st, MODE_FORWARD)) != VS_OK) return r;
        r = run_chunks(c, num_cameras, chunk,
                       [&](uint32_t v0, uint32_t, float** rgba, uint32_t** ids, bool) {
                           *rgba = out_rgba + (size_t)v0 * px * 4;
                           *ids = out_tri_ids ? out_tri_ids + (size_t)v0 * scene->dev.k * px : nullptr;
                           return VS_OK;
                       },
                       [](uint32_t, uint32_t) { return VS_OK; });
        if (r != VS_OK) return r;
        if ((r = end_call(c)) != VS_OK) return r;
        bool retry = false;
        if ((r = tiled_overflow_check(c, &retry)) != VS_OK) return r;
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
    std::lock_guard<std::mutex> lock(scene->mu);
    DeviceGuard guard(scene->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t chunk = pick_chunk(scene, params, num_cameras, false);
    Call c;
    if ((r = begin_call(scene, c, cameras, num_cameras, params, st, MODE_BACKWARD)) != VS_OK) return r;
    c.grad_rgba = grad_rgba; c.grad_tex = gt;
    r = run_chunks(c, num_cameras, chunk,
                   [](uint32_t, uint32_t, float** rgba, uint32_t** ids, bool) { *rgba = nullptr; *ids = nullptr; return VS_OK; },
                   [](uint32_t, uint32_t) { return VS_OK; });
    if (r != VS_OK) return r;
    return end_call(c);
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
    std::lock_guard<std::mutex> lock(scene->mu);
    DeviceGuard guard(scene->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t chunk = pick_chunk(scene, params, num_cameras, false);
    const size_t px = (size_t)params->width * params->height, kpx = px * scene->dev.k;
    first_capacity_guess(scene, chunk);
    for (int attempt = 0; attempt < 4; ++attempt) {
        Call c;
        if ((r = begin_call(scene, c, cameras, num_cameras, params, st, MODE_AOV)) != VS_OK) return r;
        c.aov = aov;
        r = run_chunks(c, num_cameras, chunk,
                       [&](uint32_t v0, uint32_t nv, float** rgba, uint32_t** ids, bool consumer) -> vs_status {
                           *rgba = out_rgba + (size_t)v0 * px * 4;
                           *ids = aov->tri_ids ? aov->tri_ids + (size_t)v0 * kpx : nullptr;
                           if (!*ids && c.tiled) {   // per-tile path: k_raster needs the id planes before the consumer runs
                               ScratchSet& ss = scene->sets[(scene->chunk_seq + v0 / chunk) % VS_NUM_SETS];
                               if (!consumer && ss.used) CU(cudaStreamWaitEvent(c.st, ss.ev_done, 0));
                               CU(ss.aov_ids.reserve(kpx * 4 * nv + 16, scene->pool, c.st));
                               *ids = (uint32_t*)ss.aov_ids.p;
                           }
                           return VS_OK;
                       },
                       [](uint32_t, uint32_t) { return VS_OK; });
        if (r != VS_OK) return r;
        if ((r = end_call(c)) != VS_OK) return r;
        bool retry = false;
        if ((r = tiled_overflow_check(c, &retry)) != VS_OK) return r;
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
    std::lock_guard<std::mutex> lock(scene->mu);
    DeviceGuard guard(scene->device);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const uint32_t chunk = pick_chunk(scene, params, num_cameras, true);
    const size_t px = (size_t)params->width * params->height;
    const size_t rgba_bytes = px * 16, ids_bytes = px * 4 * scene->dev.k;
    first_capacity_guess(scene, chunk);
    for (int attempt = 0; attempt < 4; ++attempt) {
        Call c;
        if ((r = begin_call(scene, c, cameras, num_cameras, params, st, MODE_FORWARD)) != VS_OK) return r;
        // device staging buffer b = (chunk index) & 1; its previous download must have finished before it is rendered into
        r = run_chunks(c, num_cameras, chunk,
                       [&](uint32_t v0, uint32_t, float** rgba, uint32_t** ids, bool consumer) -> vs_status {
                           const uint32_t b = (v0 / chunk) & 1u;
                           if (consumer || c.tiled) {
                               if (scene->stage_used[b]) CU(cudaStreamWaitEvent(st, scene->ev_copy[b], 0));
                               CU(scene->stage_rgba[b].reserve(rgba_bytes * chunk, scene->pool, st));
                               if (out_tri_ids) CU(scene->stage_ids[b].reserve(ids_bytes * chunk, scene->pool, st));
                           }
                           *rgba = (float*)scene->stage_rgba[b].p;
                           *ids = out_tri_ids ? (uint32_t*)scene->stage_ids[b].p : nullptr;
                           return VS_OK;
                       },
                       [&](uint32_t v0, uint32_t nv) -> vs_status {
                           const uint32_t b = (v0 / chunk) & 1u;
                           CU(cudaEventRecord(scene->ev_render[b], st));
                           CU(cudaStreamWaitEvent(scene->copy_stream, scene->ev_render[b], 0));
                           CU(cudaMemcpyAsync(out_rgba + (size_t)v0 * px * 4, scene->stage_rgba[b].p, rgba_bytes * nv, cudaMemcpyDeviceToHost,
                                              scene->copy_stream));
                           if (out_tri_ids)
                               CU(cudaMemcpyAsync(out_tri_ids + (size_t)v0 * scene->dev.k * px, scene->stage_ids[b].p, ids_bytes * nv,
                                                  cudaMemcpyDeviceToHost, scene->copy_stream));
                           CU(cudaEventRecord(scene->ev_copy[b], scene->copy_stream));
                           scene->stage_used[b] = true;
                           return VS_OK;
                       });
        if (r != VS_OK) return r;
        if ((r = end_call(c)) != VS_OK) return r;
        bool retry = false;
        if ((r = tiled_overflow_check(c, &retry)) != VS_OK) return r;
        CU(cudaStreamSynchronize(scene->copy_stream));   // host outputs: the call returns with everything landed
        if (!retry) return VS_OK;
    }
    return fail(VS_ERR_CUDA, "triangle reference list kept overflowing");
}

extern "C" vs_status vs_query_last_render(vs_scene* scene, vs_render_stats* out)
{
    g_err[0] = 0;
    if (!scene || !out) return fail(VS_ERR_INVALID_ARG, "NULL argument");
    memset(out, 0, sizeof(*out));
    std::lock_guard<std::mutex> lock(scene->mu);
    if (scene->last_ticket < 0) return VS_OK;
    DeviceGuard guard(scene->device);
    const Ticket& tk = scene->tickets[scene->last_ticket];
    CU(cudaEventSynchronize(tk.ev_end));   // the only host wait of the render API (besides vs_render_host's downloads)
    const unsigned long long* h = tk.host_counters;
    out->dropped_triangles = h[VS_CNT_DROPPED];
    out->degenerate_triangles = h[VS_CNT_DEGENERATE];
    out->tile_refs = h[VS_CNT_REFS];
    out->shaded_fragments = h[VS_CNT_FRAGS];
    out->unique_texels = h[VS_CNT_TEXELS];
    out->scratch_bytes = scene->scratch_peak;
    // guard bands of every scratch buffer (written by no kernel unless it runs out of bounds); the streams of OTHER calls may
    // still be running, so wait for the device first -- this is the statistics call, not the hot path
    CU(cudaDeviceSynchronize());
    for (int si = 0; si < VS_NUM_SETS; ++si)
        for (int bi = 0;; ++bi) {
            const char* name = "";
            const DevBuf* db = scene->sets[si].named(bi, &name);
            if (!db) break;
            if (!db->guards_intact()) return fail(VS_ERR_CUDA, "scratch guard band of %s (set %d) was overwritten: a kernel wrote out of bounds", name, si);
        }
    for (int ti = 0; ti < VS_NUM_TICKETS; ++ti)
        if (!scene->tickets[ti].cams.guards_intact()) return fail(VS_ERR_CUDA, "scratch guard band of the camera buffer was overwritten");
    for (int i = 0; i < 2; ++i)
        if (!scene->stage_rgba[i].guards_intact() || !scene->stage_ids[i].guards_intact())
            return fail(VS_ERR_CUDA, "scratch guard band of a staging buffer was overwritten");
    out->kernel_launches = scene->launches;
    out->raster_launches = scene->raster_launches;
    out->shade_launches = scene->shade_launches;
    for (const vs_scene::Span& sp : scene->spans) {
        float ms = 0.0f;
        if (cudaEventElapsedTime(&ms, sp.a, sp.b) != cudaSuccess) { cudaGetLastError(); continue; }   // a span of a call still in flight
        (sp.stage == 0 ? out->ms_transform : sp.stage == 1 ? out->ms_binning : sp.stage == 2 ? out->ms_raster : out->ms_shade) += ms;
    }
    scene->spans.clear();
    scene->events_used = 0;
    scene->launches = scene->raster_launches = scene->shade_launches = 0;
    return VS_OK;
}

// ---- hooks for vs_noalloc.cu (vs_render_static); declared in vs_internal.cuh ----
vs_status vs_internal_validate_render(const vs_scene* scene, const vs_camera* cams, uint32_t n, const vs_render_params* p,
                                      const void* out_rgba)
{
    g_err[0] = 0;
    return validate_render(scene, cams, n, p, out_rgba);
}

void vs_internal_scene_view(const vs_scene* scene, const VsSceneDev** dev, int* tex_f16, int* device)
{
    *dev = &scene->dev; *tex_f16 = scene->tex_f16; *device = scene->device;
}

vs_status vs_internal_fail(vs_status s, const char* message) { return fail(s, "%s", message); }

// vs_noalloc.cu -- vs_render_static: the direct path of vs_render (S1 k_transform, S2+S4 k_raster_direct / k_raster_big,
// the surface-order sort, S5-S7 k_shade / k_shade_banded) for callers that must not allocate.  include/vs.h states the
// contract; DESIGN.md §1 the pipeline.
//
// Everything the pass writes besides the caller's outputs lives in ONE file-scope `static __device__` array of
// VS_STATIC_SCRATCH_BYTES (64 MiB; zero-initialised when the module is loaded; every GPU that loads the library holds it
// until the process exits).  The launchers are the ones vs_render uses, handed a VsChunk whose pointers lie inside the
// array, so the images and ids are bit-identical to vs_render's.
//
// In host code the NAME of a __device__ array is a host-side stand-in, not a device address.  The device address is
// fetched with cudaGetSymbolAddress, once per device, with that device current, in THIS file (the array is static: no
// other translation unit can name it), and only that pointer is ever given to a kernel or a memset.
//
// No cudaMalloc / cudaFree / cudaMallocAsync / mem-pool call and no allocating library routine is reachable from here:
// cudaMemcpyAsync (cameras, 64 bytes each, from the caller's host array), cudaMemsetAsync, cudaFuncSetAttribute and kernel
// launches only.
//
// Sharing: every call, scene and stream uses the same array, and it keeps the last call's contents.  What must start at
// zero (key image, tile masks, the big-triangle count, the counters) is cleared by every call on its own stream, so stale
// contents never matter -- but calls whose device work overlaps RACE.  Host-side, g_static_mu serialises the enqueueing.
#include <cstdio>
#include <mutex>

#include "../../include/vs.h"
#include "vs_common.cuh"
#include "vs_internal.cuh"

static __device__ __align__(256) unsigned char g_static_scratch[VS_STATIC_SCRATCH_BYTES];

#define VS_STATIC_MAX_DEVICES 64
#define VS_STATIC_BIG_CAPACITY 65536u   // entries of the very-large-triangle list (as in vs_render)
static std::mutex g_static_mu;
static unsigned char* g_static_base[VS_STATIC_MAX_DEVICES];   // device address of g_static_scratch per device; nullptr = not set up

namespace {
struct DeviceScope {   // makes `device` current and restores the caller's device on every exit path
    int prev = -1;
    bool switched = false;
    explicit DeviceScope(int device)
    {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != device) switched = cudaSetDevice(device) == cudaSuccess;
    }
    ~DeviceScope() { if (switched) cudaSetDevice(prev); }
};
}   // namespace

static vs_status static_fail(vs_status s, const char* what, cudaError_t e)
{
    char msg[384];
    snprintf(msg, sizeof(msg), "vs_render_static: %s: %s", what, cudaGetErrorString(e));
    cudaGetLastError();   // do not leave the error behind for the caller's next CUDA call
    return vs_internal_fail(s, msg);
}

#define CUS(call)                                                          \
    do {                                                                   \
        cudaError_t e_ = (call);                                           \
        if (e_ != cudaSuccess) return static_fail(VS_ERR_CUDA, #call, e_); \
    } while (0)

// Set-up, once per device: the device address of the static array.  g_static_mu is held and `device` is current.
static vs_status static_scratch_base(int device, unsigned char** base)
{
    if (device < 0 || device >= VS_STATIC_MAX_DEVICES)
        return vs_internal_fail(VS_ERR_UNSUPPORTED, "vs_render_static: device ordinal beyond 63");
    if (!g_static_base[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return static_fail(VS_ERR_CUDA, "cudaGetSymbolAddress(static scratch)", e);
        if (!p || ((unsigned long long)p & 255ull))
            return vs_internal_fail(VS_ERR_CUDA, "vs_render_static: the static scratch has no (aligned) device address");
        g_static_base[device] = (unsigned char*)p;
    }
    *base = g_static_base[device];
    return VS_OK;
}

// Carves the pass's buffers out of the static array: every buffer starts on a 256-byte boundary.
struct StaticLayout {
    size_t cams, counters, big_count, big_list, tile_mask, order, order_work, vtx, keys, end;
};

static StaticLayout static_layout(const VsSceneDev& sc, const VsFrame& fr, uint32_t views, bool ordered)
{
    StaticLayout L{};
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t at = off; off += (bytes + 255) & ~(size_t)255; return at; };
    const size_t ntile = (size_t)views * fr.tiles_x * fr.tiles_y;
    L.cams = take((size_t)views * sizeof(VsCamDev));
    L.counters = take(VS_CNT_N * 8);
    L.big_count = take(16);
    L.big_list = take((size_t)VS_STATIC_BIG_CAPACITY * 8);
    L.tile_mask = take(ntile * 4);
    L.order = take(ordered ? ntile * 4 + 16 : 0);
    L.order_work = take(ordered ? (2 * ntile + VS_ORDER_BINS) * 4 + 16 : 0);
    L.vtx = take((size_t)sc.v_total * views * 16 + 16);
    L.keys = take((size_t)views * sc.k * fr.width * fr.height * 8 + 16);
    L.end = off;
    return L;
}

extern "C" vs_status vs_render_static(vs_scene* scene, const vs_camera* cameras, uint32_t num_cameras,
                                      const vs_render_params* params, float* out_rgba, uint32_t* out_tri_ids,
                                      void* cuda_stream)
{
    vs_status r = vs_internal_validate_render(scene, cameras, num_cameras, params, out_rgba);
    if (r != VS_OK) return r;
    if (params->flags & ~(uint32_t)(VS_FLAG_ATTENUATION | VS_FLAG_SCREEN_ORDER))
        return vs_internal_fail(VS_ERR_UNSUPPORTED, "vs_render_static: only VS_FLAG_ATTENUATION and VS_FLAG_SCREEN_ORDER are supported "
                                                    "(direct path, no statistics)");
    if (num_cameras == 0) return VS_OK;
    const VsSceneDev* devp = nullptr;
    int tex_f16 = 0, device = 0;
    vs_internal_scene_view(scene, &devp, &tex_f16, &device);
    const VsSceneDev& sc = *devp;

    VsFrame fr{};
    fr.width = params->width; fr.height = params->height;
    fr.tiles_x = (params->width + VS_TILE_W - 1) / VS_TILE_W; fr.tiles_y = (params->height + VS_TILE_H - 1) / VS_TILE_H;
    fr.near_plane = params->near_plane; fr.t_min = params->t_min;
    for (int i = 0; i < 3; ++i) fr.bg[i] = params->background[i];
    fr.attenuate = (params->flags & VS_FLAG_ATTENUATION) ? 1u : 0u;
    // (same rule as vs_render: banded scenes keep screen order)
    const bool ordered = !(params->flags & VS_FLAG_SCREEN_ORDER) && !sc.banded;

    // sizes first, against the fixed capacity (num_cameras <= 2^16 keeps every product below 2^64)
    if (num_cameras > 65536u)
        return vs_internal_fail(VS_ERR_UNSUPPORTED, "vs_render_static: more than 65536 cameras in one call");
    const StaticLayout L = static_layout(sc, fr, num_cameras, ordered);
    if (L.end > (size_t)VS_STATIC_SCRATCH_BYTES) {
        char msg[384];
        snprintf(msg, sizeof(msg), "vs_render_static: this call needs %zu bytes of scratch (%u cameras x %u layers x %u x %u px, "
                 "%u vertices) but the static scratch holds %zu: render fewer cameras per call or use vs_render",
                 L.end, num_cameras, sc.k, params->width, params->height, sc.v_total, (size_t)VS_STATIC_SCRATCH_BYTES);
        return vs_internal_fail(VS_ERR_UNSUPPORTED, msg);
    }

    std::lock_guard<std::mutex> lock(g_static_mu);
    DeviceScope scope(device);
    unsigned char* base = nullptr;
    if ((r = static_scratch_base(device, &base)) != VS_OK) return r;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t ntile = (size_t)num_cameras * fr.tiles_x * fr.tiles_y;

    VsChunk ch{};
    ch.views = num_cameras;
    ch.cams = (const VsCamDev*)(base + L.cams);
    ch.vtx = (int4*)(base + L.vtx);
    ch.counters = (unsigned long long*)(base + L.counters);
    ch.out_rgba = out_rgba;
    ch.ids = out_tri_ids;
    ch.ids_is_output = out_tri_ids != nullptr;
    ch.keys = (unsigned long long*)(base + L.keys);
    ch.big_list = (uint2*)(base + L.big_list);
    ch.big_count = (uint32_t*)(base + L.big_count);
    ch.big_capacity = VS_STATIC_BIG_CAPACITY;
    ch.tile_mask = (uint32_t*)(base + L.tile_mask);
    ch.tile_count = ch.tile_mask;
    ch.order = ordered ? (const uint32_t*)(base + L.order) : nullptr;

    // the array keeps the previous call's contents: cameras in, and zeros where the kernels expect zeros
    static_assert(sizeof(VsCamDev) == sizeof(vs_camera), "camera layout");
    CUS(cudaMemcpyAsync(base + L.cams, cameras, (size_t)num_cameras * sizeof(VsCamDev), cudaMemcpyHostToDevice, st));
    CUS(cudaMemsetAsync(base + L.counters, 0, VS_CNT_N * 8, st));
    CUS(cudaMemsetAsync(base + L.big_count, 0, 16, st));
    CUS(cudaMemsetAsync(base + L.tile_mask, 0, ntile * 4, st));
    CUS(cudaMemsetAsync(base + L.keys, 0, (size_t)num_cameras * sc.k * fr.width * fr.height * 8, st));

    CUS(vs_launch_transform(sc, fr, ch, st));
    CUS(vs_launch_raster_direct(sc, fr, ch, st, 0u));
    if (ordered) CUS(vs_launch_order(sc, fr, ch, (uint32_t*)(base + L.order), (uint32_t*)(base + L.order_work), st));
    if (sc.banded) CUS(vs_launch_shade_banded(sc, fr, ch, st));
    else CUS(vs_launch_shade(sc, tex_f16, fr, ch, st));
    return VS_OK;
}

// vs_kernels_order.cu -- shading order of a chunk's (view, tile) pairs: surface order instead of screen order.
// DESIGN.md §7 ("surface-ordered shading").
//
// The views of one vs_render call look at the same textures, and a texel that one view needs is needed by every other
// view that sees the same piece of surface.  In screen order (all tiles of view 0, then view 1, ...) a view streams
// ~1.3 GB of texels through the 126 MB L2, so nothing survives until the next view asks for it.  These kernels sort the
// chunk's (view, tile) pairs by WHERE ON THE OBJECT the tile looks: the key is the Morton code of the object-space cell
// (32^3 over the scene's bounding box) of the front-most triangle at the tile's centre.  k_shade / k_backward then take
// their (view, tile) from the sorted list, so the CTAs resident at any time shade the same few surface cells in all the
// views that see them, and the texels (and the gradient texels of the backward pass) are shared through L2.
// The order changes scheduling only: every pixel is computed by the same instructions on the same operands.
//
// Counting sort: k_order_key (key + rank inside its bin), k_order_scan (one CTA, exclusive scan of the 32769 bins),
// k_order_scatter.  The rank comes from an atomic counter, so the order INSIDE a bin varies from run to run; nothing
// downstream depends on it.
#include "vs_common.cuh"

__device__ __forceinline__ uint32_t vs_spread3(uint32_t v)   // 5 bits -> every third bit
{
    v = (v | (v << 8)) & 0x0000F00Fu;
    v = (v | (v << 4)) & 0x000C30C3u;
    v = (v | (v << 2)) & 0x00249249u;
    return v;
}

#ifndef VS_ORDER_LAYER_NUM
#define VS_ORDER_LAYER_NUM 3   // the probe starts at layer k * VS_ORDER_LAYER_NUM / 8
#endif

// Hilbert curve index of cell (x, y) of a 2^bits x 2^bits grid
__device__ __forceinline__ uint32_t vs_hilbert2(uint32_t x, uint32_t y, int bits)
{
    uint32_t d = 0;
    for (uint32_t s = 1u << (bits - 1); s > 0; s >>= 1) {
        const uint32_t rx = (x & s) ? 1u : 0u, ry = (y & s) ? 1u : 0u;
        d += s * s * ((3u * rx) ^ ry);
        if (ry == 0) {   // rotate the quadrant
            if (rx == 1) { x = s - 1 - (x & (s - 1)); y = s - 1 - (y & (s - 1)); } else { x &= s - 1; y &= s - 1; }
            const uint32_t t = x; x = y; y = t;
        } else { x &= s - 1; y &= s - 1; }
    }
    return d;
}

__global__ void __launch_bounds__(256)
k_order_key(const VsSceneDev sc, const VsFrame fr, const unsigned long long* __restrict__ keys, const uint32_t* __restrict__ tile_mask,
            uint32_t views, uint32_t* __restrict__ okey, uint32_t* __restrict__ orank, uint32_t* __restrict__ hist)
{
    const uint32_t tiles = fr.tiles_x * fr.tiles_y;
    const uint32_t vt = blockIdx.x * blockDim.x + threadIdx.x;
    if (vt >= views * tiles) return;
    const uint32_t view = vt / tiles, tile = vt - view * tiles;
    const int W = (int)fr.width, H = (int)fr.height;
    const size_t plane = (size_t)W * H;
    const int x0 = (int)(tile % fr.tiles_x) * VS_TILE_W, y0 = (int)(tile / fr.tiles_x) * VS_TILE_H;
    const uint32_t lmask = tile_mask[vt];
    uint32_t key = VS_ORDER_BINS - 1u;   // nothing found: background and silhouette-corner tiles go last
    if (lmask) {
        // centre of the tile first, then the centres of its quadrants; per probe the keys of all layers are requested at once
        const int probe_x[5] = {8, 4, 12, 12, 4}, probe_y[5] = {8, 4, 12, 4, 12};
        // the reference layer: start a third of the way in (VS_ORDER_LAYER_NUM / 8 of k).  Seen from different directions, the
        // fragments of a pixel's deeper layers lie on different parts of the inner shells (parallax); a reference layer in
        // the middle of the shaded ones halves the largest offset (k_shade DRAM reads 11.7 -> 8.5 GB per 16-view C4 launch)
        const uint32_t l0 = (sc.k * VS_ORDER_LAYER_NUM) / 8u;
        for (int p = 0; p < 5; ++p) {
            const int px = min(x0 + probe_x[p], W - 1), py = min(y0 + probe_y[p], H - 1);
            const unsigned long long* kp = keys + (size_t)view * sc.k * plane + (size_t)py * W + px;
            unsigned long long kk[VS_MAX_LAYERS];
#pragma unroll
            for (int l = 0; l < VS_MAX_LAYERS; ++l) kk[l] = ((uint32_t)l < sc.k && ((lmask >> l) & 1u)) ? kp[(size_t)l * plane] : 0ull;
            unsigned long long hit = 0ull;
            uint32_t hl = 0, best = 0xFFFFFFFFu;   // the hit layer that comes first in the order l0, l0 + 1, ..., k - 1, 0, ..., l0 - 1
#pragma unroll
            for (int l = 0; l < VS_MAX_LAYERS; ++l) {
                const uint32_t rank = ((uint32_t)l + sc.k - l0) % sc.k;
                if (kk[l] && rank < best) { best = rank; hit = kk[l]; hl = (uint32_t)l; }
            }
            if (!hit) continue;
            const uint32_t lid = 0xFFFFFFFFu - (uint32_t)hit;
            const uint4 tri = __ldg(&sc.tris[sc.tri_off[hl] + lid]);
            const float* P = sc.positions + (size_t)tri.x * 3;
            const float cx = (__ldg(P) - sc.bb_min[0]) * sc.bb_scale[0], cy = (__ldg(P + 1) - sc.bb_min[1]) * sc.bb_scale[1];
            const float cz = (__ldg(P + 2) - sc.bb_min[2]) * sc.bb_scale[2];
            if (VS_ORDER_MODE == 0) {
                const uint32_t ix = (uint32_t)min(max((int)cx, 0), 31), iy = (uint32_t)min(max((int)cy, 0), 31);
                const uint32_t iz = (uint32_t)min(max((int)cz, 0), 31);
                key = vs_spread3(ix) | (vs_spread3(iy) << 1) | (vs_spread3(iz) << 2);
            } else {
                // direction from the box centre in box units -> octahedral map -> 2^VS_ORDER_BITS squared cells along a Hilbert
                // curve: a range of consecutive keys is a compact patch of the object's surface
                float dx = cx - 16.0f, dy = cy - 16.0f, dz = cz - 16.0f;
                const float n1 = fabsf(dx) + fabsf(dy) + fabsf(dz);
                const float inv = n1 > 0.0f ? 1.0f / n1 : 0.0f;
                dx *= inv; dy *= inv; dz *= inv;
                float ox = dx, oy = dy;
                if (dz < 0.0f) { ox = (1.0f - fabsf(dy)) * (dx < 0.0f ? -1.0f : 1.0f); oy = (1.0f - fabsf(dx)) * (dy < 0.0f ? -1.0f : 1.0f); }
                constexpr int NC = 1 << VS_ORDER_BITS;
                const uint32_t ux = (uint32_t)min(max((int)((ox * 0.5f + 0.5f) * (float)NC), 0), NC - 1);
                const uint32_t uy = (uint32_t)min(max((int)((oy * 0.5f + 0.5f) * (float)NC), 0), NC - 1);
                key = vs_hilbert2(ux, uy, VS_ORDER_BITS);
            }
            break;
        }
    }
    okey[vt] = key;
    // rank inside the bin: one atomic per distinct key of the warp (most background tiles share ONE bin: per-thread atomics on
    // it serialise in L2 and took 55 of the kernel's 60 us)
    const uint32_t active = __activemask();
    const uint32_t peers = __match_any_sync(active, key);
    const uint32_t leader = (uint32_t)__ffs(peers) - 1u, lane = threadIdx.x & 31u;
    uint32_t base = 0;
    if (lane == leader) base = atomicAdd(&hist[key], (uint32_t)__popc(peers));
    base = __shfl_sync(peers, base, (int)leader);
    orank[vt] = base + (uint32_t)__popc(peers & ((1u << lane) - 1u));
}

// one CTA of 1024 threads: hist[VS_ORDER_BINS] -> exclusive prefix sums, in place
__global__ void __launch_bounds__(1024)
k_order_scan(uint32_t* __restrict__ hist)
{
    constexpr uint32_t PER = (VS_ORDER_BINS + 1023u) / 1024u;
    __shared__ uint32_t warp_sum[32];
    const uint32_t t = threadIdx.x, lane = t & 31, warp = t >> 5;
    uint32_t v[PER], sum = 0;
#pragma unroll
    for (uint32_t i = 0; i < PER; ++i) {
        const uint32_t b = t * PER + i;
        v[i] = b < VS_ORDER_BINS ? hist[b] : 0u;
        sum += v[i];
    }
    uint32_t incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= (uint32_t)o) incl += u;
    }
    if (lane == 31) warp_sum[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = warp_sum[lane], wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, wi, o);
            if (lane >= (uint32_t)o) wi += u;
        }
        warp_sum[lane] = wi - w;
    }
    __syncthreads();
    uint32_t run = warp_sum[warp] + incl - sum;
#pragma unroll
    for (uint32_t i = 0; i < PER; ++i) {
        const uint32_t b = t * PER + i;
        if (b < VS_ORDER_BINS) hist[b] = run;
        run += v[i];
    }
}

__global__ void __launch_bounds__(256)
k_order_scatter(const uint32_t* __restrict__ okey, const uint32_t* __restrict__ orank, const uint32_t* __restrict__ base, uint32_t n,
                uint32_t* __restrict__ order)
{
    const uint32_t vt = blockIdx.x * blockDim.x + threadIdx.x;
    if (vt < n) order[base[okey[vt]] + orank[vt]] = vt;
}

// order[views * tiles] <- the chunk's (view * tiles + tile) indices in surface order.  `work` holds 2 * views * tiles +
// VS_ORDER_BINS words.  Needs the finished key image of the direct path (before the consumer clears it).
cudaError_t vs_launch_order(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, uint32_t* order, uint32_t* work, cudaStream_t st)
{
    const uint32_t n = ch.views * fr.tiles_x * fr.tiles_y;
    if (n == 0) return cudaSuccess;
    uint32_t* okey = work, *orank = work + n, *hist = work + 2 * (size_t)n;
    cudaError_t e = cudaMemsetAsync(hist, 0, VS_ORDER_BINS * 4, st);
    if (e != cudaSuccess) return e;
    k_order_key<<<(n + 255) / 256, 256, 0, st>>>(sc, fr, ch.keys, ch.tile_mask, ch.views, okey, orank, hist);
    k_order_scan<<<1, 1024, 0, st>>>(hist);
    k_order_scatter<<<(n + 255) / 256, 256, 0, st>>>(okey, orank, hist, n, order);
    return cudaGetLastError();
}

// ---- scene bounding box (scene creation) ----
__device__ __forceinline__ int vs_float_ordered(float f)
{
    const int i = __float_as_int(f);
    return i ^ ((i >> 31) & 0x7FFFFFFF);
}

// bb[0..2] = min, bb[3..5] = max of the positions, as order-preserving ints (initialised by the launcher)
__global__ void __launch_bounds__(256)
k_bbox(const float* __restrict__ pos, uint32_t n_vertices, int* __restrict__ bb)
{
    int lo[3] = {0x7FFFFFFF, 0x7FFFFFFF, 0x7FFFFFFF}, hi[3] = {(int)0x80000000, (int)0x80000000, (int)0x80000000};
    for (uint32_t v = blockIdx.x * blockDim.x + threadIdx.x; v < n_vertices; v += gridDim.x * blockDim.x)
        for (int a = 0; a < 3; ++a) {
            const int o = vs_float_ordered(pos[(size_t)v * 3 + a]);
            lo[a] = min(lo[a], o); hi[a] = max(hi[a], o);
        }
    for (int a = 0; a < 3; ++a) {
        lo[a] = __reduce_min_sync(0xFFFFFFFFu, lo[a]); hi[a] = __reduce_max_sync(0xFFFFFFFFu, hi[a]);
    }
    if ((threadIdx.x & 31) == 0)
        for (int a = 0; a < 3; ++a) { atomicMin(&bb[a], lo[a]); atomicMax(&bb[3 + a], hi[a]); }
}

cudaError_t vs_launch_bbox(const float* pos, uint32_t n_vertices, int* bb6, cudaStream_t st)
{
    const int init[6] = {0x7FFFFFFF, 0x7FFFFFFF, 0x7FFFFFFF, (int)0x80000000, (int)0x80000000, (int)0x80000000};
    cudaError_t e = cudaMemcpyAsync(bb6, init, sizeof(init), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return e;
    if (n_vertices == 0) return cudaSuccess;
    k_bbox<<<148, 256, 0, st>>>(pos, n_vertices, bb6);
    return cudaGetLastError();
}

// vs_kernels_geom.cu -- S0 scene packing, S1 vertex transform, S2 triangle setup + S3 tile binning
// (count / warp-scan prefix sum / scatter).  DESIGN.md §1, §3.1-3.2, §7.
#include "vs_common.cuh"

// ------------------------------------------------------------------------------------------------
// S0: scene packing (once per scene)
// ------------------------------------------------------------------------------------------------
__global__ void k_pack_tris(const uint32_t* __restrict__ idx, const float* __restrict__ pos, uint32_t nt, uint32_t nv,
                            uint32_t voff, uint32_t layer, uint4* __restrict__ out, float4* __restrict__ nrm, uint32_t* err)
{
    uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nt) return;
    uint32_t a = idx[3 * (size_t)t], b = idx[3 * (size_t)t + 1], c = idx[3 * (size_t)t + 2];
    if (a >= nv || b >= nv || c >= nv) { atomicOr(err, 1u); a = b = c = 0; }
    out[t] = make_uint4(a + voff, b + voff, c + voff, (layer << 28) | t);
    // unit geometric normal (for the transparency attenuation): fp64 cross product of the fp32 positions, once per scene
    const double ax = (double)pos[3 * (size_t)b] - (double)pos[3 * (size_t)a], ay = (double)pos[3 * (size_t)b + 1] - (double)pos[3 * (size_t)a + 1],
                 az = (double)pos[3 * (size_t)b + 2] - (double)pos[3 * (size_t)a + 2];
    const double bx = (double)pos[3 * (size_t)c] - (double)pos[3 * (size_t)a], by = (double)pos[3 * (size_t)c + 1] - (double)pos[3 * (size_t)a + 1],
                 bz = (double)pos[3 * (size_t)c + 2] - (double)pos[3 * (size_t)a + 2];
    const double nx = ay * bz - az * by, ny = az * bx - ax * bz, nz = ax * by - ay * bx;
    const double len = sqrt(nx * nx + ny * ny + nz * nz);
    const double inv = len > 0.0 ? 1.0 / len : 0.0;
    nrm[t] = make_float4((float)(nx * inv), (float)(ny * inv), (float)(nz * inv), 0.0f);
}

__global__ void k_check_finite(const float* __restrict__ v, size_t n, uint32_t* err)
{
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && !isfinite(v[i])) atomicOr(err, 2u);
}

// API layout [texel][c][ch] (float or half) -> internal [texel][ch][np_pad]: channel-major so that a
// 16-byte vector holds consecutive coefficients of ONE channel; rows zero-padded to np_pad.
// frag: the mma A-fragment order of vs_common.cuh (fp16, np_pad == 16) instead of the channel-major one.
template <typename T>
__global__ void k_pack_texture(const T* __restrict__ src, uint32_t n_texels, uint32_t n_coef, uint32_t np_pad, uint32_t frag,
                               T* __restrict__ dst)
{
    const uint32_t dst_elems = 4 * np_pad, src_elems = n_coef * 4;
    size_t total = (size_t)n_texels * dst_elems;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        size_t texel = i / dst_elems;
        uint32_t e = (uint32_t)(i - texel * dst_elems);
        uint32_t ch = e / np_pad, c = e - ch * np_pad;
        if (frag) {   // inverse of vs_frag_half_index
            const uint32_t v = e >> 3, r = e & 7u;
            ch = (v >> 2) + 2u * ((r >> 1) & 1u);
            c = (v & 3u) * 2u + (r & 1u) + 8u * (r >> 2);
        }
        dst[i] = c < n_coef ? src[texel * src_elems + 4 * c + ch] : T(0);
    }
}

// banded 8-bit textures: API texel of (2b+1) x 4 bytes -> internal texel of VS_BAND_STRIDE(b) bytes, zero padded
__global__ void k_pack_band(const unsigned char* __restrict__ src, uint32_t n_texels, uint32_t src_stride, uint32_t dst_stride,
                            unsigned char* __restrict__ dst)
{
    const size_t total = (size_t)n_texels * dst_stride;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const size_t texel = i / dst_stride;
        const uint32_t e = (uint32_t)(i - texel * dst_stride);
        dst[i] = e < src_stride ? src[texel * src_stride + e] : (unsigned char)0;
    }
}

cudaError_t vs_launch_pack_band(const unsigned char* src, uint32_t n_texels, uint32_t band, unsigned char* dst, cudaStream_t st)
{
    k_pack_band<<<148 * 8, 256, 0, st>>>(src, n_texels, (2 * band + 1) * 4, VS_BAND_STRIDE(band), dst);
    return cudaGetLastError();
}

cudaError_t vs_launch_pack_tris(const uint32_t* indices, const float* layer_positions, uint32_t num_tris, uint32_t num_vertices,
                                uint32_t vtx_off, uint32_t layer, uint4* out, float4* out_normals, uint32_t* error_flag, cudaStream_t st)
{
    if (num_tris == 0) return cudaSuccess;
    k_pack_tris<<<(num_tris + 255) / 256, 256, 0, st>>>(indices, layer_positions, num_tris, num_vertices, vtx_off, layer, out,
                                                        out_normals, error_flag);
    return cudaGetLastError();
}

// per-vertex normals [n][3] -> float4 (w = 0)
__global__ void k_pack_normals(const float* __restrict__ src, uint32_t n, float4* __restrict__ dst)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = make_float4(src[3 * (size_t)i], src[3 * (size_t)i + 1], src[3 * (size_t)i + 2], 0.0f);
}

cudaError_t vs_launch_pack_normals(const float* src, uint32_t n, float4* dst, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    k_pack_normals<<<(n + 255) / 256, 256, 0, st>>>(src, n, dst);
    return cudaGetLastError();
}

cudaError_t vs_launch_check_finite(const float* v, size_t n, uint32_t* error_flag, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    k_check_finite<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(v, n, error_flag);
    return cudaGetLastError();
}

cudaError_t vs_launch_pack_texture(const void* src, int f16, uint32_t n_texels, uint32_t n_coef, uint32_t np_pad, uint32_t frag_layout,
                                   uint4* dst, cudaStream_t st)
{
    const int blocks = 148 * 16;
    if (f16)
        k_pack_texture<__half><<<blocks, 256, 0, st>>>((const __half*)src, n_texels, n_coef, np_pad, frag_layout, (__half*)dst);
    else
        k_pack_texture<float><<<blocks, 256, 0, st>>>((const float*)src, n_texels, n_coef, np_pad, 0u, (float*)dst);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// S1: vertex transform (fp32-exact).  One thread per (view, vertex).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_transform(VsSceneDev sc, VsFrame fr, const VsCamDev* __restrict__ cams,
                                                   int4* __restrict__ vtx)
{
    const uint32_t v = blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= sc.v_total) return;
    const uint32_t view = blockIdx.y;
    const VsCamDev c = cams[view];
    float px = sc.positions[3 * (size_t)v], py = sc.positions[3 * (size_t)v + 1], pz = sc.positions[3 * (size_t)v + 2];
    float xc = __fmaf_rn(c.R[0], px, __fmaf_rn(c.R[1], py, __fmaf_rn(c.R[2], pz, c.t[0])));
    float yc = __fmaf_rn(c.R[3], px, __fmaf_rn(c.R[4], py, __fmaf_rn(c.R[5], pz, c.t[1])));
    float w = __fmaf_rn(c.R[6], px, __fmaf_rn(c.R[7], py, __fmaf_rn(c.R[8], pz, c.t[2])));
    int bad = 0;
    if (!(w >= fr.near_plane)) bad = 1;
    float q = __fdiv_rn(1.0f, w);
    float xs = __fmaf_rn(c.fx, __fmul_rn(xc, q), c.cx);
    float ys = __fmaf_rn(c.fy, __fmul_rn(yc, q), c.cy);
    if (!bad && !(fabsf(xs) < 16384.0f && fabsf(ys) < 16384.0f)) bad = 2;
    int X = 0, Y = 0;
    if (!bad) {
        X = __float2int_rn(__fmul_rn(xs, 256.0f));  // round-half-even
        Y = __float2int_rn(__fmul_rn(ys, 256.0f));
    }
    vtx[(size_t)view * sc.v_total + v] = make_int4(X, Y, __float_as_int(q), bad);
}

cudaError_t vs_launch_transform(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    if (sc.v_total == 0) return cudaSuccess;
    dim3 grid((sc.v_total + 255) / 256, ch.views);
    k_transform<<<grid, 256, 0, st>>>(sc, fr, ch.cams, ch.vtx);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// S2 + S3: triangle setup and tile binning.  One thread per (view, triangle).
//   k_bin_count  : setup, sample bounding box -> tile range; remembers the packed range per
//                  (view, triangle) and counts references per (view, tile).
//   k_scan       : exclusive prefix sum of the counters of the whole chunk.
//   k_bin_scatter: re-reads the packed range (no vertex gathers) and writes the triangle id into
//                  the tile's list.
// A triangle is referenced by every tile its sample-point bounding box touches.  Consecutive
// triangles of a mesh mostly fall into a handful of tiles, so the tile atomics are CTA-aggregated in
// a small shared-memory table and every distinct global counter is touched once per CTA.
// ------------------------------------------------------------------------------------------------
#define VS_RANGE_NONE 0xFFFFFFFFu   // triangle references no tile
#define VS_RANGE_WIDE 0xFFFFFFFEu   // more than 64 tiles in one direction: the scatter pass recomputes the range
#define VS_BIN_THREADS 512
#define VS_BIN_SLOTS 256            // per-CTA tile table (open addressing, <= VS_BIN_PROBES probes)
#define VS_BIN_PROBES 8
#define VS_BIN_EMPTY 0xFFFFFFFFu

__device__ __forceinline__ bool vs_tile_range(const VsSceneDev& sc, const VsFrame& fr, const int4* __restrict__ vv, uint32_t t,
                                              int& tx0, int& tx1, int& ty0, int& ty1, int& status)
{
    const uint4 tri = __ldg(&sc.tris[t]);
    const int4 a = __ldg(&vv[tri.x]), b = __ldg(&vv[tri.y]), c = __ldg(&vv[tri.z]);
    VsTri T;
    status = vs_setup_tri(a, b, c, T);
    int i0, i1, j0, j1;
    if (status != 0 || !vs_tri_pixel_bbox(T, (int)fr.width, (int)fr.height, i0, i1, j0, j1)) return false;
    tx0 = i0 / VS_TILE_W; tx1 = i1 / VS_TILE_W; ty0 = j0 / VS_TILE_H; ty1 = j1 / VS_TILE_H;
    return true;
}

__device__ __forceinline__ uint32_t vs_pack_range(int tx0, int tx1, int ty0, int ty1)
{
    const int nx = tx1 - tx0 + 1, ny = ty1 - ty0 + 1;
    return (nx > 64 || ny > 64) ? VS_RANGE_WIDE
                                : ((uint32_t)tx0 | ((uint32_t)ty0 << 10) | ((uint32_t)(nx - 1) << 20) | ((uint32_t)(ny - 1) << 26));
}

// Per-CTA tile table.  Consecutive triangles of a mesh mostly fall into a handful of tiles, so a CTA
// first sums its references per tile in shared memory and then touches every distinct global
// counter once.  vs_bin_find returns the slot of `tile` (inserting it) or -1 when the probe sequence
// is exhausted (the caller then falls back to a global atomic of its own).
__device__ __forceinline__ int vs_bin_find(uint32_t* __restrict__ keys, uint32_t tile)
{
    uint32_t h = (tile * 2654435761u) >> 24;  // 8 bits
#pragma unroll 1
    for (int p = 0; p < VS_BIN_PROBES; ++p) {
        const uint32_t s = (h + (uint32_t)p) & (VS_BIN_SLOTS - 1);
        const uint32_t k = keys[s];
        if (k == tile) return (int)s;
        if (k == VS_BIN_EMPTY) {
            const uint32_t old = atomicCAS(&keys[s], VS_BIN_EMPTY, tile);
            if (old == VS_BIN_EMPTY || old == tile) return (int)s;
        }
    }
    return -1;
}

// Pass 1: setup + sample bounding box -> tile range per (view, triangle) and reference counts per
// (view, tile).  The chunk's total is read off the prefix sum afterwards (no counter traffic here).
__global__ void __launch_bounds__(VS_BIN_THREADS) k_bin_count(VsSceneDev sc, VsFrame fr, const int4* __restrict__ vtx,
                                                              uint32_t* __restrict__ tri_tiles, uint32_t* __restrict__ tile_count,
                                                              unsigned long long* counters)
{
    __shared__ uint32_t skey[VS_BIN_SLOTS], scnt[VS_BIN_SLOTS];
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31;
    const uint32_t view = blockIdx.y;
    const uint32_t tiles = fr.tiles_x * fr.tiles_y;
    for (uint32_t i = threadIdx.x; i < VS_BIN_SLOTS; i += blockDim.x) { skey[i] = VS_BIN_EMPTY; scnt[i] = 0; }
    __syncthreads();
    int status = -1, tx0 = 0, tx1 = -1, ty0 = 0, ty1 = -1;
    bool any = false;
    if (t < sc.t_total) {
        any = vs_tile_range(sc, fr, vtx + (size_t)view * sc.v_total, t, tx0, tx1, ty0, ty1, status);
        tri_tiles[(size_t)view * sc.t_total + t] = any ? vs_pack_range(tx0, tx1, ty0, ty1) : VS_RANGE_NONE;
    }
    if (any)
        for (int ty = ty0; ty <= ty1; ++ty)
            for (int tx = tx0; tx <= tx1; ++tx) {
                const uint32_t tile = (uint32_t)ty * fr.tiles_x + (uint32_t)tx;
                const int s = vs_bin_find(skey, tile);
                if (s >= 0) atomicAdd(&scnt[s], 1u);
                else atomicAdd(&tile_count[view * tiles + tile], 1u);
            }
    const unsigned full = 0xFFFFFFFFu;
    const unsigned dropped = __popc(__ballot_sync(full, status == 1));
    const unsigned degen = __popc(__ballot_sync(full, status == 2));
    if (lane == 0) {
        if (dropped) atomicAdd(&counters[VS_CNT_DROPPED], (unsigned long long)dropped);
        if (degen) atomicAdd(&counters[VS_CNT_DEGENERATE], (unsigned long long)degen);
    }
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < VS_BIN_SLOTS; i += blockDim.x)
        if (skey[i] != VS_BIN_EMPTY) atomicAdd(&tile_count[view * tiles + skey[i]], scnt[i]);
}

// Pass 2: re-reads the packed range (no vertex gathers), reserves the CTA's references of every
// distinct tile with one global atomic, and writes the triangle ids into the tiles' lists.
__global__ void __launch_bounds__(VS_BIN_THREADS) k_bin_scatter(VsSceneDev sc, VsFrame fr, const int4* __restrict__ vtx,
                                                                const uint32_t* __restrict__ tri_tiles, uint32_t* __restrict__ tile_cursor,
                                                                const uint32_t* __restrict__ tile_off, uint32_t* __restrict__ tile_tris,
                                                                uint32_t ref_capacity)
{
    __shared__ uint32_t skey[VS_BIN_SLOTS], scnt[VS_BIN_SLOTS];
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t view = blockIdx.y;
    const uint32_t tiles = fr.tiles_x * fr.tiles_y;
    for (uint32_t i = threadIdx.x; i < VS_BIN_SLOTS; i += blockDim.x) { skey[i] = VS_BIN_EMPTY; scnt[i] = 0; }
    __syncthreads();
    const uint32_t packed = t < sc.t_total ? __ldg(&tri_tiles[(size_t)view * sc.t_total + t]) : VS_RANGE_NONE;
    int tx0 = 0, tx1 = -1, ty0 = 0, ty1 = -1;
    if (packed == VS_RANGE_WIDE) {
        int status;
        vs_tile_range(sc, fr, vtx + (size_t)view * sc.v_total, t, tx0, tx1, ty0, ty1, status);
    } else if (packed != VS_RANGE_NONE) {
        tx0 = (int)(packed & 1023u); ty0 = (int)((packed >> 10) & 1023u);
        tx1 = tx0 + (int)((packed >> 20) & 63u); ty1 = ty0 + (int)(packed >> 26);
    }
    // phase 1: count per tile inside the CTA; references that miss the table go out directly
    for (int ty = ty0; ty <= ty1; ++ty)
        for (int tx = tx0; tx <= tx1; ++tx) {
            const uint32_t tile = (uint32_t)ty * fr.tiles_x + (uint32_t)tx;
            const int s = vs_bin_find(skey, tile);
            if (s >= 0) atomicAdd(&scnt[s], 1u);
            else {
                const uint32_t g = view * tiles + tile;
                const uint32_t pos = __ldg(&tile_off[g]) + atomicAdd(&tile_cursor[g], 1u);
                if (pos < ref_capacity) tile_tris[pos] = t;
            }
        }
    __syncthreads();
    // phase 2: one reservation per distinct tile; scnt becomes the next free position of the CTA's run
    for (uint32_t i = threadIdx.x; i < VS_BIN_SLOTS; i += blockDim.x)
        if (skey[i] != VS_BIN_EMPTY) {
            const uint32_t g = view * tiles + skey[i];
            scnt[i] = __ldg(&tile_off[g]) + atomicAdd(&tile_cursor[g], scnt[i]);
        }
    __syncthreads();
    // phase 3: write the references (the table is read-only now, so lookups cannot insert)
    for (int ty = ty0; ty <= ty1; ++ty)
        for (int tx = tx0; tx <= tx1; ++tx) {
            const uint32_t tile = (uint32_t)ty * fr.tiles_x + (uint32_t)tx;
            const uint32_t h = (tile * 2654435761u) >> 24;
            for (int p = 0; p < VS_BIN_PROBES; ++p) {
                const uint32_t s = (h + (uint32_t)p) & (VS_BIN_SLOTS - 1);
                const uint32_t k = skey[s];
                if (k == tile) {
                    const uint32_t pos = atomicAdd(&scnt[s], 1u);
                    if (pos < ref_capacity) tile_tris[pos] = t;
                    break;
                }
                if (k == VS_BIN_EMPTY) break;  // went out directly in phase 1
            }
        }
}

cudaError_t vs_launch_bin_count(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    if (sc.t_total == 0) return cudaSuccess;
    dim3 grid((sc.t_total + VS_BIN_THREADS - 1) / VS_BIN_THREADS, ch.views);
    k_bin_count<<<grid, VS_BIN_THREADS, 0, st>>>(sc, fr, ch.vtx, ch.tri_tiles, ch.tile_count, ch.counters);
    return cudaGetLastError();
}

cudaError_t vs_launch_bin_scatter(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    if (sc.t_total == 0) return cudaSuccess;
    dim3 grid((sc.t_total + VS_BIN_THREADS - 1) / VS_BIN_THREADS, ch.views);
    k_bin_scatter<<<grid, VS_BIN_THREADS, 0, st>>>(sc, fr, ch.vtx, ch.tri_tiles, ch.tile_cursor, ch.tile_off, ch.tile_tris, ch.ref_capacity);
    return cudaGetLastError();
}

// Exclusive prefix sum of the tile counters of the whole chunk, off[n] = total.  One 1024-thread
// block per view: the block first sums the counters of all earlier views (its base; no block waits
// on another), then scans its own view in coalesced 1024-element pieces with warp-shuffle scans.
__device__ __forceinline__ uint32_t vs_block_scan_1024(uint32_t v, uint32_t* warp_sums, uint32_t& total)
{
    const uint32_t lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t incl = v;
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= (uint32_t)o) incl += u;
    }
    __syncthreads();  // warp_sums may still be read from the previous call
    if (lane == 31) warp_sums[wid] = incl;
    __syncthreads();
    uint32_t w = warp_sums[lane], wi = w;
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, wi, o);
        if (lane >= (uint32_t)o) wi += u;
    }
    total = __shfl_sync(0xFFFFFFFFu, wi, 31);
    const uint32_t wbase = __shfl_sync(0xFFFFFFFFu, wi - w, wid);
    return wbase + incl - v;  // exclusive
}

__global__ void __launch_bounds__(1024) k_scan(const uint32_t* __restrict__ count, uint32_t tiles, uint32_t views,
                                               uint32_t* __restrict__ off, uint32_t ref_capacity, unsigned long long* counters)
{
    __shared__ uint32_t warp_sums[32];
    const uint32_t view = blockIdx.x, tid = threadIdx.x;
    uint32_t mine = 0;
    for (uint32_t i = tid; i < view * tiles; i += 1024) mine += __ldg(&count[i]);
    uint32_t base;
    vs_block_scan_1024(mine, warp_sums, base);
    const uint32_t* c = count + (size_t)view * tiles;
    uint32_t* o = off + (size_t)view * tiles;
    for (uint32_t i0 = 0; i0 < tiles; i0 += 1024) {
        const uint32_t i = i0 + tid;
        const uint32_t v = i < tiles ? __ldg(&c[i]) : 0u;
        uint32_t total;
        const uint32_t ex = vs_block_scan_1024(v, warp_sums, total);
        if (i < tiles) o[i] = base + ex;
        base += total;
    }
    if (view == views - 1 && tid == 0) {
        off[(size_t)views * tiles] = base;
        atomicAdd(&counters[VS_CNT_REFS], (unsigned long long)base);
        if (base > ref_capacity) atomicMax(&counters[VS_CNT_OVERFLOW], (unsigned long long)base);
    }
}

cudaError_t vs_launch_bin_scan(const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    k_scan<<<ch.views, 1024, 0, st>>>(ch.tile_count, fr.tiles_x * fr.tiles_y, ch.views, ch.tile_off, ch.ref_capacity, ch.counters);
    return cudaGetLastError();
}

// vs_kernels_geom.cu -- S0 scene packing, S1 vertex transform, S2 triangle setup + S3 tile binning
// (count / warp-scan prefix sum / scatter).  DESIGN.md §1, §3.1-3.2, §7.
#include "vs_common.cuh"

// ------------------------------------------------------------------------------------------------
// S0: scene packing (once per scene)
// ------------------------------------------------------------------------------------------------
__global__ void k_pack_tris(const uint32_t* __restrict__ idx, uint32_t nt, uint32_t nv, uint32_t voff, uint32_t layer,
                            uint4* __restrict__ out, uint32_t* err)
{
    uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nt) return;
    uint32_t a = idx[3 * (size_t)t], b = idx[3 * (size_t)t + 1], c = idx[3 * (size_t)t + 2];
    if (a >= nv || b >= nv || c >= nv) { atomicOr(err, 1u); a = b = c = 0; }
    out[t] = make_uint4(a + voff, b + voff, c + voff, layer);
}

__global__ void k_check_finite(const float* __restrict__ v, size_t n, uint32_t* err)
{
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && !isfinite(v[i])) atomicOr(err, 2u);
}

// API layout [texel][n][4] (float or half) -> internal [texel][texel_vecs] 16-byte vectors:
// the same element order, zero-padded to a multiple of 16 bytes per texel.
template <typename T>
__global__ void k_pack_texture(const T* __restrict__ src, uint32_t n_texels, uint32_t n_coef, uint32_t texel_vecs,
                               T* __restrict__ dst)
{
    const uint32_t per_vec = 16 / sizeof(T);
    const uint32_t dst_elems = texel_vecs * per_vec, src_elems = n_coef * 4;
    size_t total = (size_t)n_texels * dst_elems;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        size_t texel = i / dst_elems;
        uint32_t e = (uint32_t)(i - texel * dst_elems);
        dst[i] = e < src_elems ? src[texel * src_elems + e] : T(0);
    }
}

cudaError_t vs_launch_pack_tris(const uint32_t* indices, uint32_t num_tris, uint32_t num_vertices, uint32_t vtx_off,
                                uint32_t layer, uint4* out, uint32_t* error_flag, cudaStream_t st)
{
    if (num_tris == 0) return cudaSuccess;
    k_pack_tris<<<(num_tris + 255) / 256, 256, 0, st>>>(indices, num_tris, num_vertices, vtx_off, layer, out, error_flag);
    return cudaGetLastError();
}

cudaError_t vs_launch_check_finite(const float* v, size_t n, uint32_t* error_flag, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    k_check_finite<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(v, n, error_flag);
    return cudaGetLastError();
}

cudaError_t vs_launch_pack_texture(const void* src, int f16, uint32_t n_texels, uint32_t n_coef, uint32_t texel_vecs,
                                   uint4* dst, cudaStream_t st)
{
    const int blocks = 148 * 16;
    if (f16)
        k_pack_texture<__half><<<blocks, 256, 0, st>>>((const __half*)src, n_texels, n_coef, texel_vecs, (__half*)dst);
    else
        k_pack_texture<float><<<blocks, 256, 0, st>>>((const float*)src, n_texels, n_coef, texel_vecs, (float*)dst);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// S1: vertex transform (fp32-exact).  One thread per (view, vertex).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_transform(VsSceneDev sc, VsFrame fr, const VsCamDev* __restrict__ cams,
                                                   int4* __restrict__ vtx)
{
    uint32_t v = blockIdx.x * blockDim.x + threadIdx.x;
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
// S2 + S3: triangle setup and tile binning.  One thread per (view, triangle); the same code runs
// twice: COUNT (atomicAdd on the tile counters) and SCATTER (claim a slot, write the triangle id).
// A triangle is referenced by every tile its sample-point bounding box touches.
// ------------------------------------------------------------------------------------------------
template <bool SCATTER>
__global__ void __launch_bounds__(256) k_bin(VsSceneDev sc, VsFrame fr, const int4* __restrict__ vtx,
                                             uint32_t* __restrict__ tile_counter, const uint32_t* __restrict__ tile_off,
                                             uint32_t* __restrict__ tile_tris, unsigned long long* counters)
{
    uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t view = blockIdx.y;
    int status = -1;
    uint32_t refs = 0;
    if (t < sc.t_total) {
        const uint4 tri = __ldg(&sc.tris[t]);
        const int4* vv = vtx + (size_t)view * sc.v_total;
        const int4 a = __ldg(&vv[tri.x]), b = __ldg(&vv[tri.y]), c = __ldg(&vv[tri.z]);
        VsTri T;
        status = vs_setup_tri(a, b, c, T);
        int i0, i1, j0, j1;
        if (status == 0 && vs_tri_pixel_bbox(T, (int)fr.width, (int)fr.height, i0, i1, j0, j1)) {
            const int tx0 = i0 / VS_TILE_W, tx1 = i1 / VS_TILE_W, ty0 = j0 / VS_TILE_H, ty1 = j1 / VS_TILE_H;
            const uint32_t tiles = fr.tiles_x * fr.tiles_y;
            for (int ty = ty0; ty <= ty1; ++ty)
                for (int tx = tx0; tx <= tx1; ++tx) {
                    const uint32_t tile = view * tiles + (uint32_t)ty * fr.tiles_x + (uint32_t)tx;
                    const uint32_t slot = atomicAdd(&tile_counter[tile], 1u);
                    if (SCATTER) tile_tris[tile_off[tile] + slot] = t;
                    ++refs;
                }
        }
    }
    if (!SCATTER) {
        // warp-aggregated statistics
        const unsigned full = 0xFFFFFFFFu;
        unsigned dropped = __popc(__ballot_sync(full, status == 1));
        unsigned degen = __popc(__ballot_sync(full, status == 2));
        for (int o = 16; o > 0; o >>= 1) refs += __shfl_xor_sync(full, refs, o);
        if ((threadIdx.x & 31) == 0) {
            if (dropped) atomicAdd(&counters[VS_CNT_DROPPED], (unsigned long long)dropped);
            if (degen) atomicAdd(&counters[VS_CNT_DEGENERATE], (unsigned long long)degen);
            if (refs) atomicAdd(&counters[VS_CNT_REFS], (unsigned long long)refs);
        }
    }
}

cudaError_t vs_launch_bin_count(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    if (sc.t_total == 0) return cudaSuccess;
    dim3 grid((sc.t_total + 255) / 256, ch.views);
    k_bin<false><<<grid, 256, 0, st>>>(sc, fr, ch.vtx, ch.tile_count, nullptr, nullptr, ch.counters);
    return cudaGetLastError();
}

cudaError_t vs_launch_bin_scatter(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    if (sc.t_total == 0) return cudaSuccess;
    dim3 grid((sc.t_total + 255) / 256, ch.views);
    k_bin<true><<<grid, 256, 0, st>>>(sc, fr, ch.vtx, ch.tile_cursor, ch.tile_off, ch.tile_tris, ch.counters);
    return cudaGetLastError();
}

// Exclusive prefix sum of the tile counters of the whole chunk: one 1024-thread block, each thread
// scans a contiguous run serially, warp-shuffle scan across the threads.  off[n] = total.
__global__ void __launch_bounds__(1024) k_scan(const uint32_t* __restrict__ count, uint32_t n, uint32_t* __restrict__ off)
{
    __shared__ uint32_t warp_sums[32];
    const uint32_t tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const uint32_t per = (n + 1023) / 1024;
    const uint32_t begin = min(tid * per, n), end = min(begin + per, n);
    uint32_t sum = 0;
    for (uint32_t i = begin; i < end; ++i) sum += count[i];
    uint32_t incl = sum;
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= (uint32_t)o) incl += v;
    }
    if (lane == 31) warp_sums[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        uint32_t w = warp_sums[lane], wi = w;
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t v = __shfl_up_sync(0xFFFFFFFFu, wi, o);
            if (lane >= (uint32_t)o) wi += v;
        }
        warp_sums[lane] = wi - w;  // exclusive
    }
    __syncthreads();
    uint32_t run = warp_sums[wid] + incl - sum;
    for (uint32_t i = begin; i < end; ++i) {
        off[i] = run;
        run += count[i];
    }
    if (tid == 1023) off[n] = run;
}

cudaError_t vs_launch_bin_scan(const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    const uint32_t n = ch.views * fr.tiles_x * fr.tiles_y;
    k_scan<<<1, 1024, 0, st>>>(ch.tile_count, n, ch.tile_off);
    return cudaGetLastError();
}

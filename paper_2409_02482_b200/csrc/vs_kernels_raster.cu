// vs_kernels_raster.cu -- S4 coverage + per-layer nearest-fragment resolve.  DESIGN.md §1, §3.3-3.4, §7.
//
// One CTA per (view, 16x16 screen tile); its 8 warps walk the tile's triangle list independently
// (no CTA barrier inside the loop), 32 references at a time, in two lane mappings:
//   phase 1, lane = triangle: gather, integer setup, sample bounding box clipped to the tile.  A
//     triangle whose clipped box fits 4x4 samples ("small": ~all of them on the paper-shaped scenes,
//     ~6 px per triangle) gets its 16-bit coverage mask from three biased int32 edge functions stepped
//     with exact adds, and leaves a 12-word record in the warp's shared-memory slab.
//   phase 2, lane = covered sample: the warp's masks are compacted (shuffle scan of the popcounts,
//     every lane appends (lane, bit) codes to a queue) so that all 32 lanes evaluate one covered sample
//     each: fp32-exact depth key (IEEE division) and a 64-bit shared-memory max.  Only covered samples
//     pay for the division and the atomic, and they pay for it with full lanes.
//   large triangles (clipped box wider than 4 samples) are broadcast one at a time and the warp maps
//     its lanes to 8x4 pixel chunks of the box (int32 edges below 32 px of extent, else int64).
// The per-pixel, per-layer maximum key (float bits of 1/w << 32 | ~triangle id) lives in shared memory
// for all k layers of the tile at once and is written out as the triangle-id planes the shading
// kernel (and the parity tests) read.
#include "vs_common.cuh"
#include "vs_plain.cuh"

#define VS_RS_FIELDS 12                      // words per small-triangle record
#define VS_RS_QUEUE 512u                    // (lane, sample) codes per compaction round
#define VS_RS_WARP_WORDS (VS_RS_FIELDS * 32 + 256)  // + queue of 512 uint16 codes

__device__ __forceinline__ void vs_key_max(unsigned long long* slot, unsigned long long key)
{
    // 64-bit shared-memory max: the plain read doubles as the expected value of the first compare-and-swap
    unsigned long long old = *slot;
    while (key > old) {
        const unsigned long long assumed = old;
        old = atomicCAS(slot, assumed, key);
        if (old == assumed) break;
    }
}

__device__ __forceinline__ float vs_to_float(int v) { return __int2float_rn(v); }
__device__ __forceinline__ float vs_to_float(long long v) { return __ll2float_rn(v); }

// fp32-exact depth key of DESIGN.md §3.4 from the three (unbiased) edge values
__device__ __forceinline__ float vs_depth_from_edges(float f0, float f1, float f2, float q0, float q1, float q2, float fA)
{
    const float num = __fmaf_rn(f2, q2, __fmaf_rn(f1, q1, __fmul_rn(f0, q0)));
    return __fdiv_rn(num, fA);
}

// Large-triangle path: the whole warp, lane = pixel of an 8x4 chunk of the clipped box.
template <typename I>
__device__ __forceinline__ void vs_raster_large(int X0, int Y0, int X1, int Y1, int X2, int Y2, float q0, float q1, float q2,
                                                float fA, int i0, int i1, int j0, int j1, int px0, int py0,
                                                unsigned long long* __restrict__ kl, uint32_t lid, uint32_t lane)
{
    const int dx0 = X2 - X1, dy0 = Y2 - Y1, dx1 = X0 - X2, dy1 = Y0 - Y2, dx2 = X1 - X0, dy2 = Y1 - Y0;
    const int m0 = ((dy0 < 0) || (dy0 == 0 && dx0 > 0)) ? 0 : 1;
    const int m1 = ((dy1 < 0) || (dy1 == 0 && dx1 > 0)) ? 0 : 1;
    const int m2 = ((dy2 < 0) || (dy2 == 0 && dx2 > 0)) ? 0 : 1;
    for (int cj = j0; cj <= j1; cj += 4)
        for (int ci = i0; ci <= i1; ci += 8) {
            const int i = ci + (int)(lane & 7), j = cj + (int)(lane >> 3);
            if (i > i1 || j > j1) continue;
            const int Sx = 256 * i + 128, Sy = 256 * j + 128;
            const I e0 = (I)dx0 * (I)(Sy - Y1) - (I)dy0 * (I)(Sx - X1);
            const I e1 = (I)dx1 * (I)(Sy - Y2) - (I)dy1 * (I)(Sx - X2);
            const I e2 = (I)dx2 * (I)(Sy - Y0) - (I)dy2 * (I)(Sx - X0);
            if (e0 >= (I)m0 && e1 >= (I)m1 && e2 >= (I)m2) {
                const float qp = vs_depth_from_edges(vs_to_float(e0), vs_to_float(e1), vs_to_float(e2), q0, q1, q2, fA);
                vs_key_max(&kl[(j - py0) * VS_TILE_W + (i - px0)], vs_make_key(qp, lid));
            }
        }
}

__global__ void __launch_bounds__(256, 4)
k_raster(const VsSceneDev sc, const VsFrame fr, const int4* __restrict__ vtx, const uint32_t* __restrict__ tile_off,
         const uint32_t* __restrict__ tile_tris, uint32_t ref_capacity, uint32_t* __restrict__ ids, int fill_empty)
{
    extern __shared__ __align__(16) unsigned long long keys[];  // [k][256], then 8 warp slabs
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t tile = blockIdx.x, view = blockIdx.y;
    const uint32_t tiles = fr.tiles_x * fr.tiles_y;
    const int px0 = (int)(tile % fr.tiles_x) * VS_TILE_W, py0 = (int)(tile / fr.tiles_x) * VS_TILE_H;
    const int W = (int)fr.width, H = (int)fr.height;
    const uint32_t begin = min(tile_off[view * tiles + tile], ref_capacity), end = min(tile_off[view * tiles + tile + 1], ref_capacity);
    const int px = px0 + (int)(tid & 15), py = py0 + (int)(tid >> 4);
    const bool inimg = px < W && py < H;

    if (begin == end) {  // nothing binned here; the shading kernel does not read ids of empty tiles
        if (fill_empty && inimg)
            for (uint32_t l = 0; l < sc.k; ++l) ids[(((size_t)view * sc.k + l) * H + py) * W + px] = VS_MISS;
        return;
    }
    // the list is handed out 32 references at a time: the first two batches of a warp are fixed, the later ones
    // come from a shared counter so that the warps finish together
    __shared__ uint32_t s_next;
    for (uint32_t i = tid; i < sc.k * VS_TILE_PIX; i += 256) keys[i] = 0ull;
    if (tid == 0) s_next = begin + 512u;
    __syncthreads();

    int* rec = reinterpret_cast<int*>(keys + sc.k * VS_TILE_PIX) + warp * VS_RS_WARP_WORDS;  // [field][lane]
    unsigned short* queue = reinterpret_cast<unsigned short*>(rec + VS_RS_FIELDS * 32);       // [512]
    const int4* __restrict__ vv = vtx + (size_t)view * sc.v_total;
    const int tx1 = min(px0 + VS_TILE_W, W) - 1, ty1 = min(py0 + VS_TILE_H, H) - 1;

    // software pipeline over the gather chain tile_tris -> tris -> vertices: the reference of batch n+2 and the
    // index record of batch n+1 are in flight while batch n is rasterised
    uint32_t base = begin + warp * 32, base1 = base + 256u;
    uint32_t gt = base + lane < end ? __ldg(&tile_tris[base + lane]) : 0u;
    uint32_t gt1 = base1 + lane < end ? __ldg(&tile_tris[base1 + lane]) : 0u;
    uint4 tri = __ldg(&sc.tris[gt]);
    for (; base < end; ) {  // warp-uniform
        const uint32_t idx = base + lane;
        uint32_t base2 = 0;
        if (lane == 0) base2 = atomicAdd(&s_next, 32u);
        base2 = __shfl_sync(0xFFFFFFFFu, base2, 0);
        const uint32_t gt2 = base2 + lane < end ? __ldg(&tile_tris[base2 + lane]) : 0u;
        const uint4 tri1 = __ldg(&sc.tris[gt1]);
        // ---------------- phase 1: lane = triangle ----------------
        bool large = false;
        VsTri T;
        int i0 = 0, i1 = -1, j0 = 0, j1 = -1;
        uint32_t layer = 0, lid = 0;
        bool narrow = false, valid = false;
        if (idx < end) {
            const int4 a = __ldg(&vv[tri.x]), b = __ldg(&vv[tri.y]), c = __ldg(&vv[tri.z]);
            if (vs_setup_tri(a, b, c, T) == 0) {
                const int minX = min(T.X0, min(T.X1, T.X2)), maxX = max(T.X0, max(T.X1, T.X2));
                const int minY = min(T.Y0, min(T.Y1, T.Y2)), maxY = max(T.Y0, max(T.Y1, T.Y2));
                i0 = max((minX + 127) >> 8, px0); i1 = min((maxX - 128) >> 8, tx1);
                j0 = max((minY + 127) >> 8, py0); j1 = min((maxY - 128) >> 8, ty1);
                layer = vs_tri_layer(tri.w); lid = vs_tri_lid(tri.w);
                narrow = maxX - minX < 8192 && maxY - minY < 8192;  // every int32 intermediate < 2^28
                valid = i0 <= i1 && j0 <= j1;
                large = valid && !(narrow && i1 - i0 < 8 && j1 - j0 < 8);
            }
        }
        uint32_t mlo = 0, mhi = 0;  // coverage of the clipped box, sample (r, c) -> bit 8r + c of mhi:mlo
        int E0 = 0, E1 = 0, E2 = 0, sx0 = 0, sx1 = 0, sx2 = 0, sy0 = 0, sy1 = 0, sy2 = 0;
        const bool small = valid && !large;
        if (small) {
            // edge e_i runs (i+1) -> (i+2) and weights vertex i; sample (i0, j0)
            const int dx0 = T.X2 - T.X1, dy0 = T.Y2 - T.Y1, dx1 = T.X0 - T.X2, dy1 = T.Y0 - T.Y2;
            const int dx2 = T.X1 - T.X0, dy2 = T.Y1 - T.Y0;
            const int Sx = 256 * i0 + 128, Sy = 256 * j0 + 128;
            E0 = dx0 * (Sy - T.Y1) - dy0 * (Sx - T.X1);
            E1 = dx1 * (Sy - T.Y2) - dy1 * (Sx - T.X2);
            E2 = dx2 * (Sy - T.Y0) - dy2 * (Sx - T.X0);
            sx0 = -256 * dy0; sx1 = -256 * dy1; sx2 = -256 * dy2;  // one pixel in +x
            sy0 = 256 * dx0; sy1 = 256 * dx1; sy2 = 256 * dx2;     // one pixel in +y
            rec[0 * 32 + lane] = E0; rec[1 * 32 + lane] = E1;
            rec[2 * 32 + lane] = sx0; rec[3 * 32 + lane] = sx1;
            rec[4 * 32 + lane] = sy0; rec[5 * 32 + lane] = sy1;
            rec[6 * 32 + lane] = (int)T.A2;
            rec[7 * 32 + lane] = __float_as_int(T.q0); rec[8 * 32 + lane] = __float_as_int(T.q1);
            rec[9 * 32 + lane] = __float_as_int(T.q2);
            rec[10 * 32 + lane] = (int)lid;
            rec[11 * 32 + lane] = (int)(layer * VS_TILE_PIX) + (j0 - py0) * VS_TILE_W + (i0 - px0);
            // covered <=> E_e > 0 || (E_e == 0 && topleft_e) <=> F_e := E_e - (topleft_e ? 0 : 1) >= 0
            E0 -= ((dy0 < 0) || (dy0 == 0 && dx0 > 0)) ? 0 : 1;
            E1 -= ((dy1 < 0) || (dy1 == 0 && dx1 > 0)) ? 0 : 1;
            E2 -= ((dy2 < 0) || (dy2 == 0 && dx2 > 0)) ? 0 : 1;
        }
        const int nr = small ? j1 - j0 + 1 : 0, nc = small ? i1 - i0 + 1 : 0;
        {
            // rows of up to 8 samples, row and column counts uniform over the warp (the lanes' boxes are alike);
            // samples of a row are visited from column cols-1 down to 0 so that each funnel shift pushes the next lower bit
            const int rows = __reduce_max_sync(0xFFFFFFFFu, nr);
            const int cols = __reduce_max_sync(0xFFFFFFFFu, nc);  // columns >= cols are masked off below for every lane
            int a0 = E0 + (cols - 1) * sx0, a1 = E1 + (cols - 1) * sx1, a2 = E2 + (cols - 1) * sx2;
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                if (r < rows) {
                    uint32_t bits = 0;
                    int c0 = a0, c1 = a1, c2 = a2;
#pragma unroll
                    for (int c = 7; c >= 0; --c) {
                        if (c < cols) {  // warp-uniform
                            bits = __funnelshift_l((uint32_t)(c0 | c1 | c2), bits, 1);
                            c0 -= sx0; c1 -= sx1; c2 -= sx2;
                        }
                    }
                    bits = ~bits & 0xFFu;
                    if (r < 4) mlo |= bits << (8 * r); else mhi |= bits << (8 * (r - 4));
                    a0 += sy0; a1 += sy1; a2 += sy2;
                }
            }
            const uint32_t colm = 0x01010101u * ((1u << nc) - 1u);
            mlo &= colm & (nr >= 4 ? 0xFFFFFFFFu : ((1u << (8 * nr)) - 1u));
            mhi &= colm & (nr >= 8 ? 0xFFFFFFFFu : (nr > 4 ? ((1u << (8 * (nr - 4))) - 1u) : 0u));
        }
        // ---------------- compaction: (lane, bit) codes of the covered samples ----------------
        const uint32_t cnt = (uint32_t)(__popc(mlo) + __popc(mhi));
        uint32_t incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, incl, o);
            if (lane >= (uint32_t)o) incl += u;
        }
        const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31);
        for (uint32_t win = 0; win < total; win += VS_RS_QUEUE) {  // one round unless the warp covers > 512 samples
            {
                uint32_t off = incl - cnt - win;  // wraps for codes in front of the window: fails the bound test
                uint32_t m = mlo;
                while (m) {
                    const int bit = __ffs(m) - 1;
                    m &= m - 1;
                    if (off < VS_RS_QUEUE) queue[off] = (unsigned short)((lane << 6) | (uint32_t)bit);
                    ++off;
                }
                m = mhi;
                while (m) {
                    const int bit = __ffs(m) - 1;
                    m &= m - 1;
                    if (off < VS_RS_QUEUE) queue[off] = (unsigned short)((lane << 6) | 32u | (uint32_t)bit);
                    ++off;
                }
            }
            __syncwarp();
            // ---------------- phase 2: lane = covered sample ----------------
            const uint32_t n = min(total - win, (uint32_t)VS_RS_QUEUE);
            for (uint32_t s = lane; s < n; s += 32) {
                const uint32_t code = queue[s];
                const uint32_t src = code >> 6;
                const int r = (int)((code >> 3) & 7u), c = (int)(code & 7u);
                const int e0 = rec[0 * 32 + src] + r * rec[4 * 32 + src] + c * rec[2 * 32 + src];
                const int e1 = rec[1 * 32 + src] + r * rec[5 * 32 + src] + c * rec[3 * 32 + src];
                const int A2 = rec[6 * 32 + src];
                const int e2 = A2 - e0 - e1;  // E0 + E1 + E2 == A2 at every point
                const float qp = vs_depth_from_edges(__int2float_rn(e0), __int2float_rn(e1), __int2float_rn(e2),
                                                     __int_as_float(rec[7 * 32 + src]), __int_as_float(rec[8 * 32 + src]),
                                                     __int_as_float(rec[9 * 32 + src]), __int2float_rn(A2));
                vs_key_max(&keys[rec[11 * 32 + src] + r * VS_TILE_W + c], vs_make_key(qp, (uint32_t)rec[10 * 32 + src]));
            }
            __syncwarp();
        }
        // ---------------- large triangles: lane = pixel of an 8x4 chunk ----------------
        uint32_t lm = __ballot_sync(0xFFFFFFFFu, large);
        while (lm) {
            const int src = __ffs(lm) - 1;
            lm &= lm - 1;
            const int X0 = __shfl_sync(0xFFFFFFFFu, T.X0, src), Y0 = __shfl_sync(0xFFFFFFFFu, T.Y0, src);
            const int X1 = __shfl_sync(0xFFFFFFFFu, T.X1, src), Y1 = __shfl_sync(0xFFFFFFFFu, T.Y1, src);
            const int X2 = __shfl_sync(0xFFFFFFFFu, T.X2, src), Y2 = __shfl_sync(0xFFFFFFFFu, T.Y2, src);
            const float q0 = __shfl_sync(0xFFFFFFFFu, T.q0, src), q1 = __shfl_sync(0xFFFFFFFFu, T.q1, src);
            const float q2 = __shfl_sync(0xFFFFFFFFu, T.q2, src);
            const long long A2 = __shfl_sync(0xFFFFFFFFu, T.A2, src);
            const int bi0 = __shfl_sync(0xFFFFFFFFu, i0, src), bi1 = __shfl_sync(0xFFFFFFFFu, i1, src);
            const int bj0 = __shfl_sync(0xFFFFFFFFu, j0, src), bj1 = __shfl_sync(0xFFFFFFFFu, j1, src);
            const uint32_t blid = __shfl_sync(0xFFFFFFFFu, lid, src), blayer = __shfl_sync(0xFFFFFFFFu, layer, src);
            const bool bnarrow = __shfl_sync(0xFFFFFFFFu, (int)narrow, src) != 0;
            unsigned long long* kl = keys + blayer * VS_TILE_PIX;
            if (bnarrow) vs_raster_large<int>(X0, Y0, X1, Y1, X2, Y2, q0, q1, q2, __ll2float_rn(A2), bi0, bi1, bj0, bj1, px0, py0, kl, blid, lane);
            else vs_raster_large<long long>(X0, Y0, X1, Y1, X2, Y2, q0, q1, q2, __ll2float_rn(A2), bi0, bi1, bj0, bj1, px0, py0, kl, blid, lane);
        }
        __syncwarp();  // the slab is rewritten by the next batch
        base = base1; gt = gt1; tri = tri1;
        base1 = base2; gt1 = gt2;
    }
    __syncthreads();

    if (inimg)
        for (uint32_t l = 0; l < sc.k; ++l) {
            const unsigned long long key = keys[l * VS_TILE_PIX + tid];
            ids[(((size_t)view * sc.k + l) * H + py) * W + px] = key ? 0xFFFFFFFFu - (uint32_t)key : VS_MISS;
        }
}

cudaError_t vs_launch_raster(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    const size_t smem = (size_t)sc.k * VS_TILE_PIX * 8 + 8 * VS_RS_WARP_WORDS * 4;
    dim3 grid(fr.tiles_x * fr.tiles_y, ch.views);
    k_raster<<<grid, 256, smem, st>>>(sc, fr, ch.vtx, ch.tile_off, ch.tile_tris, ch.ref_capacity, ch.ids, ch.ids_is_output);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// VS_FLAG_REFERENCE_PATH: brute force, one thread per pixel, every triangle of every layer tested.
// Same arithmetic contract, no binning, no cooperation -- a debugging aid for small scenes.
// ------------------------------------------------------------------------------------------------
template <int F16>
__global__ void __launch_bounds__(128)
k_reference(const VsSceneDev sc, const VsFrame fr, const VsCamDev* __restrict__ cams, const int4* __restrict__ vtx,
            float* __restrict__ out_rgba, uint32_t* __restrict__ out_ids)
{
    const int W = (int)fr.width, H = (int)fr.height;
    const int px = blockIdx.x * 16 + (threadIdx.x & 15), py = blockIdx.y * 8 + (threadIdx.x >> 4);
    const uint32_t view = blockIdx.z;
    if (px >= W || py >= H) return;
    const int4* __restrict__ vv = vtx + (size_t)view * sc.v_total;
    float Y[VS_MAX_COEF];
    float vx, vy, vz;
    vs_view_dir(cams[view], px, py, vx, vy, vz);
    vs_sh_basis<3>(vx, vy, vz, Y);
    float Tr = 1.0f, C[3] = {0.0f, 0.0f, 0.0f};
    bool alive = true;
    for (uint32_t l = 0; l < sc.k; ++l) {
        unsigned long long best = 0ull;
        for (uint32_t gt = sc.tri_off[l]; gt < sc.tri_off[l + 1]; ++gt) {
            const uint4 tri = sc.tris[gt];
            VsTri T;
            if (vs_setup_tri(vv[tri.x], vv[tri.y], vv[tri.z], T) != 0) continue;
            int m0, m1, m2;
            vs_edge_mins(T, m0, m1, m2);
            VsEdges e;
            vs_edges_at(T, px, py, e);
            if (e.E0 >= m0 && e.E1 >= m1 && e.E2 >= m2) {
                const unsigned long long key = vs_make_key(vs_depth_q(T, e.E0, e.E1, e.E2), gt - sc.tri_off[l]);
                if (key > best) best = key;
            }
        }
        const bool hit = best != 0ull;
        const uint32_t lid = 0xFFFFFFFFu - (uint32_t)best;
        if (out_ids) out_ids[(((size_t)view * sc.k + l) * H + py) * W + px] = hit ? lid : VS_MISS;
        if (!hit || !alive) continue;
        float s[4], uv[2];
        vs_plain_logits<F16>(sc, vv, l, lid, px, py, Y, s, uv);
        float A = vs_sigmoid(s[3]);
        if (fr.attenuate) A *= vs_alpha_w(vx, vy, vz, vs_fragment_normal(sc, vv, l, lid, px, py));
        for (int ch = 0; ch < 3; ++ch) C[ch] += Tr * A * vs_sigmoid(s[ch]);
        Tr *= (1.0f - A);
        if (Tr < fr.t_min) alive = false;
    }
    reinterpret_cast<float4*>(out_rgba)[((size_t)view * H + py) * W + px] =
        make_float4(C[0] + Tr * fr.bg[0], C[1] + Tr * fr.bg[1], C[2] + Tr * fr.bg[2], 1.0f - Tr);
}

cudaError_t vs_launch_reference(const VsSceneDev& sc, int f16, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    dim3 grid((fr.width + 15) / 16, (fr.height + 7) / 8, ch.views);
    uint32_t* ids = ch.ids_is_output ? ch.ids : nullptr;
    if (f16) k_reference<1><<<grid, 128, 0, st>>>(sc, fr, ch.cams, ch.vtx, ch.out_rgba, ids);
    else k_reference<0><<<grid, 128, 0, st>>>(sc, fr, ch.cams, ch.vtx, ch.out_rgba, ids);
    return cudaGetLastError();
}

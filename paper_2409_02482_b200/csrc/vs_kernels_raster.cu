// vs_kernels_raster.cu -- S4 coverage + per-layer nearest-fragment resolve.  DESIGN.md §1, §3.3-3.4, §7.
//
// One CTA per (view, 16x16 screen tile); one thread per binned triangle.  A thread walks the
// triangle's sample bounding box inside the tile in 4x4 blocks: the three biased edge functions are
// stepped with exact integer adds and their sign bits funnel-shifted into a 16-bit coverage mask
// (5 integer instructions per sample, no branches), so only covered samples pay for the fp32 depth
// key and the shared-memory 64-bit max.  Triangles whose extent is < 32 px run this in int32 (every
// intermediate is < 2^28, i.e. the same integers as the int64 definition); larger ones in int64.
// The per-pixel, per-layer maximum key (float bits of 1/w << 32 | ~triangle id) lives in shared memory
// for all k layers of the tile at once and is written out as the triangle-id planes the shading
// kernel (and the parity tests) read.
#include "vs_common.cuh"

__device__ __forceinline__ void vs_key_max(unsigned long long* slot, unsigned long long key)
{
    if (key > *slot) atomicMax(slot, key);
}

__device__ __forceinline__ int vs_sign_word(int v) { return v; }
__device__ __forceinline__ int vs_sign_word(long long v) { return (int)(v >> 32); }
__device__ __forceinline__ float vs_to_float(int v) { return __int2float_rn(v); }
__device__ __forceinline__ float vs_to_float(long long v) { return __ll2float_rn(v); }

// Rasterise one set-up triangle over pixels [i0,i1] x [j0,j1] (already clipped to the tile and the
// image) into the tile's key plane `kl`.  I = int (small triangles) or long long.
template <typename I>
__device__ __forceinline__ void vs_raster_tri(const VsTri& T, int i0, int i1, int j0, int j1, int px0, int py0,
                                              unsigned long long* __restrict__ kl, uint32_t lid)
{
    // edge e_i runs (i+1) -> (i+2) and weights vertex i
    const int dx0 = T.X2 - T.X1, dy0 = T.Y2 - T.Y1;
    const int dx1 = T.X0 - T.X2, dy1 = T.Y0 - T.Y2;
    const int dx2 = T.X1 - T.X0, dy2 = T.Y1 - T.Y0;
    // covered <=> E_e > 0 || (E_e == 0 && topleft_e) <=> F_e := E_e - (topleft_e ? 0 : 1) >= 0
    const int m0 = ((dy0 < 0) || (dy0 == 0 && dx0 > 0)) ? 0 : 1;
    const int m1 = ((dy1 < 0) || (dy1 == 0 && dx1 > 0)) ? 0 : 1;
    const int m2 = ((dy2 < 0) || (dy2 == 0 && dx2 > 0)) ? 0 : 1;
    const int Sx = 256 * i0 + 128, Sy = 256 * j0 + 128;
    I f0 = (I)dx0 * (I)(Sy - T.Y1) - (I)dy0 * (I)(Sx - T.X1) - (I)m0;
    I f1 = (I)dx1 * (I)(Sy - T.Y2) - (I)dy1 * (I)(Sx - T.X2) - (I)m1;
    I f2 = (I)dx2 * (I)(Sy - T.Y0) - (I)dy2 * (I)(Sx - T.X0) - (I)m2;
    const I sx0 = -(I)256 * (I)dy0, sx1 = -(I)256 * (I)dy1, sx2 = -(I)256 * (I)dy2;  // one pixel in +x
    const I sy0 = (I)256 * (I)dx0, sy1 = (I)256 * (I)dx1, sy2 = (I)256 * (I)dx2;     // one pixel in +y
    const float fA = vs_to_float((I)T.A2);
    for (int bj = j0; bj <= j1; bj += 4) {
        I r0 = f0, r1 = f1, r2 = f2;
        const int nr = min(4, j1 - bj + 1);
        for (int bi = i0; bi <= i1; bi += 4) {
            // coverage mask of the 4x4 block at (bi, bj): sample (r, c) -> bit 4r + c.  Samples are
            // visited from (3,3) down to (0,0) so that each funnel shift pushes the next lower bit.
            uint32_t bits = 0;
            I a0 = r0 + 3 * sy0 + 3 * sx0, a1 = r1 + 3 * sy1 + 3 * sx1, a2 = r2 + 3 * sy2 + 3 * sx2;
#pragma unroll
            for (int r = 3; r >= 0; --r) {
                I c0 = a0, c1 = a1, c2 = a2;
#pragma unroll
                for (int c = 3; c >= 0; --c) {
                    bits = __funnelshift_l((uint32_t)vs_sign_word(c0 | c1 | c2), bits, 1);
                    c0 -= sx0; c1 -= sx1; c2 -= sx2;
                }
                a0 -= sy0; a1 -= sy1; a2 -= sy2;
            }
            const int nc = min(4, i1 - bi + 1);
            uint32_t cov = ~bits & (0x1111u * ((1u << nc) - 1u)) & ((1u << (4 * nr)) - 1u);
            while (cov) {
                const int bit = __ffs(cov) - 1;
                cov &= cov - 1;
                const int r = bit >> 2, c = bit & 3;
                const I e0 = r0 + (I)r * sy0 + (I)c * sx0 + (I)m0;
                const I e1 = r1 + (I)r * sy1 + (I)c * sx1 + (I)m1;
                const I e2 = r2 + (I)r * sy2 + (I)c * sx2 + (I)m2;
                // depth key, fp32-exact
                const float num = __fmaf_rn(vs_to_float(e2), T.q2, __fmaf_rn(vs_to_float(e1), T.q1, __fmul_rn(vs_to_float(e0), T.q0)));
                const float qp = __fdiv_rn(num, fA);
                vs_key_max(&kl[(bj + r - py0) * VS_TILE_W + (bi + c - px0)], vs_make_key(qp, lid));
            }
            r0 += 4 * sx0; r1 += 4 * sx1; r2 += 4 * sx2;
        }
        f0 += 4 * sy0; f1 += 4 * sy1; f2 += 4 * sy2;
    }
}

__global__ void __launch_bounds__(256, 4)
k_raster(const VsSceneDev sc, const VsFrame fr, const int4* __restrict__ vtx, const uint32_t* __restrict__ tile_off,
         const uint32_t* __restrict__ tile_tris, uint32_t ref_capacity, uint32_t* __restrict__ ids, int fill_empty)
{
    extern __shared__ __align__(16) unsigned long long keys[];  // [k][256]
    const uint32_t tid = threadIdx.x;
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
    for (uint32_t i = tid; i < sc.k * VS_TILE_PIX; i += 256) keys[i] = 0ull;
    __syncthreads();

    const int4* __restrict__ vv = vtx + (size_t)view * sc.v_total;
    const int tx1 = min(px0 + VS_TILE_W, W) - 1, ty1 = min(py0 + VS_TILE_H, H) - 1;
    for (uint32_t idx = begin + tid; idx < end; idx += 256) {
        const uint32_t gt = __ldg(&tile_tris[idx]);
        const uint4 tri = __ldg(&sc.tris[gt]);
        const int4 a = __ldg(&vv[tri.x]), b = __ldg(&vv[tri.y]), c = __ldg(&vv[tri.z]);
        VsTri T;
        if (vs_setup_tri(a, b, c, T) != 0) continue;
        const int minX = min(T.X0, min(T.X1, T.X2)), maxX = max(T.X0, max(T.X1, T.X2));
        const int minY = min(T.Y0, min(T.Y1, T.Y2)), maxY = max(T.Y0, max(T.Y1, T.Y2));
        const int i0 = max((minX + 127) >> 8, px0), i1 = min((maxX - 128) >> 8, tx1);
        const int j0 = max((minY + 127) >> 8, py0), j1 = min((maxY - 128) >> 8, ty1);
        if (i0 > i1 || j0 > j1) continue;
        const uint32_t layer = tri.w, lid = gt - sc.tri_off[layer];
        unsigned long long* kl = keys + layer * VS_TILE_PIX;
        if (maxX - minX < 8192 && maxY - minY < 8192) vs_raster_tri<int>(T, i0, i1, j0, j1, px0, py0, kl, lid);
        else vs_raster_tri<long long>(T, i0, i1, j0, j1, px0, py0, kl, lid);
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
    const size_t smem = (size_t)sc.k * VS_TILE_PIX * 8;
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
        VsFrag f;
        vs_fragment_setup(sc, vv, l, lid, px, py, f);
        const uint32_t Wt = sc.tex_w[l], nv = sc.texel_vecs;
        const uint32_t offs[4] = {(f.cy0 * Wt + f.cx0) * nv, (f.cy0 * Wt + f.cx1) * nv, (f.cy1 * Wt + f.cx0) * nv, (f.cy1 * Wt + f.cx1) * nv};
        const float ws[4] = {(1.0f - f.a) * (1.0f - f.b), f.a * (1.0f - f.b), (1.0f - f.a) * f.b, f.a * f.b};
        float s[4] = {0.0f, 0.0f, 0.0f, 0.0f};
        for (uint32_t c = 0; c < sc.n_coef; ++c)
            for (int ch = 0; ch < 4; ++ch) {
                float v = 0.0f;
                for (int q = 0; q < 4; ++q) {
                    float tv;
                    if (F16) tv = __half2float(reinterpret_cast<const __half*>(sc.tex[l] + offs[q])[ch * sc.np_pad + c]);
                    else tv = reinterpret_cast<const float*>(sc.tex[l] + offs[q])[ch * sc.np_pad + c];
                    v += ws[q] * tv;
                }
                s[ch] += Y[c] * v;
            }
        const float A = vs_sigmoid(s[3]);
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

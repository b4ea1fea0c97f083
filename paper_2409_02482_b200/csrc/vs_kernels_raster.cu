// vs_kernels_raster.cu -- S4 coverage + per-layer nearest-fragment resolve, fused with S5 UV
// interpolation + bilinear texel fetch, S6 SH evaluation + sigmoid and S7 fixed-order compositing.
// One CTA per (view, 16x16 screen tile).  DESIGN.md §1, §3.3-3.8, §7.
//
// Phase 1 (raster): one thread per binned triangle walks the triangle's sample bounding box inside
//   the tile with exact integer edge functions and keeps, per pixel and per layer, the maximum
//   64-bit key (float bits of 1/w << 32 | ~triangle id) in shared memory.  Triangles whose box
//   inside the tile exceeds VS_BIG_PIXELS samples are queued and rasterised by a whole warp.
// Phase 2 (shade): a warp owns an 8x4 pixel block.  "Owner" lanes (lane = pixel) turn the winning
//   triangle of a layer into 4 texel offsets + 4 bilinear weights; then the warp re-maps itself to
//   4 fragments x 8 lanes: each octet streams one fragment's four texels as 16-byte vectors (one
//   full 128-byte line per octet per texel at SH degree 3 / fp16), blends, dots with the pixel's SH
//   basis (held in registers for all layers) and hands 4 partial channel sums back through shared
//   memory.  Owners add the partials, apply the sigmoid and composite front to back.
#include "vs_common.cuh"

#define VS_BIG_PIXELS 32

struct __align__(16) VsFragRec {
    uint32_t o00, o01, o10, o11;  // 16-byte-vector offsets of the four texels inside the layer texture
    float w00, w01, w10, w11;     // bilinear weights
};

__device__ __forceinline__ void vs_key_max(unsigned long long* slot, unsigned long long key)
{
    if (key > *slot) atomicMax(slot, key);
}

// Owner-side fragment setup: winning triangle of layer l at pixel (px,py) -> texel offsets + weights.
__device__ __forceinline__ void vs_fragment_record(const VsSceneDev& sc, const int4* __restrict__ vv, uint32_t l,
                                                   uint32_t local_tri, int px, int py, VsFragRec& r)
{
    const uint4 tri = __ldg(&sc.tris[sc.tri_off[l] + local_tri]);
    const int4 a = __ldg(&vv[tri.x]), b = __ldg(&vv[tri.y]), c = __ldg(&vv[tri.z]);
    VsTri T;
    vs_setup_tri(a, b, c, T);
    const uint32_t i1 = T.swapped ? tri.z : tri.y, i2 = T.swapped ? tri.y : tri.z;
    const float2 uv0 = __ldg(&sc.uvs[tri.x]), uv1 = __ldg(&sc.uvs[i1]), uv2 = __ldg(&sc.uvs[i2]);
    VsEdges e;
    vs_edges_at(T, px, py, e);
    // perspective-correct barycentrics b'_i ~ E_i q_i
    const float g0 = __ll2float_rn(e.E0) * T.q0, g1 = __ll2float_rn(e.E1) * T.q1, g2 = __ll2float_rn(e.E2) * T.q2;
    const float inv = __fdividef(1.0f, g0 + g1 + g2);
    const float b1 = g1 * inv, b2 = g2 * inv;
    const int Wt = (int)sc.tex_w[l], Ht = (int)sc.tex_h[l];
    const float fW = (float)Wt, fH = (float)Ht;
    // texel coordinate = (u0 W - 0.5) + (b1 du1 + b2 du2) W, carried as integer + fraction so that
    // the fraction keeps full fp32 resolution at 4096^2
    float ph = __fmul_rn(uv0.x, fW), pl = __fmaf_rn(uv0.x, fW, -ph);
    float x0 = fminf(fmaxf(ph - 0.5f, -1048576.0f), 1048576.0f);
    float fl = floorf(x0);
    float t = ((x0 - fl) + pl) + (b1 * (uv1.x - uv0.x) + b2 * (uv2.x - uv0.x)) * fW;
    float ft = floorf(t);
    const float aa = t - ft;
    const int ix0 = __float2int_rd(fl) + __float2int_rd(ft);
    ph = __fmul_rn(uv0.y, fH); pl = __fmaf_rn(uv0.y, fH, -ph);
    x0 = fminf(fmaxf(ph - 0.5f, -1048576.0f), 1048576.0f);
    fl = floorf(x0);
    t = ((x0 - fl) + pl) + (b1 * (uv1.y - uv0.y) + b2 * (uv2.y - uv0.y)) * fH;
    ft = floorf(t);
    const float bb = t - ft;
    const int iy0 = __float2int_rd(fl) + __float2int_rd(ft);
    const uint32_t cx0 = (uint32_t)min(max(ix0, 0), Wt - 1), cx1 = (uint32_t)min(max(ix0 + 1, 0), Wt - 1);
    const uint32_t cy0 = (uint32_t)min(max(iy0, 0), Ht - 1), cy1 = (uint32_t)min(max(iy0 + 1, 0), Ht - 1);
    const uint32_t nv = sc.texel_vecs;
    r.o00 = (cy0 * (uint32_t)Wt + cx0) * nv; r.o01 = (cy0 * (uint32_t)Wt + cx1) * nv;
    r.o10 = (cy1 * (uint32_t)Wt + cx0) * nv; r.o11 = (cy1 * (uint32_t)Wt + cx1) * nv;
    r.w00 = (1.0f - aa) * (1.0f - bb); r.w01 = aa * (1.0f - bb);
    r.w10 = (1.0f - aa) * bb;          r.w11 = aa * bb;
}

template <int F16>
__device__ __forceinline__ void vs_accumulate_vec(const uint4& t00, const uint4& t01, const uint4& t10, const uint4& t11,
                                                  const float4& w, const float* Y, float4& acc)
{
    if (F16) {
        const __half2* h00 = reinterpret_cast<const __half2*>(&t00);
        const __half2* h01 = reinterpret_cast<const __half2*>(&t01);
        const __half2* h10 = reinterpret_cast<const __half2*>(&t10);
        const __half2* h11 = reinterpret_cast<const __half2*>(&t11);
        float v[8];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const float2 a = __half22float2(h00[q]), b = __half22float2(h01[q]);
            const float2 c = __half22float2(h10[q]), d = __half22float2(h11[q]);
            v[2 * q] = w.x * a.x + w.y * b.x + w.z * c.x + w.w * d.x;
            v[2 * q + 1] = w.x * a.y + w.y * b.y + w.z * c.y + w.w * d.y;
        }
        acc.x += Y[0] * v[0] + Y[1] * v[4];
        acc.y += Y[0] * v[1] + Y[1] * v[5];
        acc.z += Y[0] * v[2] + Y[1] * v[6];
        acc.w += Y[0] * v[3] + Y[1] * v[7];
    } else {
        const float4 a = *reinterpret_cast<const float4*>(&t00), b = *reinterpret_cast<const float4*>(&t01);
        const float4 c = *reinterpret_cast<const float4*>(&t10), d = *reinterpret_cast<const float4*>(&t11);
        acc.x += Y[0] * (w.x * a.x + w.y * b.x + w.z * c.x + w.w * d.x);
        acc.y += Y[0] * (w.x * a.y + w.y * b.y + w.z * c.y + w.w * d.y);
        acc.z += Y[0] * (w.x * a.z + w.y * b.z + w.z * c.z + w.w * d.z);
        acc.w += Y[0] * (w.x * a.w + w.y * b.w + w.z * c.w + w.w * d.w);
    }
}

template <int F16, int DEG, bool COUNT>
__global__ void __launch_bounds__(256, 2)
k_raster_shade(const VsSceneDev sc, const VsFrame fr, const VsCamDev* __restrict__ cams, const int4* __restrict__ vtx,
               const uint32_t* __restrict__ tile_off, const uint32_t* __restrict__ tile_tris,
               float* __restrict__ out_rgba, uint32_t* __restrict__ out_ids, uint32_t* __restrict__ texel_bits,
               unsigned long long* __restrict__ counters)
{
    constexpr int NCOEF = (DEG + 1) * (DEG + 1);
    constexpr int CPV = F16 ? 2 : 1;                 // coefficients per 16-byte vector
    constexpr int NVEC = (NCOEF + CPV - 1) / CPV;    // vectors per texel (== sc.texel_vecs)
    constexpr int SLOTS = (NVEC + 7) / 8;            // vectors per octet lane
    constexpr int NACT = NVEC < 8 ? NVEC : 8;        // octet lanes that hold data
    constexpr int YROW = SLOTS * 8 * CPV;            // floats per pixel in the Y staging buffer

    extern __shared__ __align__(16) unsigned char smem[];
    unsigned long long* keys = reinterpret_cast<unsigned long long*>(smem);               // [k][256]
    VsFragRec* rec_all = reinterpret_cast<VsFragRec*>(smem + (size_t)sc.k * VS_TILE_PIX * 8);  // [8][32]
    float4* part_all = reinterpret_cast<float4*>(reinterpret_cast<unsigned char*>(rec_all) + 8 * 32 * sizeof(VsFragRec));  // [8][32][8]
    __shared__ uint32_t bigq[256];
    __shared__ uint32_t bigcount;

    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t tile = blockIdx.x, view = blockIdx.y;
    const uint32_t tiles = fr.tiles_x * fr.tiles_y;
    const int px0 = (int)(tile % fr.tiles_x) * VS_TILE_W, py0 = (int)(tile / fr.tiles_x) * VS_TILE_H;
    const int W = (int)fr.width, H = (int)fr.height;
    const uint32_t begin = tile_off[view * tiles + tile], end = tile_off[view * tiles + tile + 1];
    const int4* __restrict__ vv = vtx + (size_t)view * sc.v_total;

    // this thread's pixel in phase 2: warp -> 8x4 block, lane -> pixel
    const int lx = (int)(warp & 1) * 8 + (int)(lane & 7), ly = (int)(warp >> 1) * 4 + (int)(lane >> 3);
    const int px = px0 + lx, py = py0 + ly;
    const bool inimg = px < W && py < H;
    const int pl = ly * VS_TILE_W + lx;

    if (begin == end) {  // nothing binned here: background
        if (inimg) {
            reinterpret_cast<float4*>(out_rgba)[((size_t)view * H + py) * W + px] = make_float4(fr.bg[0], fr.bg[1], fr.bg[2], 0.0f);
            if (out_ids)
                for (uint32_t l = 0; l < sc.k; ++l) out_ids[(((size_t)view * sc.k + l) * H + py) * W + px] = VS_MISS;
        }
        return;
    }

    for (uint32_t i = tid; i < sc.k * VS_TILE_PIX; i += 256) keys[i] = 0ull;
    if (tid == 0) bigcount = 0;
    __syncthreads();

    // ---------------- phase 1: coverage + nearest-fragment resolve ----------------
    const int tx1 = min(px0 + VS_TILE_W, W) - 1, ty1 = min(py0 + VS_TILE_H, H) - 1;
    for (uint32_t base = begin; base < end; base += 256) {
        const uint32_t idx = base + tid;
        bool pushed = false;
        if (idx < end) {
            const uint32_t gt = __ldg(&tile_tris[idx]);
            const uint4 tri = __ldg(&sc.tris[gt]);
            const int4 a = __ldg(&vv[tri.x]), b = __ldg(&vv[tri.y]), c = __ldg(&vv[tri.z]);
            VsTri T;
            int i0, i1, j0, j1;
            if (vs_setup_tri(a, b, c, T) == 0 && vs_tri_pixel_bbox(T, W, H, i0, i1, j0, j1)) {
                i0 = max(i0, px0); i1 = min(i1, tx1); j0 = max(j0, py0); j1 = min(j1, ty1);
                if (i0 <= i1 && j0 <= j1) {
                    if ((i1 - i0 + 1) * (j1 - j0 + 1) > VS_BIG_PIXELS) {
                        bigq[atomicAdd(&bigcount, 1u)] = gt;
                        pushed = true;
                    } else {
                        const uint32_t layer = tri.w, lid = gt - sc.tri_off[layer];
                        unsigned long long* kl = keys + layer * VS_TILE_PIX;
                        int m0, m1, m2;
                        vs_edge_mins(T, m0, m1, m2);
                        VsEdges e;
                        vs_edges_at(T, i0, j0, e);
                        const long long sx0 = -256ll * (T.Y2 - T.Y1), sx1 = -256ll * (T.Y0 - T.Y2), sx2 = -256ll * (T.Y1 - T.Y0);
                        const long long sy0 = 256ll * (T.X2 - T.X1), sy1 = 256ll * (T.X0 - T.X2), sy2 = 256ll * (T.X1 - T.X0);
                        for (int j = j0; j <= j1; ++j) {
                            long long e0 = e.E0, e1 = e.E1, e2 = e.E2;
                            for (int i = i0; i <= i1; ++i) {
                                if (e0 >= m0 && e1 >= m1 && e2 >= m2)
                                    vs_key_max(&kl[(j - py0) * VS_TILE_W + (i - px0)], vs_make_key(vs_depth_q(T, e0, e1, e2), lid));
                                e0 += sx0; e1 += sx1; e2 += sx2;
                            }
                            e.E0 += sy0; e.E1 += sy1; e.E2 += sy2;
                        }
                    }
                }
            }
        }
        if (__syncthreads_or(pushed)) {
            // large triangles: one warp each, lanes over the samples of the clipped box
            const uint32_t nbig = bigcount;
            for (uint32_t q = warp; q < nbig; q += 8) {
                const uint32_t gt = bigq[q];
                const uint4 tri = __ldg(&sc.tris[gt]);
                const int4 a = __ldg(&vv[tri.x]), b = __ldg(&vv[tri.y]), c = __ldg(&vv[tri.z]);
                VsTri T;
                int i0, i1, j0, j1;
                vs_setup_tri(a, b, c, T);
                vs_tri_pixel_bbox(T, W, H, i0, i1, j0, j1);
                i0 = max(i0, px0); i1 = min(i1, tx1); j0 = max(j0, py0); j1 = min(j1, ty1);
                const int bw = i1 - i0 + 1, n = bw * (j1 - j0 + 1);
                const uint32_t layer = tri.w, lid = gt - sc.tri_off[layer];
                unsigned long long* kl = keys + layer * VS_TILE_PIX;
                int m0, m1, m2;
                vs_edge_mins(T, m0, m1, m2);
                for (int s = (int)lane; s < n; s += 32) {
                    const int i = i0 + s % bw, j = j0 + s / bw;
                    VsEdges e;
                    vs_edges_at(T, i, j, e);
                    if (e.E0 >= m0 && e.E1 >= m1 && e.E2 >= m2)
                        vs_key_max(&kl[(j - py0) * VS_TILE_W + (i - px0)], vs_make_key(vs_depth_q(T, e.E0, e.E1, e.E2), lid));
                }
            }
            __syncthreads();
            if (tid == 0) bigcount = 0;
            __syncthreads();
        }
    }
    __syncthreads();

    // ---------------- phase 2: shade + composite ----------------
    const uint32_t oct = lane >> 3, oi = lane & 7;  // octet index / lane within octet
    VsFragRec* rec = rec_all + warp * 32;
    float4* part = part_all + warp * 32 * 8;
    float* ysm = reinterpret_cast<float*>(part);    // Y staging aliases the partial-sum buffer

    bool any_hit = false;
    for (uint32_t l = 0; l < sc.k; ++l) any_hit |= (keys[l * VS_TILE_PIX + pl] != 0ull);
    const bool warp_any = __any_sync(0xFFFFFFFFu, any_hit);

    float Yr[8][SLOTS][CPV];
    if (warp_any) {
        float Y[YROW];
#pragma unroll
        for (int c = 0; c < YROW; ++c) Y[c] = 0.0f;
        float vx, vy, vz;
        vs_view_dir(cams[view], px, py, vx, vy, vz);
        vs_sh_basis<DEG>(vx, vy, vz, Y);
#pragma unroll
        for (int c = 0; c < YROW; ++c) ysm[lane * YROW + c] = Y[c];
        __syncwarp();
#pragma unroll
        for (int j = 0; j < 8; ++j)
#pragma unroll
            for (int s = 0; s < SLOTS; ++s)
#pragma unroll
                for (int c = 0; c < CPV; ++c) Yr[j][s][c] = ysm[(4 * j + oct) * YROW + (oi + 8 * s) * CPV + c];
        __syncwarp();
    }

    float Tr = 1.0f, Cr = 0.0f, Cg = 0.0f, Cb = 0.0f;
    bool alive = true;
    for (uint32_t l = 0; l < sc.k; ++l) {
        const unsigned long long key = keys[l * VS_TILE_PIX + pl];
        const bool hit = key != 0ull;
        const uint32_t lid = 0xFFFFFFFFu - (uint32_t)key;
        if (out_ids && inimg) out_ids[(((size_t)view * sc.k + l) * H + py) * W + px] = hit ? lid : VS_MISS;
        const bool shade = hit && alive;
        const unsigned m = __ballot_sync(0xFFFFFFFFu, shade);
        if (m == 0) continue;  // warp-uniform
        VsFragRec r;
        r.o00 = r.o01 = r.o10 = r.o11 = 0; r.w00 = r.w01 = r.w10 = r.w11 = 0.0f;
        if (shade) vs_fragment_record(sc, vv, l, lid, px, py, r);
        if (COUNT) {  // measurement aid: mark the 2x2 footprint in this view's texel bitmap
            if (shade) {
                uint32_t* bits = texel_bits + (size_t)view * (sc.tex_bit_off[sc.k] >> 5);
                const uint32_t o4[4] = {r.o00, r.o01, r.o10, r.o11};
                for (int q = 0; q < 4; ++q) {
                    const uint32_t bit = sc.tex_bit_off[l] + o4[q] / sc.texel_vecs;
                    atomicOr(&bits[bit >> 5], 1u << (bit & 31));
                }
            }
            if (lane == 0) atomicAdd(&counters[VS_CNT_FRAGS], (unsigned long long)__popc(m));
        }
        rec[lane] = r;
        __syncwarp();
        const uint4* __restrict__ tb = sc.tex[l];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            if ((m >> (4 * j)) & 0xFu) {
                const VsFragRec* rp = &rec[4 * j + oct];
                const uint4 o = *reinterpret_cast<const uint4*>(rp);
                const float4 w = *(reinterpret_cast<const float4*>(rp) + 1);
                float4 acc = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
#pragma unroll
                for (int s = 0; s < SLOTS; ++s) {
                    const uint32_t vi = oi + 8 * s;
                    if (vi < (uint32_t)NVEC) {
                        const uint4 t00 = __ldg(tb + o.x + vi), t01 = __ldg(tb + o.y + vi);
                        const uint4 t10 = __ldg(tb + o.z + vi), t11 = __ldg(tb + o.w + vi);
                        vs_accumulate_vec<F16>(t00, t01, t10, t11, w, Yr[j][s], acc);
                    }
                }
                if (oi < (uint32_t)NACT) part[(4 * j + oct) * 8 + oi] = acc;
            }
        }
        __syncwarp();
        if (shade) {
            float4 s4 = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
#pragma unroll
            for (int s = 0; s < NACT; ++s) {
                const float4 p = part[lane * 8 + ((s + lane) % NACT)];
                s4.x += p.x; s4.y += p.y; s4.z += p.z; s4.w += p.w;
            }
            const float A = vs_sigmoid(s4.w);
            const float TA = Tr * A;
            Cr += TA * vs_sigmoid(s4.x); Cg += TA * vs_sigmoid(s4.y); Cb += TA * vs_sigmoid(s4.z);
            Tr *= (1.0f - A);
            if (Tr < fr.t_min) alive = false;
        }
        __syncwarp();
    }
    if (inimg)
        reinterpret_cast<float4*>(out_rgba)[((size_t)view * H + py) * W + px] =
            make_float4(Cr + Tr * fr.bg[0], Cg + Tr * fr.bg[1], Cb + Tr * fr.bg[2], 1.0f - Tr);
}

template <int F16, int DEG, bool COUNT>
static cudaError_t launch_rs2(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    const size_t smem = (size_t)sc.k * VS_TILE_PIX * 8 + 8 * 32 * sizeof(VsFragRec) + 8 * 32 * 8 * sizeof(float4);
    auto kern = k_raster_shade<F16, DEG, COUNT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid(fr.tiles_x * fr.tiles_y, ch.views);
    kern<<<grid, 256, smem, st>>>(sc, fr, ch.cams, ch.vtx, ch.tile_off, ch.tile_tris, ch.out_rgba, ch.out_ids,
                                  ch.texel_bits, ch.counters);
    return cudaGetLastError();
}

template <int F16, int DEG>
static cudaError_t launch_rs(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    return ch.texel_bits ? launch_rs2<F16, DEG, true>(sc, fr, ch, st) : launch_rs2<F16, DEG, false>(sc, fr, ch, st);
}

cudaError_t vs_launch_raster_shade(const VsSceneDev& sc, int f16, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    switch ((f16 ? 4 : 0) + (int)sc.sh_degree) {
        case 0: return launch_rs<0, 0>(sc, fr, ch, st);
        case 1: return launch_rs<0, 1>(sc, fr, ch, st);
        case 2: return launch_rs<0, 2>(sc, fr, ch, st);
        case 3: return launch_rs<0, 3>(sc, fr, ch, st);
        case 4: return launch_rs<1, 0>(sc, fr, ch, st);
        case 5: return launch_rs<1, 1>(sc, fr, ch, st);
        case 6: return launch_rs<1, 2>(sc, fr, ch, st);
        case 7: return launch_rs<1, 3>(sc, fr, ch, st);
    }
    return cudaErrorInvalidValue;
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
        VsFragRec r;
        vs_fragment_record(sc, vv, l, lid, px, py, r);
        const uint32_t offs[4] = {r.o00, r.o01, r.o10, r.o11};
        const float ws[4] = {r.w00, r.w01, r.w10, r.w11};
        float s[4] = {0.0f, 0.0f, 0.0f, 0.0f};
        for (uint32_t c = 0; c < sc.n_coef; ++c)
            for (int ch = 0; ch < 4; ++ch) {
                float v = 0.0f;
                for (int q = 0; q < 4; ++q) {
                    float tv;
                    if (F16) tv = __half2float(reinterpret_cast<const __half*>(sc.tex[l] + offs[q])[4 * c + ch]);
                    else tv = reinterpret_cast<const float*>(sc.tex[l] + offs[q])[4 * c + ch];
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
    if (f16) k_reference<1><<<grid, 128, 0, st>>>(sc, fr, ch.cams, ch.vtx, ch.out_rgba, ch.out_ids);
    else k_reference<0><<<grid, 128, 0, st>>>(sc, fr, ch.cams, ch.vtx, ch.out_rgba, ch.out_ids);
    return cudaGetLastError();
}

// VS_FLAG_COUNT_TEXELS: population count of the texel bitmaps
__global__ void k_popcount(const uint32_t* __restrict__ w, size_t n, unsigned long long* counter)
{
    unsigned long long c = 0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) c += __popc(w[i]);
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xFFFFFFFFu, c, o);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(counter, c);
}

cudaError_t vs_launch_popcount(const uint32_t* words, size_t n, unsigned long long* counter, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    k_popcount<<<148 * 4, 256, 0, st>>>(words, n, counter);
    return cudaGetLastError();
}

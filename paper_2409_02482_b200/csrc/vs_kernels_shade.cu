// vs_kernels_shade.cu -- S5 perspective-correct UV + bilinear texel fetch, S6 SH evaluation + sigmoid,
// S7 fixed-order front-to-back compositing.  DESIGN.md §1, §3.5-3.8, §7.
//
// One CTA per (view, 16x16 tile), a warp owns an 8x4 pixel block, lane = pixel ("owner").
// Phase A: every owner turns the winning triangle of each layer (the id planes k_raster wrote) into
//   a packed fragment record (clamped texel column/row of the 2x2 footprint + the two bilinear
//   fractions) in shared memory.  The gather chain id -> triangle -> 3 vertices + 3 uvs is paid once
//   per tile, three layers at a time, instead of once per layer inside the shading loop.
// Phase B: per layer the warp re-maps itself to 4 fragments x 8 lanes: octet `o` streams the four
//   texels of the fragment of pixel row `o`, column `j`, as 16-byte vectors (one full 128-byte line
//   per octet per texel at SH degree 3 / fp16), blends them with the bilinear weights, dots with
//   the pixel's SH basis (kept in registers for all layers) and hands 4 partial channel sums back
//   through shared memory.  Owners add the partials, apply the sigmoid and composite front to back.
#include "vs_common.cuh"

struct __align__(16) VsFragRec {
    uint32_t o00, o01, o10, o11;  // 16-byte-vector offsets of the four texels inside the layer texture
    float w00, w01, w10, w11;     // bilinear weights
};

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

// packed record: cx0 | (cx1 != cx0) << 15 | cy0 << 16 | (cy1 != cy0) << 31  (texture sides <= 32768)
__device__ __forceinline__ uint32_t vs_pack_frag(const VsFrag& f)
{
    return f.cx0 | ((f.cx1 != f.cx0) ? 0x8000u : 0u) | (f.cy0 << 16) | ((f.cy1 != f.cy0) ? 0x80000000u : 0u);
}

template <int F16, int DEG, bool COUNT>
__global__ void __launch_bounds__(256, 2)
k_shade(const VsSceneDev sc, const VsFrame fr, const VsCamDev* __restrict__ cams, const int4* __restrict__ vtx,
        const uint32_t* __restrict__ tile_off, const uint32_t* __restrict__ ids, float* __restrict__ out_rgba,
        uint32_t* __restrict__ texel_bits, unsigned long long* __restrict__ counters)
{
    constexpr int NCOEF = (DEG + 1) * (DEG + 1);
    constexpr int CPV = F16 ? 2 : 1;                 // coefficients per 16-byte vector
    constexpr int NVEC = (NCOEF + CPV - 1) / CPV;    // vectors per texel (== sc.texel_vecs)
    constexpr int SLOTS = (NVEC + 7) / 8;            // vectors per octet lane
    constexpr int NACT = NVEC < 8 ? NVEC : 8;        // octet lanes that hold data
    constexpr int YROW = SLOTS * 8 * CPV;            // floats per pixel in the Y staging buffer

    extern __shared__ __align__(16) unsigned char smem[];
    // [k][256] packed texel coordinates, then [k][256] float2 fractions (a < 0: no fragment)
    uint32_t* rec_xy = reinterpret_cast<uint32_t*>(smem);
    float2* rec_ab = reinterpret_cast<float2*>(smem + (size_t)sc.k * VS_TILE_PIX * 4);
    unsigned char* per_warp = smem + (size_t)sc.k * VS_TILE_PIX * 12;  // 8 x (1 KB records + 4 KB partial sums)

    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t tile = blockIdx.x, view = blockIdx.y;
    const uint32_t tiles = fr.tiles_x * fr.tiles_y;
    const int W = (int)fr.width, H = (int)fr.height;
    // lane -> pixel of the warp's 8x4 block: column = lane & 7, row = lane >> 3
    const int lx = (int)(warp & 1) * 8 + (int)(lane & 7), ly = (int)(warp >> 1) * 4 + (int)(lane >> 3);
    const int px = (int)(tile % fr.tiles_x) * VS_TILE_W + lx, py = (int)(tile / fr.tiles_x) * VS_TILE_H + ly;
    const bool inimg = px < W && py < H;
    const size_t pix = ((size_t)view * H + py) * W + px;

    if (tile_off[view * tiles + tile] == tile_off[view * tiles + tile + 1]) {  // nothing binned here: background
        if (inimg) reinterpret_cast<float4*>(out_rgba)[pix] = make_float4(fr.bg[0], fr.bg[1], fr.bg[2], 0.0f);
        return;
    }
    const int4* __restrict__ vv = vtx + (size_t)view * sc.v_total;

    // ---------------- phase A: fragment records of all layers ----------------
    const size_t plane = (size_t)W * H;
    const uint32_t* idp = ids + (size_t)view * sc.k * plane + (size_t)py * W + px;
    bool any_hit = false;
    for (uint32_t l0 = 0; l0 < sc.k; l0 += 3) {
        uint32_t id[3];
#pragma unroll
        for (int u = 0; u < 3; ++u) id[u] = (inimg && l0 + u < sc.k) ? __ldg(idp + (size_t)(l0 + u) * plane) : VS_MISS;
#pragma unroll
        for (int u = 0; u < 3; ++u) {
            if (l0 + u < sc.k) {
                uint32_t xy = 0;
                float2 ab = make_float2(-1.0f, 0.0f);
                if (id[u] != VS_MISS) {
                    VsFrag f;
                    vs_fragment_setup(sc, vv, l0 + u, id[u], px, py, f);
                    xy = vs_pack_frag(f);
                    ab = make_float2(f.a, f.b);
                    any_hit = true;
                }
                rec_xy[(l0 + u) * VS_TILE_PIX + tid] = xy;
                rec_ab[(l0 + u) * VS_TILE_PIX + tid] = ab;
            }
        }
    }
    // each thread reads back only its own records: no barrier needed

    // ---------------- phase B: shade + composite ----------------
    const uint32_t oct = lane >> 3, oi = lane & 7;  // octet index (= pixel row) / lane within octet
    VsFragRec* rec = reinterpret_cast<VsFragRec*>(per_warp + warp * 5120);
    float4* part = reinterpret_cast<float4*>(per_warp + warp * 5120 + 1024);
    float* ysm = reinterpret_cast<float*>(part);    // Y staging aliases the partial-sum buffer

    if (!__any_sync(0xFFFFFFFFu, any_hit)) {
        if (inimg) reinterpret_cast<float4*>(out_rgba)[pix] = make_float4(fr.bg[0], fr.bg[1], fr.bg[2], 0.0f);
        return;
    }
    float Yr[8][SLOTS][CPV];
    {
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
                for (int c = 0; c < CPV; ++c) Yr[j][s][c] = ysm[(8 * oct + j) * YROW + (oi + 8 * s) * CPV + c];
        __syncwarp();
    }

    float Tr = 1.0f, Cr = 0.0f, Cg = 0.0f, Cb = 0.0f;
    bool alive = true;
    for (uint32_t l = 0; l < sc.k; ++l) {
        const float2 ab = rec_ab[l * VS_TILE_PIX + tid];
        const bool shade = ab.x >= 0.0f && alive;
        const unsigned m = __ballot_sync(0xFFFFFFFFu, shade);
        if (m == 0) continue;  // warp-uniform
        VsFragRec r;
        r.o00 = r.o01 = r.o10 = r.o11 = 0; r.w00 = r.w01 = r.w10 = r.w11 = 0.0f;
        if (shade) {
            const uint32_t xy = rec_xy[l * VS_TILE_PIX + tid];
            const uint32_t cx0 = xy & 0x7FFFu, cy0 = (xy >> 16) & 0x7FFFu;
            const uint32_t Wt = sc.tex_w[l], nv = (uint32_t)NVEC;
            const uint32_t row0 = cy0 * Wt, row1 = row0 + ((xy >> 31) ? Wt : 0u);
            const uint32_t cx1 = cx0 + ((xy >> 15) & 1u);
            r.o00 = (row0 + cx0) * nv; r.o01 = (row0 + cx1) * nv;
            r.o10 = (row1 + cx0) * nv; r.o11 = (row1 + cx1) * nv;
            r.w00 = (1.0f - ab.x) * (1.0f - ab.y); r.w01 = ab.x * (1.0f - ab.y);
            r.w10 = (1.0f - ab.x) * ab.y;          r.w11 = ab.x * ab.y;
            if (COUNT) {  // measurement aid: mark the 2x2 footprint in this view's texel bitmap
                uint32_t* bits = texel_bits + (size_t)view * (sc.tex_bit_off[sc.k] >> 5);
                const uint32_t o4[4] = {r.o00, r.o01, r.o10, r.o11};
                for (int q = 0; q < 4; ++q) {
                    const uint32_t bit = sc.tex_bit_off[l] + o4[q] / nv;
                    atomicOr(&bits[bit >> 5], 1u << (bit & 31));
                }
            }
        }
        if (COUNT && lane == 0) atomicAdd(&counters[VS_CNT_FRAGS], (unsigned long long)__popc(m));
        rec[lane] = r;
        __syncwarp();
        const uint4* __restrict__ tb = sc.tex[l];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            if (m & (0x01010101u << j)) {  // some pixel of column j is shaded
                const VsFragRec* rp = &rec[8 * oct + j];
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
                if (oi < (uint32_t)NACT) part[(8 * oct + j) * 8 + oi] = acc;
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
        reinterpret_cast<float4*>(out_rgba)[pix] = make_float4(Cr + Tr * fr.bg[0], Cg + Tr * fr.bg[1], Cb + Tr * fr.bg[2], 1.0f - Tr);
}

template <int F16, int DEG, bool COUNT>
static cudaError_t launch_sh2(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    const size_t smem = (size_t)sc.k * VS_TILE_PIX * 12 + 8 * 5120;
    auto kern = k_shade<F16, DEG, COUNT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid(fr.tiles_x * fr.tiles_y, ch.views);
    kern<<<grid, 256, smem, st>>>(sc, fr, ch.cams, ch.vtx, ch.tile_off, ch.ids, ch.out_rgba, ch.texel_bits, ch.counters);
    return cudaGetLastError();
}

template <int F16, int DEG>
static cudaError_t launch_sh(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    return ch.texel_bits ? launch_sh2<F16, DEG, true>(sc, fr, ch, st) : launch_sh2<F16, DEG, false>(sc, fr, ch, st);
}

cudaError_t vs_launch_shade(const VsSceneDev& sc, int f16, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    switch ((f16 ? 4 : 0) + (int)sc.sh_degree) {
        case 0: return launch_sh<0, 0>(sc, fr, ch, st);
        case 1: return launch_sh<0, 1>(sc, fr, ch, st);
        case 2: return launch_sh<0, 2>(sc, fr, ch, st);
        case 3: return launch_sh<0, 3>(sc, fr, ch, st);
        case 4: return launch_sh<1, 0>(sc, fr, ch, st);
        case 5: return launch_sh<1, 1>(sc, fr, ch, st);
        case 6: return launch_sh<1, 2>(sc, fr, ch, st);
        case 7: return launch_sh<1, 3>(sc, fr, ch, st);
    }
    return cudaErrorInvalidValue;
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

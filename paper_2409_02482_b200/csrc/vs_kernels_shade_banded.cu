// vs_kernels_shade_banded.cu -- S5-S7 for the paper's banded 8-bit texture format (§4.5 "Mixed
// resolutions" / "Squeezing and quantization").
//
// A fragment reads, per SH band b, the 2x2 footprint of THAT band's image (its own resolution): 4, 12, 20, 28 bytes per
// texel (padded to 4, 16, 32, 32), 64 coefficient bytes per texel set instead of the 128 of the fp16 format, and the
// higher bands touch 4-64x fewer distinct texels.  The byte textures of a whole C4 scene (315 MB) nearly fit the L2,
// so this path is bound by the plain FP32/ALU pipes, not by HBM: ~580 lane-ops per fragment (256 byte->float
// conversions, 256 bilinear FMAs, 64 SH FMAs).  There is no reason for the octet mapping of k_shade (which exists to
// form 128-byte line requests): one lane = one pixel, all layers composited in registers; shared memory only holds the
// per-(pixel, layer) UV records that phase A gathers level by level.
//
//   s_ch = sum_b sum_m Y_{b,m} (v_min + v_scale * bilinear_b(t)[m][ch]) = v_min sum_c Y_c + v_scale sum_c Y_c blend_c[ch]
//
// bytes -> float: PRMT of the byte into the mantissa of 2^23 (0x4B000000), then an add of -2^23 (exact).  The pipes are
// balanced on purpose (both issue one warp instruction per 2 clocks per SM sub-partition): per coefficient word 16 PRMT on
// the alu pipe against 8 FADD2 + 8 FFMA2 + 2 FMUL2 on the fma pipe, all packed fp32 pairs (texels 0|1 and 2|3).
#include "vs_common.cuh"


// byte SEL of two words -> the pair (2^23 + byte of wa, 2^23 + byte of wb): the byte lands in the mantissa of 0x4B000000
template <int SEL>
__device__ __forceinline__ f32x2 vs_bytes_magic(uint32_t wa, uint32_t wb)
{
    // the constant is the FIRST operand so that the selector is an immediate of PRMT (one register holds 0x4B000000)
    return vs_pack2(__uint_as_float(__byte_perm(0x4B000000u, wa, 0x3104 + SEL)),
                    __uint_as_float(__byte_perm(0x4B000000u, wb, 0x3104 + SEL)));
}

// One coefficient (4-byte word = its 4 channels) of the four texels of a footprint.  acc[ch] holds the pair
// (sum over texels 0, 2 | sum over texels 1, 3) of Z_q * byte: per channel 4 PRMT (alu pipe), 2 FADD2 of -2^23 (exact)
// and 2 FFMA2 (fma pipe); Z01 = (Z_0, Z_1), Z23 = (Z_2, Z_3), Z_q = bilinear weight x SH basis value x v_scale.
__device__ __forceinline__ void vs_acc_coef(uint32_t w0, uint32_t w1, uint32_t w2, uint32_t w3, f32x2 Z01, f32x2 Z23, f32x2* acc)
{
    const f32x2 NM = vs_pack2(-8388608.0f, -8388608.0f);
    acc[0] = vs_fma2(Z01, vs_add2(vs_bytes_magic<0>(w0, w1), NM), acc[0]);
    acc[0] = vs_fma2(Z23, vs_add2(vs_bytes_magic<0>(w2, w3), NM), acc[0]);
    acc[1] = vs_fma2(Z01, vs_add2(vs_bytes_magic<1>(w0, w1), NM), acc[1]);
    acc[1] = vs_fma2(Z23, vs_add2(vs_bytes_magic<1>(w2, w3), NM), acc[1]);
    acc[2] = vs_fma2(Z01, vs_add2(vs_bytes_magic<2>(w0, w1), NM), acc[2]);
    acc[2] = vs_fma2(Z23, vs_add2(vs_bytes_magic<2>(w2, w3), NM), acc[2]);
    acc[3] = vs_fma2(Z01, vs_add2(vs_bytes_magic<3>(w0, w1), NM), acc[3]);
    acc[3] = vs_fma2(Z23, vs_add2(vs_bytes_magic<3>(w2, w3), NM), acc[3]);
}

// band B of one fragment: 2x2 footprint at the band's own resolution, accumulated into the four channel sums
template <int B>
__device__ __forceinline__ void vs_band(const VsSceneDev& sc, uint32_t l, float u0, float du, float v0, float dv, const float* Y,
                                        f32x2* acc)
{
    constexpr int NB = 2 * B + 1;                 // coefficients = 4-byte words of this band
    constexpr uint32_t STRIDE = VS_BAND_STRIDE(B);
    const int Wb = (int)sc.bw[l][B], Hb = (int)sc.bh[l][B];
    uint32_t cx0, cx1, cy0, cy1;
    float fa, fb;
    vs_texel_coord(u0, du, (float)Wb, Wb, cx0, cx1, fa);
    vs_texel_coord(v0, dv, (float)Hb, Hb, cy0, cy1, fb);
    const unsigned char* base = sc.btex[l][B];
    const uint32_t o[4] = {(cy0 * (uint32_t)Wb + cx0) * STRIDE, (cy0 * (uint32_t)Wb + cx1) * STRIDE,
                           (cy1 * (uint32_t)Wb + cx0) * STRIDE, (cy1 * (uint32_t)Wb + cx1) * STRIDE};
    const float ga = 1.0f - fa, gb = (1.0f - fb) * sc.v_scale, hb = fb * sc.v_scale;
    const f32x2 W01 = vs_pack2(ga * gb, fa * gb), W23 = vs_pack2(ga * hb, fa * hb);   // bilinear weights x v_scale
    uint32_t w[4][NB <= 1 ? 1 : (NB <= 4 ? 4 : 8)];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        if (B == 0) {
            w[q][0] = __ldg(reinterpret_cast<const uint32_t*>(base + o[q]));
        } else {
            const uint4 t0 = __ldg(reinterpret_cast<const uint4*>(base + o[q]));
            w[q][0] = t0.x; w[q][1] = t0.y; w[q][2] = t0.z; w[q][3] = t0.w;
            if (B >= 2) {
                const uint4 t1 = __ldg(reinterpret_cast<const uint4*>(base + o[q]) + 1);
                w[q][4] = t1.x; w[q][5] = t1.y; w[q][6] = t1.z; w[q][7] = t1.w;
            }
        }
    }
#pragma unroll
    for (int m = 0; m < NB; ++m) {
        const f32x2 yy = vs_pack2(Y[B * B + m], Y[B * B + m]);
        vs_acc_coef(w[0][m], w[1][m], w[2][m], w[3][m], vs_mul2(W01, yy), vs_mul2(W23, yy), acc);
    }
}

template <int DEG, bool COUNT>
#ifndef VS_BANDED_MIN_CTAS
#define VS_BANDED_MIN_CTAS 3
#endif
__global__ void __launch_bounds__(256, VS_BANDED_MIN_CTAS)
k_shade_banded(const VsSceneDev sc, const VsFrame fr, const VsCamDev* __restrict__ cams, const int4* __restrict__ vtx,
               const uint32_t* __restrict__ tile_off, const uint32_t* __restrict__ ids, unsigned long long* __restrict__ keys,
               uint32_t* __restrict__ out_ids, float* __restrict__ out_rgba, unsigned long long* __restrict__ counters)
{
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t tile = blockIdx.x, view = blockIdx.y;
    const uint32_t tiles = fr.tiles_x * fr.tiles_y;
    const int W = (int)fr.width, H = (int)fr.height;
    const int lx = (int)(warp & 1) * 8 + (int)(lane & 7), ly = (int)(warp >> 1) * 4 + (int)(lane >> 3);
    const int px = (int)(tile % fr.tiles_x) * VS_TILE_W + lx, py = (int)(tile / fr.tiles_x) * VS_TILE_H + ly;
    const bool inimg = px < W && py < H;
    const size_t pix = ((size_t)view * H + py) * W + px;
    const size_t plane = (size_t)W * H;
    const size_t pix0 = (size_t)view * sc.k * plane + (size_t)py * W + px;

    // tiled path: tile_off = reference list offsets; direct path: tile_off = per-tile masks of the layers drawn into
    const uint32_t lmask = keys ? tile_off[view * tiles + tile] : 0xFFFFFFFFu;
    if (keys ? lmask == 0u : tile_off[view * tiles + tile] == tile_off[view * tiles + tile + 1]) {
        if (out_ids && inimg)
            for (uint32_t l = 0; l < sc.k; ++l) out_ids[pix0 + (size_t)l * plane] = VS_MISS;
        if (inimg) reinterpret_cast<float4*>(out_rgba)[pix] = make_float4(fr.bg[0], fr.bg[1], fr.bg[2], 0.0f);
        return;
    }
    const int4* __restrict__ vv = vtx + (size_t)view * sc.v_total;

    // ---------------- phase A: perspective-correct UV (base + offset) of every layer's fragment -> shared memory ----------------
    // The gather chain key/id -> index record -> 3 vertices + 3 uvs is walked level by level over all layers (all keys,
    // then all index records, then the vertices), so a tile pays ~4 dependent round trips instead of 3 per layer.
    extern __shared__ __align__(16) unsigned char smem[];
    float4* rec = reinterpret_cast<float4*>(smem);     // [k][256] {u0, du, v0, dv}
    uint32_t hitmask = 0;
    {
        uint32_t id[VS_MAX_LAYERS];
        if (keys) {
            // direct path: the key image of k_raster_direct; what is read is cleared for the next pass over this buffer
            unsigned long long key[VS_MAX_LAYERS];
#pragma unroll
            for (int u = 0; u < VS_MAX_LAYERS; ++u)
                key[u] = (inimg && u < (int)sc.k && ((lmask >> u) & 1u)) ? keys[pix0 + (size_t)u * plane] : 0ull;
#pragma unroll
            for (int u = 0; u < VS_MAX_LAYERS; ++u) {
                id[u] = key[u] ? 0xFFFFFFFFu - (uint32_t)key[u] : VS_MISS;
                if (key[u]) keys[pix0 + (size_t)u * plane] = 0ull;
                if (out_ids && inimg && u < (int)sc.k) out_ids[pix0 + (size_t)u * plane] = id[u];
            }
        } else {
#pragma unroll
            for (int u = 0; u < VS_MAX_LAYERS; ++u)
                id[u] = (inimg && u < (int)sc.k) ? __ldg(ids + pix0 + (size_t)u * plane) : VS_MISS;
        }
        uint4 tri[VS_MAX_LAYERS];
#pragma unroll
        for (int u = 0; u < VS_MAX_LAYERS; ++u)
            tri[u] = id[u] != VS_MISS ? __ldg(&sc.tris[sc.tri_off[u] + id[u]]) : make_uint4(0, 0, 0, 0);
#pragma unroll
        for (int u = 0; u < VS_MAX_LAYERS; ++u) {
            if (u < (int)sc.k && id[u] != VS_MISS) {
                float4 r;
                vs_fragment_uv(sc, vv, tri[u], px, py, r.x, r.y, r.z, r.w);
                rec[u * VS_TILE_PIX + tid] = r;
                hitmask |= 1u << u;
            }
        }
        if (fr.attenuate) {
            // alpha_w of every fragment (all of a pixel's fragments share its view direction) -> second record plane
            float* rec_aw = reinterpret_cast<float*>(smem + (size_t)sc.k * VS_TILE_PIX * 16);
            float ax, ay, az;
            vs_view_dir(cams[view], px, py, ax, ay, az);
#pragma unroll
            for (int u = 0; u < VS_MAX_LAYERS; ++u)
                if (u < (int)sc.k && id[u] != VS_MISS)
                    rec_aw[u * VS_TILE_PIX + tid] = vs_alpha_w(ax, ay, az, vs_fragment_normal(sc, vv, u, id[u], px, py));
        }
    }
    // each thread reads back only its own records: no barrier needed
    if (!__any_sync(0xFFFFFFFFu, hitmask != 0u)) {
        if (inimg) reinterpret_cast<float4*>(out_rgba)[pix] = make_float4(fr.bg[0], fr.bg[1], fr.bg[2], 0.0f);
        return;
    }

    // ---------------- phase B: per layer, four band footprints -> logits -> composite (registers only) ----------------
    float Y[16];
#pragma unroll
    for (int c = 0; c < 16; ++c) Y[c] = 0.0f;
    {
        float vx, vy, vz;
        vs_view_dir(cams[view], px, py, vx, vy, vz);
        vs_sh_basis<DEG>(vx, vy, vz, Y);
    }
    float ysum = 0.0f;
#pragma unroll
    for (int c = 0; c < (DEG + 1) * (DEG + 1); ++c) ysum += Y[c];
    const float sbase = sc.v_min * ysum;          // v_min sum_c Y_c: the constant part of every channel's logit
    const float* rec_aw = reinterpret_cast<const float*>(smem + (size_t)sc.k * VS_TILE_PIX * 16);

    float Tr = 1.0f, Cr = 0.0f, Cg = 0.0f, Cb = 0.0f;
    bool alive = true;
    unsigned nfrag = 0;
    for (uint32_t l = 0; l < sc.k; ++l) {
        if (!((hitmask >> l) & 1u) || !alive) continue;
        const float4 r = rec[l * VS_TILE_PIX + tid];
        const float u0 = r.x, du = r.y, v0 = r.z, dv = r.w;
        f32x2 acc[4];
        acc[0] = acc[1] = acc[2] = acc[3] = vs_pack2(sbase, 0.0f);
        vs_band<0>(sc, l, u0, du, v0, dv, Y, acc);
        if (DEG >= 1) vs_band<1>(sc, l, u0, du, v0, dv, Y, acc);
        if (DEG >= 2) vs_band<2>(sc, l, u0, du, v0, dv, Y, acc);
        if (DEG >= 3) vs_band<3>(sc, l, u0, du, v0, dv, Y, acc);
        float s0, s1, s2, s3, hi;
        vs_unpack2(acc[0], s0, hi); s0 += hi;
        vs_unpack2(acc[1], s1, hi); s1 += hi;
        vs_unpack2(acc[2], s2, hi); s2 += hi;
        vs_unpack2(acc[3], s3, hi); s3 += hi;
        if (COUNT) ++nfrag;
        float A = vs_sigmoid(s3);
        if (fr.attenuate) A *= rec_aw[l * VS_TILE_PIX + tid];
        const float TA = Tr * A;
        Cr += TA * vs_sigmoid(s0); Cg += TA * vs_sigmoid(s1); Cb += TA * vs_sigmoid(s2);
        Tr *= (1.0f - A);
        if (Tr < fr.t_min) alive = false;
    }
    if (COUNT) {
        for (int o = 16; o > 0; o >>= 1) nfrag += __shfl_xor_sync(0xFFFFFFFFu, nfrag, o);
        if (lane == 0 && nfrag) atomicAdd(&counters[VS_CNT_FRAGS], (unsigned long long)nfrag);
    }
    if (inimg)
        reinterpret_cast<float4*>(out_rgba)[pix] = make_float4(Cr + Tr * fr.bg[0], Cg + Tr * fr.bg[1], Cb + Tr * fr.bg[2], 1.0f - Tr);
}

template <int DEG, bool COUNT>
static cudaError_t launch_b(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    dim3 grid(fr.tiles_x * fr.tiles_y, ch.views);
    auto kern = k_shade_banded<DEG, COUNT>;
    const size_t smem = (size_t)sc.k * VS_TILE_PIX * (fr.attenuate ? 20 : 16);
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (ch.keys)
        kern<<<grid, 256, smem, st>>>(sc, fr, ch.cams, ch.vtx, ch.tile_mask, nullptr, ch.keys, ch.ids_is_output ? ch.ids : nullptr,
                                   ch.out_rgba, ch.counters);
    else
        kern<<<grid, 256, smem, st>>>(sc, fr, ch.cams, ch.vtx, ch.tile_off, ch.ids, nullptr, nullptr, ch.out_rgba, ch.counters);
    return cudaGetLastError();
}

cudaError_t vs_launch_shade_banded(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    const bool cnt = ch.count_fragments != 0;
    switch (sc.sh_degree) {
        case 0: return cnt ? launch_b<0, true>(sc, fr, ch, st) : launch_b<0, false>(sc, fr, ch, st);
        case 1: return cnt ? launch_b<1, true>(sc, fr, ch, st) : launch_b<1, false>(sc, fr, ch, st);
        case 2: return cnt ? launch_b<2, true>(sc, fr, ch, st) : launch_b<2, false>(sc, fr, ch, st);
        case 3: return cnt ? launch_b<3, true>(sc, fr, ch, st) : launch_b<3, false>(sc, fr, ch, st);
    }
    return cudaErrorInvalidValue;
}

// vs_kernels_backward.cu -- backward pass to the texels (§4.5: the textures are
// fitted through the very lookup the renderer performs).  Given dL/d(out_rgba) of a batch of views it
// accumulates dL/d(texture coefficient) of every layer, by the chain rule through S7 blend -> S6 sigmoid / SH dot ->
// S5 bilinear weights.  S1-S4 (transform, coverage, nearest fragment) run unchanged before it: this kernel takes the
// place of k_shade and consumes (and clears) the same key image.
//
// One lane = one pixel.  Pass 1 re-shades the pixel's fragments front to back with the plain routine of vs_plain.cuh and
// keeps (rgb, sigma, alpha_w, T) of every layer it composites; pass 2 walks them back to front with the recurrence
//   R_end = bg . g_rgb - g_a ;  dL/dA_l = T_l (rgb_l . g_rgb - R_l) ;  R_{l-1} = A_l (rgb_l . g_rgb) + (1 - A_l) R_l
// and scatters w_q Y_c dL/ds_ch into the gradient textures ([texel][c][ch] fp32 = the API layout of the textures) with
// fire-and-forget vector reductions: one RED.ADD.v4.F32 per (texel, coefficient), 4 (deg + 1)^2 per fragment, issued by
// octets of lanes so that an instruction covers whole 128-byte lines.  The scatter is the cost: 1 KB of reductions per
// fragment at degree 3 against 512 bytes read.  fp32 sums in arbitrary order: parity is to a relative tolerance.
#include "vs_common.cuh"
#include "vs_plain.cuh"

__device__ __forceinline__ void vs_red_add4(float* p, float a, float b, float c, float d)
{
#ifdef VS_BW_EXP_NORED     // timing experiment only (wrong gradients): everything but the reductions
    if (a != 12345.678f) return;
#endif
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

template <int F16>
__global__ void __launch_bounds__(256, 3)
k_backward(const VsSceneDev sc, const VsFrame fr, const VsCamDev* __restrict__ cams, const int4* __restrict__ vtx,
           const uint32_t* __restrict__ tile_mask, unsigned long long* __restrict__ keys, const float* __restrict__ grad_out,
           VsGradTex gt, const uint32_t* __restrict__ order)
{
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t tiles = fr.tiles_x * fr.tiles_y;
    uint32_t tile = blockIdx.x, view = blockIdx.y;
    if (order) {   // surface order (vs_kernels_order.cu): the views' updates of a gradient texel meet in L2
        const uint32_t e = __ldg(&order[view * tiles + tile]);
        view = e / tiles; tile = e - view * tiles;
    }
    const int W = (int)fr.width, H = (int)fr.height;
    const int lx = (int)(warp & 1) * 8 + (int)(lane & 7), ly = (int)(warp >> 1) * 4 + (int)(lane >> 3);
    const int px = (int)(tile % fr.tiles_x) * VS_TILE_W + lx, py = (int)(tile / fr.tiles_x) * VS_TILE_H + ly;
    const uint32_t lmask = tile_mask[view * tiles + tile];
    if (lmask == 0u) return;                                 // tile-uniform
    const bool inimg = px < W && py < H;                     // lanes outside the image stay for the warp-wide phases
    const size_t plane = (size_t)W * H;
    const size_t pix0 = (size_t)view * sc.k * plane + (size_t)py * W + px;
    const int4* __restrict__ vv = vtx + (size_t)view * sc.v_total;

    float Y[VS_MAX_COEF];
    float vx, vy, vz;
    vs_view_dir(cams[view], px, py, vx, vy, vz);
    vs_sh_basis<3>(vx, vy, vz, Y);

    // pass 1: forward, front to back
    uint32_t ids[VS_MAX_LAYERS];
    float rgb[VS_MAX_LAYERS][3], sig3[VS_MAX_LAYERS], aw[VS_MAX_LAYERS], Tl[VS_MAX_LAYERS];
    uint32_t used = 0;                       // layers that were composited (bit l)
    float Tr = 1.0f;
    bool alive = true;
    for (uint32_t l = 0; l < sc.k; ++l) {
        ids[l] = VS_MISS;
        if (!inimg || !((lmask >> l) & 1u)) continue;
        const unsigned long long key = vs_key_load(&keys[pix0 + (size_t)l * plane]);
        if (!key) continue;
        vs_key_clear(&keys[pix0 + (size_t)l * plane]);   // cleared for the next pass over this buffer, as k_shade does
        if (!alive) continue;
        const uint32_t lid = 0xFFFFFFFFu - (uint32_t)key;
        float s[4], uv[2];
        vs_plain_logits<F16>(sc, vv, l, lid, px, py, Y, s, uv);
        ids[l] = lid;
        rgb[l][0] = vs_sigmoid(s[0]); rgb[l][1] = vs_sigmoid(s[1]); rgb[l][2] = vs_sigmoid(s[2]);
        sig3[l] = vs_sigmoid(s[3]);
        aw[l] = fr.attenuate ? vs_alpha_w(vx, vy, vz, vs_fragment_normal(sc, vv, l, lid, px, py)) : 1.0f;
        Tl[l] = Tr;
        used |= 1u << l;
        Tr *= (1.0f - sig3[l] * aw[l]);
        if (Tr < fr.t_min) alive = false;
    }
    // pass 2: backward, back to front.  The owner lane runs the recurrence and leaves (texel offsets, bilinear weights,
    // dL/ds) of its fragment in the warp's slab; then the warp re-maps itself to 4 fragments x 8 lanes: octet `o` takes
    // the fragment of pixel row o, column j, and its lane i adds the coefficients c = i and c = 8 + i (a float4 of 4
    // channels each) of the four texels -- every reduction instruction covers whole 128-byte lines of the gradient
    // texture instead of 32 scattered 16-byte pieces.
    extern __shared__ __align__(16) unsigned char smem[];
    float* ysm = reinterpret_cast<float*>(smem + warp * 3584);                 // [pixel][16] SH basis
    uint4* rec_o = reinterpret_cast<uint4*>(smem + warp * 3584 + 2048);         // float4 index of the 4 texels' coefficient 0
    float4* rec_w = reinterpret_cast<float4*>(smem + warp * 3584 + 2560);       // bilinear weights (all 0: nothing to add)
    float4* rec_d = reinterpret_cast<float4*>(smem + warp * 3584 + 3072);       // dL/ds of the four channels
#pragma unroll
    for (int c = 0; c < 16; c += 4) reinterpret_cast<float4*>(ysm + lane * 16)[c >> 2] = make_float4(Y[c], Y[c + 1], Y[c + 2], Y[c + 3]);
    const uint32_t oct = lane >> 3, oi = lane & 7;
    float4 g = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    if (inimg) g = reinterpret_cast<const float4*>(grad_out)[((size_t)view * H + py) * W + px];
    float R = fr.bg[0] * g.x + fr.bg[1] * g.y + fr.bg[2] * g.z - g.w;
    for (int l = (int)sc.k - 1; l >= 0; --l) {
        const bool act = (used >> l) & 1u;
        if (__ballot_sync(0xFFFFFFFFu, act) == 0u) continue;   // warp-uniform
        uint4 ro = make_uint4(0, 0, 0, 0);
        float4 rw = make_float4(0.0f, 0.0f, 0.0f, 0.0f), rd = rw;
        if (act) {
            const float A = sig3[l] * aw[l];
            const float cg = rgb[l][0] * g.x + rgb[l][1] * g.y + rgb[l][2] * g.z;
            const float TA = Tl[l] * A;
            rd.x = TA * g.x * rgb[l][0] * (1.0f - rgb[l][0]);
            rd.y = TA * g.y * rgb[l][1] * (1.0f - rgb[l][1]);
            rd.z = TA * g.z * rgb[l][2] * (1.0f - rgb[l][2]);
            rd.w = Tl[l] * (cg - R) * aw[l] * sig3[l] * (1.0f - sig3[l]);
            R = A * cg + (1.0f - A) * R;
            // footprint of the fragment (same arithmetic as the forward)
            const uint4 tri = __ldg(&sc.tris[sc.tri_off[l] + ids[l]]);
            float u0, du, v0, dv;
            vs_fragment_uv(sc, vv, tri, px, py, u0, du, v0, dv);
            const int Wt = (int)sc.tex_w[l], Ht = (int)sc.tex_h[l];
            uint32_t cx0, cx1, cy0, cy1;
            float fa, fb;
            vs_texel_coord(u0, du, (float)Wt, Wt, cx0, cx1, fa);
            vs_texel_coord(v0, dv, (float)Ht, Ht, cy0, cy1, fb);
            const uint32_t nc = sc.n_coef;     // texel t starts at float4 index t * n_coef (< 2^32: checked at scene creation)
            ro = make_uint4((cy0 * Wt + cx0) * nc, (cy0 * Wt + cx1) * nc, (cy1 * Wt + cx0) * nc, (cy1 * Wt + cx1) * nc);
            rw = make_float4((1.0f - fa) * (1.0f - fb), fa * (1.0f - fb), (1.0f - fa) * fb, fa * fb);
        }
        rec_o[lane] = ro; rec_w[lane] = rw; rec_d[lane] = rd;
        __syncwarp();
        float4* __restrict__ gl = reinterpret_cast<float4*>(gt.p[l]);
#pragma unroll 2
        for (int j = 0; j < 8; ++j) {
            const uint32_t p = oct * 8 + j;       // owner lane of the fragment (pixel row oct, column j)
            const float4 w = rec_w[p];
            if (w.x == 0.0f && w.y == 0.0f && w.z == 0.0f && w.w == 0.0f) continue;
            uint4 o = rec_o[p];
#ifdef VS_BW_EXP_REDMASK   // timing experiment only (wrong gradients): the reductions stay inside a cache-resident window of float4s
            o.x &= (uint32_t)VS_BW_EXP_REDMASK; o.y &= (uint32_t)VS_BW_EXP_REDMASK; o.z &= (uint32_t)VS_BW_EXP_REDMASK; o.w &= (uint32_t)VS_BW_EXP_REDMASK;
#endif
            const float4 d = rec_d[p];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const uint32_t c = oi + 8 * h;
                if (c >= sc.n_coef) continue;
                const float y = ysm[p * 16 + c];
                float wy = w.x * y; vs_red_add4(reinterpret_cast<float*>(gl + o.x + c), wy * d.x, wy * d.y, wy * d.z, wy * d.w);
                wy = w.y * y;       vs_red_add4(reinterpret_cast<float*>(gl + o.y + c), wy * d.x, wy * d.y, wy * d.z, wy * d.w);
                wy = w.z * y;       vs_red_add4(reinterpret_cast<float*>(gl + o.z + c), wy * d.x, wy * d.y, wy * d.z, wy * d.w);
                wy = w.w * y;       vs_red_add4(reinterpret_cast<float*>(gl + o.w + c), wy * d.x, wy * d.y, wy * d.z, wy * d.w);
            }
        }
        __syncwarp();
    }
}

cudaError_t vs_launch_backward(const VsSceneDev& sc, int f16, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    dim3 grid(fr.tiles_x * fr.tiles_y, ch.views);
    const size_t smem = 8 * 3584;
    if (f16) k_backward<1><<<grid, 256, smem, st>>>(sc, fr, ch.cams, ch.vtx, ch.tile_mask, ch.keys, ch.grad_out, ch.grad_tex, ch.order);
    else k_backward<0><<<grid, 256, smem, st>>>(sc, fr, ch.cams, ch.vtx, ch.tile_mask, ch.keys, ch.grad_out, ch.grad_tex, ch.order);
    return cudaGetLastError();
}

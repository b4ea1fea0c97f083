// vs_plain.cuh -- plain (one thread per fragment, no cooperation) S5-S6 for every texture format: the four channel
// logits of the fragment of triangle `lid` of layer l at pixel (px, py).  Used by the brute-force kernel
// (VS_FLAG_REFERENCE_PATH) and by the per-layer render-buffer kernel (vs_render_aov); same arithmetic contract
// as the fast kernels, written for clarity first (16-byte texel loads, nothing else).
#pragma once
#include "vs_common.cuh"

template <int F16>
__device__ inline void vs_plain_logits(const VsSceneDev& sc, const int4* __restrict__ vv, uint32_t l, uint32_t lid, int px, int py,
                                       const float* Y, float* s, float* uv)
{
    const uint4 tri = __ldg(&sc.tris[sc.tri_off[l] + lid]);
    float u0, du, v0, dv;
    vs_fragment_uv(sc, vv, tri, px, py, u0, du, v0, dv);
    uv[0] = u0 + du; uv[1] = v0 + dv;
    s[0] = s[1] = s[2] = s[3] = 0.0f;
    if (sc.banded) {
        float ysum = 0.0f;
        for (uint32_t c = 0; c < sc.n_coef; ++c) ysum += Y[c];
        for (int ch = 0; ch < 4; ++ch) s[ch] = sc.v_min * ysum;
        for (uint32_t b = 0; b <= sc.sh_degree; ++b) {
            const int Wb = (int)sc.bw[l][b], Hb = (int)sc.bh[l][b];
            const uint32_t stride = VS_BAND_STRIDE(b);
            uint32_t cx0, cx1, cy0, cy1;
            float fa, fb;
            vs_texel_coord(u0, du, (float)Wb, Wb, cx0, cx1, fa);
            vs_texel_coord(v0, dv, (float)Hb, Hb, cy0, cy1, fb);
            const unsigned char* t[4] = {sc.btex[l][b] + (size_t)(cy0 * Wb + cx0) * stride, sc.btex[l][b] + (size_t)(cy0 * Wb + cx1) * stride,
                                         sc.btex[l][b] + (size_t)(cy1 * Wb + cx0) * stride, sc.btex[l][b] + (size_t)(cy1 * Wb + cx1) * stride};
            const float ws[4] = {(1.0f - fa) * (1.0f - fb), fa * (1.0f - fb), (1.0f - fa) * fb, fa * fb};
            for (uint32_t m = 0; m < 2 * b + 1; ++m)
                for (int ch = 0; ch < 4; ++ch) {
                    float v = 0.0f;
                    for (int q = 0; q < 4; ++q) v += ws[q] * (float)t[q][4 * m + ch];
                    s[ch] += Y[b * b + m] * (sc.v_scale * v);
                }
        }
        return;
    }
    VsFrag f;
    const int Wt = (int)sc.tex_w[l], Ht = (int)sc.tex_h[l];
    vs_texel_coord(u0, du, (float)Wt, Wt, f.cx0, f.cx1, f.a);
    vs_texel_coord(v0, dv, (float)Ht, Ht, f.cy0, f.cy1, f.b);
    const uint32_t nv = sc.texel_vecs;
    const uint32_t offs[4] = {(f.cy0 * Wt + f.cx0) * nv, (f.cy0 * Wt + f.cx1) * nv, (f.cy1 * Wt + f.cx0) * nv, (f.cy1 * Wt + f.cx1) * nv};
    const float ws[4] = {(1.0f - f.a) * (1.0f - f.b), f.a * (1.0f - f.b), (1.0f - f.a) * f.b, f.a * f.b};
    if (F16 && sc.frag_layout) {
        // mma A-fragment order (vs_common.cuh): vector v holds channels (v >> 2) and (v >> 2) + 2, coefficients 2t, 2t+1, 2t+8, 2t+9
#pragma unroll
        for (int v = 0; v < 8; ++v) {   // fully unrolled: every index below is a constant
            uint4 t[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) t[q] = __ldg(sc.tex[l] + offs[q] + v);
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const int ch = (v >> 2) + 2 * ((r >> 1) & 1), c = (v & 3) * 2 + (r & 1) + 8 * (r >> 2);
                float val = 0.0f;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const uint32_t w = (r >> 1) == 0 ? t[q].x : (r >> 1) == 1 ? t[q].y : (r >> 1) == 2 ? t[q].z : t[q].w;
                    const __half2 h = *reinterpret_cast<const __half2*>(&w);
                    val += ws[q] * ((r & 1) ? __high2float(h) : __low2float(h));
                }
                s[ch] += ((uint32_t)c < sc.n_coef ? Y[c] : 0.0f) * val;
            }
        }
        return;
    }
    // internal texel layout [ch][np_pad]: 16-byte vectors of consecutive coefficients of one channel
    const uint32_t vpc = nv >> 2;   // vectors per channel: 1, 2 or 4
#pragma unroll 1
    for (int ch = 0; ch < 4; ++ch) {
        // all vectors of this channel row of the four texels are requested before the first is used
        uint4 t[4][4];
#pragma unroll
        for (int v = 0; v < 4; ++v)
#pragma unroll
            for (int q = 0; q < 4; ++q)
                t[v][q] = (uint32_t)v < vpc ? __ldg(sc.tex[l] + offs[q] + ch * vpc + v) : make_uint4(0, 0, 0, 0);
        float acc = 0.0f;
#pragma unroll
        for (int v = 0; v < 4; ++v) {
            constexpr int EPV = F16 ? 8 : 4;
#pragma unroll
            for (int e = 0; e < EPV; ++e) {
                const int c = v * EPV + e;                     // zero padding adds 0
                if ((uint32_t)v >= vpc || c >= VS_MAX_COEF) continue;
                float val = 0.0f;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const int wi = F16 ? (e >> 1) : e;
                    const uint32_t w = wi == 0 ? t[v][q].x : wi == 1 ? t[v][q].y : wi == 2 ? t[v][q].z : t[v][q].w;
                    float tv;
                    if (F16) {
                        const __half2 h = *reinterpret_cast<const __half2*>(&w);
                        tv = (e & 1) ? __high2float(h) : __low2float(h);
                    } else {
                        tv = __uint_as_float(w);
                    }
                    val += ws[q] * tv;
                }
                acc += ((uint32_t)c < sc.n_coef ? Y[c] : 0.0f) * val;
            }
        }
        s[ch] = acc;
    }
}

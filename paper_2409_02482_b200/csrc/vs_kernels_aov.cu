// vs_kernels_aov.cu -- per-layer render buffers (PAPER.md:L763-803 supplement Fig. "render
// buffers": surface normals, surface UVs, surface opacity, surface colours of every layer).  An inspection output, not
// the hot path: one thread per (view, pixel) re-shades the winning fragment of every layer from the triangle-id planes
// with the plain per-fragment routine (vs_plain.cuh) and writes what the compositor would have consumed.
#include "vs_common.cuh"
#include "vs_plain.cuh"

template <int F16>
__global__ void __launch_bounds__(128)
k_layer_aov(const VsSceneDev sc, const VsFrame fr, const VsCamDev* __restrict__ cams, const int4* __restrict__ vtx,
            const uint32_t* __restrict__ ids, float* __restrict__ layer_rgba, float* __restrict__ layer_uv, float* __restrict__ layer_normal)
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
    for (uint32_t l = 0; l < sc.k; ++l) {
        const size_t o = (((size_t)view * sc.k + l) * H + py) * W + px;
        const uint32_t lid = ids[o];
        float4 rgba = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        float uv[2] = {0.0f, 0.0f};
        float4 n = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (lid != VS_MISS) {
            float s[4];
            vs_plain_logits<F16>(sc, vv, l, lid, px, py, Y, s, uv);
            n = vs_fragment_normal(sc, vv, l, lid, px, py);
            float A = vs_sigmoid(s[3]);
            if (fr.attenuate) A *= vs_alpha_w(vx, vy, vz, n);
            rgba = make_float4(vs_sigmoid(s[0]), vs_sigmoid(s[1]), vs_sigmoid(s[2]), A);
            if (vx * n.x + vy * n.y + vz * n.z > 0.0f) { n.x = -n.x; n.y = -n.y; n.z = -n.z; }   // face the viewer
        }
        if (layer_rgba) reinterpret_cast<float4*>(layer_rgba)[o] = rgba;
        if (layer_uv) reinterpret_cast<float2*>(layer_uv)[o] = make_float2(uv[0], uv[1]);
        if (layer_normal) { layer_normal[3 * o] = n.x; layer_normal[3 * o + 1] = n.y; layer_normal[3 * o + 2] = n.z; }
    }
}

cudaError_t vs_launch_layer_aov(const VsSceneDev& sc, int f16, const VsFrame& fr, uint32_t views, const VsCamDev* cams, const int4* vtx,
                                const uint32_t* ids, float* layer_rgba, float* layer_uv, float* layer_normal, cudaStream_t st)
{
    dim3 grid((fr.width + 15) / 16, (fr.height + 7) / 8, views);
    if (f16) k_layer_aov<1><<<grid, 128, 0, st>>>(sc, fr, cams, vtx, ids, layer_rgba, layer_uv, layer_normal);
    else k_layer_aov<0><<<grid, 128, 0, st>>>(sc, fr, cams, vtx, ids, layer_rgba, layer_uv, layer_normal);
    return cudaGetLastError();
}

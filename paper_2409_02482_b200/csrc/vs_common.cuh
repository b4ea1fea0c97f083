// vs_common.cuh -- shared declarations of the CUDA path (never included by oracle/).
// Arithmetic contract: DESIGN.md §3 (fp32-exact steps use the _rn intrinsics, which nvcc never
// contracts or relaxes; integer steps are exact by construction).
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>

#define VS_MAX_LAYERS 9
#define VS_MAX_COEF 16
#define VS_TILE_W 16
#define VS_TILE_H 16
#define VS_TILE_PIX (VS_TILE_W * VS_TILE_H)
#define VS_MISS 0xFFFFFFFFu
#ifndef VS_ORDER_BITS
#define VS_ORDER_BITS 6        // surface-order sort keys: cells per axis of the octahedral map = 2^VS_ORDER_BITS (5..8 measure the same)
#endif
#ifndef VS_ORDER_MODE
#define VS_ORDER_MODE 1        // 1: Hilbert index of the octahedral map of the direction from the box centre; 0: Morton code of a 32^3 cell
#endif
#define VS_ORDER_BINS ((VS_ORDER_MODE == 0 ? 32768u : (1u << (2 * VS_ORDER_BITS))) + 1u)   // + one bin for "nothing at the probes"

// Device-side description of an immutable scene (passed by value to kernels).
struct VsSceneDev {
    const float* positions;   // [v_total][3], all layers concatenated
    const float2* uvs;        // [v_total]
    const uint4* tris;        // [t_total] {i0, i1, i2 : global vertex index, w : layer << 28 | index of the triangle in its layer}
    const float4* tri_nrm;    // [t_total] unit geometric normal in world space (fp64 cross product rounded to fp32), w = 0;
                              //           zero vector for zero-area triangles.  Read only under VS_FLAG_ATTENUATION
    const float4* vtx_nrm;    // [v_total] optional per-vertex normals (vs_scene_set_vertex_normals), w = 0; nullptr if none
    uint32_t vnrm_mask;       // bit l: layer l has per-vertex normals (the attenuation then uses the interpolated normal)
    uint32_t v_total, t_total;
    uint32_t k, sh_degree, n_coef;
    uint32_t texel_vecs;                  // 16-byte vectors per texel in the internal layout (= 4 * np_pad * elem / 16)
    uint32_t np_pad;                      // coefficients per channel row of the internal layout [texel][ch][np_pad]
    uint32_t frag_layout;                 // 1: fp16 texels of 16 (padded) coefficients stored in mma A-fragment order (see below)
    float bb_min[3], bb_scale[3];         // object-space bounding box of all vertices: cell = (p - bb_min) * bb_scale in [0, 32) (vs_kernels_order.cu)
    uint32_t tri_off[VS_MAX_LAYERS + 1];  // global triangle id of each layer's triangle 0
    uint32_t vtx_off[VS_MAX_LAYERS + 1];  // global vertex index of each layer's vertex 0
    const uint4* tex[VS_MAX_LAYERS];      // [tex_h][tex_w][texel_vecs] 16-byte vectors
    uint32_t tex_w[VS_MAX_LAYERS], tex_h[VS_MAX_LAYERS];
    uint32_t tex_bit_off[VS_MAX_LAYERS + 1];  // VS_FLAG_COUNT_TEXELS: first bitmap bit of each layer (multiple of 32)
    // banded 8-bit scenes (vs_scene_create_banded): band b of layer l is [bh][bw] texels of
    // VS_BAND_STRIDE(b) = {4, 16, 32, 32} bytes holding its (2b+1) x 4 bytes in API order, zero padded
    uint32_t banded;
    float v_min, v_scale;                      // sh = v_min + v_scale * byte, v_scale = (v_max - v_min) / 255
    const unsigned char* btex[VS_MAX_LAYERS][4];
    uint32_t bw[VS_MAX_LAYERS][4], bh[VS_MAX_LAYERS][4];
};
#define VS_BAND_STRIDE(b) ((b) == 0 ? 4u : (b) == 1 ? 16u : 32u)

struct VsCamDev {  // == vs_camera
    float fx, fy, cx, cy;
    float R[9];
    float t[3];
};

struct VsFrame {
    uint32_t width, height, tiles_x, tiles_y;
    float near_plane, t_min;
    float bg[3];
    uint32_t attenuate;       // VS_FLAG_ATTENUATION: opacity *= alpha_w(view direction, face normal)
};

// counters[0] dropped, [1] degenerate, [2] tile refs, [3] shaded fragments, [4] unique texels,
// [5] max over chunks of the references a chunk needed when that exceeded ref_capacity (0 = no overflow)
enum { VS_CNT_DROPPED = 0, VS_CNT_DEGENERATE = 1, VS_CNT_REFS = 2, VS_CNT_FRAGS = 3, VS_CNT_TEXELS = 4, VS_CNT_OVERFLOW = 5, VS_CNT_N = 8 };

__host__ __device__ inline uint32_t vs_tri_layer(uint32_t w) { return w >> 28; }
__host__ __device__ inline uint32_t vs_tri_lid(uint32_t w) { return w & 0x0FFFFFFFu; }

// ---- packed fp32 pairs (sm_100: FADD2 / FMUL2 / FFMA2 issue one instruction for two lanes' worth of fp32 work) ----
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 vs_pack2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void vs_unpack2(f32x2 v, float& lo, float& hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 vs_fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f32x2 vs_mul2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 vs_add2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}

// ---- triangle setup shared by the binning, raster and shading kernels ----------
struct VsTri {
    int X0, Y0, X1, Y1, X2, Y2;
    float q0, q1, q2;
    long long A2;
    bool swapped;  // vertices 1 and 2 were exchanged to make A2 > 0
};

// vtx record = {X, Y, float_as_int(q), bad}
__device__ __forceinline__ int vs_setup_tri(const int4& a, const int4& b, const int4& c, VsTri& t)
{
    if ((a.w | b.w | c.w) != 0) return 1;  // behind the near plane or off the guard band: dropped
    long long A2 = (long long)(b.x - a.x) * (long long)(c.y - a.y) - (long long)(c.x - a.x) * (long long)(b.y - a.y);
    if (A2 == 0) return 2;
    t.X0 = a.x; t.Y0 = a.y; t.q0 = __int_as_float(a.z);
    if (A2 < 0) {
        t.X1 = c.x; t.Y1 = c.y; t.q1 = __int_as_float(c.z);
        t.X2 = b.x; t.Y2 = b.y; t.q2 = __int_as_float(b.z);
        t.A2 = -A2; t.swapped = true;
    } else {
        t.X1 = b.x; t.Y1 = b.y; t.q1 = __int_as_float(b.z);
        t.X2 = c.x; t.Y2 = c.y; t.q2 = __int_as_float(c.z);
        t.A2 = A2; t.swapped = false;
    }
    return 0;
}

// Pixel range whose sample points 256 i + 128 fall inside the triangle's bounding box, clipped to
// [0, w-1] x [0, h-1].  Returns false if empty.
__device__ __forceinline__ bool vs_tri_pixel_bbox(const VsTri& t, int w, int h, int& i0, int& i1, int& j0, int& j1)
{
    int minX = min(t.X0, min(t.X1, t.X2)), maxX = max(t.X0, max(t.X1, t.X2));
    int minY = min(t.Y0, min(t.Y1, t.Y2)), maxY = max(t.Y0, max(t.Y1, t.Y2));
    i0 = max((minX + 127) >> 8, 0);      // ceil((minX - 128) / 256)
    i1 = min((maxX - 128) >> 8, w - 1);  // floor((maxX - 128) / 256)
    j0 = max((minY + 127) >> 8, 0);
    j1 = min((maxY - 128) >> 8, h - 1);
    return i0 <= i1 && j0 <= j1;
}

// Edge functions at the sample point of pixel (i, j): e0 = 1->2 weights vertex 0,
// e1 = 2->0 weights vertex 1, e2 = 0->1 weights vertex 2.
struct VsEdges {
    long long E0, E1, E2;
};

__device__ __forceinline__ long long vs_edge(int Xa, int Ya, int Xb, int Yb, int Sx, int Sy)
{
    return (long long)(Xb - Xa) * (long long)(Sy - Ya) - (long long)(Yb - Ya) * (long long)(Sx - Xa);
}

__device__ __forceinline__ bool vs_topleft(int Xa, int Ya, int Xb, int Yb)
{
    int dx = Xb - Xa, dy = Yb - Ya;
    return (dy < 0) || (dy == 0 && dx > 0);
}

__device__ __forceinline__ void vs_edges_at(const VsTri& t, int i, int j, VsEdges& e)
{
    int Sx = 256 * i + 128, Sy = 256 * j + 128;
    e.E0 = vs_edge(t.X1, t.Y1, t.X2, t.Y2, Sx, Sy);
    e.E1 = vs_edge(t.X2, t.Y2, t.X0, t.Y0, Sx, Sy);
    e.E2 = vs_edge(t.X0, t.Y0, t.X1, t.Y1, Sx, Sy);
}

// Top-left biases: covered <=> E_e + bias_e > 0 with bias = 0 for top/left edges, -1... expressed as
// E_e >= min_e where min_e = 0 if the edge owns its samples, else 1.
__device__ __forceinline__ void vs_edge_mins(const VsTri& t, int& m0, int& m1, int& m2)
{
    m0 = vs_topleft(t.X1, t.Y1, t.X2, t.Y2) ? 0 : 1;
    m1 = vs_topleft(t.X2, t.Y2, t.X0, t.Y0) ? 0 : 1;
    m2 = vs_topleft(t.X0, t.Y0, t.X1, t.Y1) ? 0 : 1;
}

// Depth key, fp32-exact: qp = fma(f2,q2, fma(f1,q1, f0*q0)) / fA
__device__ __forceinline__ float vs_depth_q(const VsTri& t, long long E0, long long E1, long long E2)
{
    float f0 = __ll2float_rn(E0), f1 = __ll2float_rn(E1), f2 = __ll2float_rn(E2);
    float fA = __ll2float_rn(t.A2);
    float num = __fmaf_rn(f2, t.q2, __fmaf_rn(f1, t.q1, __fmul_rn(f0, t.q0)));
    return __fdiv_rn(num, fA);
}

__device__ __forceinline__ unsigned long long vs_make_key(float qp, uint32_t local_tri)
{
    return ((unsigned long long)__float_as_uint(qp) << 32) | (unsigned long long)(0xFFFFFFFFu - local_tri);
}

// The last stage's read-and-clear of the key image (k_shade, k_backward).  VS_KEYS_STREAM: 1 = evict-first cache hints on both
// (a key line is touched once per pass and only competes with the texels for L2), 0 = plain accesses.
#ifndef VS_KEYS_STREAM
#define VS_KEYS_STREAM 0
#endif
__device__ __forceinline__ unsigned long long vs_key_load(const unsigned long long* p)
{
#if VS_KEYS_STREAM
    return __ldcs(p);
#else
    return *p;
#endif
}
__device__ __forceinline__ void vs_key_clear(unsigned long long* p)
{
#if VS_KEYS_STREAM
    __stcs(p, 0ull);
#else
    *p = 0ull;
#endif
}

// Real SH basis, fp32, tolerance domain.
template <int DEG>
__device__ __forceinline__ void vs_sh_basis(float x, float y, float z, float* Y)
{
    Y[0] = 0.28209479177387814f;
    if (DEG >= 1) {
        Y[1] = 0.4886025119029199f * y;
        Y[2] = 0.4886025119029199f * z;
        Y[3] = 0.4886025119029199f * x;
    }
    if (DEG >= 2) {
        float xx = x * x, yy = y * y, zz = z * z;
        Y[4] = 1.0925484305920792f * x * y;
        Y[5] = 1.0925484305920792f * y * z;
        Y[6] = 0.31539156525252005f * (3.0f * zz - 1.0f);
        Y[7] = 1.0925484305920792f * x * z;
        Y[8] = 0.5462742152960396f * (xx - yy);
        if (DEG >= 3) {
            Y[9] = 0.5900435899266435f * y * (3.0f * xx - yy);
            Y[10] = 2.890611442640554f * x * y * z;
            Y[11] = 0.4570457994644658f * y * (5.0f * zz - 1.0f);
            Y[12] = 0.3731763325901154f * z * (5.0f * zz - 3.0f);
            Y[13] = 0.4570457994644658f * x * (5.0f * zz - 1.0f);
            Y[14] = 1.445305721320277f * z * (xx - yy);
            Y[15] = 0.5900435899266435f * x * (xx - 3.0f * yy);
        }
    }
}

// Unit view direction of pixel (i, j), world frame (DESIGN.md §3.7 / reading Q4).
__device__ __forceinline__ void vs_view_dir(const VsCamDev& c, int i, int j, float& x, float& y, float& z)
{
    float dx = ((float)i + 0.5f - c.cx) / c.fx;
    float dy = ((float)j + 0.5f - c.cy) / c.fy;
    float wx = c.R[0] * dx + c.R[3] * dy + c.R[6];
    float wy = c.R[1] * dx + c.R[4] * dy + c.R[7];
    float wz = c.R[2] * dx + c.R[5] * dy + c.R[8];
    float inv = rsqrtf(wx * wx + wy * wy + wz * wz);
    x = wx * inv; y = wy * inv; z = wz * inv;
}

__device__ __forceinline__ float vs_sigmoid(float s)
{
    return __fdividef(1.0f, 1.0f + __expf(-s));
}

// transparency attenuation alpha_w = 2 Sigmoid(10 |v . n|) - 1; v, n unit (n may be 0)
__device__ __forceinline__ float vs_alpha_w(float vx, float vy, float vz, const float4 n)
{
    const float d = fabsf(fmaf(vx, n.x, fmaf(vy, n.y, vz * n.z)));
    return fmaf(2.0f, vs_sigmoid(10.0f * d), -1.0f);
}

// ---- fragment setup (S5 addressing): winning triangle of a layer at pixel
// (px, py) -> clamped texel columns / rows of the 2x2 footprint and the bilinear fractions.
struct VsFrag {
    uint32_t cx0, cx1, cy0, cy1;
    float a, b;
};

__device__ __forceinline__ void vs_texel_coord(float u0, float du, float fW, int Wt, uint32_t& c0, uint32_t& c1, float& frac)
{
    // texel coordinate = (u0 W - 0.5) + du W, carried as integer + fraction so that the fraction
    // keeps full fp32 resolution at 4096^2 (u0 W is split into its rounded product and the FMA residual)
    const float ph = __fmul_rn(u0, fW), pl = __fmaf_rn(u0, fW, -ph);
    const float x0 = fminf(fmaxf(ph - 0.5f, -1048576.0f), 1048576.0f);
    const float fl = floorf(x0);
    const float t = ((x0 - fl) + pl) + du * fW;
    const float ft = floorf(t);
    frac = t - ft;
    const int i0 = __float2int_rd(fl) + __float2int_rd(ft);
    c0 = (uint32_t)min(max(i0, 0), Wt - 1);
    c1 = (uint32_t)min(max(i0 + 1, 0), Wt - 1);
}

// Perspective-correct barycentrics b'_1, b'_2 of the sample of pixel (px, py) in the triangle of the transformed vertices a, b, c
// (b'_i ~ E_i q_i).  The oracle orients the triangle first (swap of vertices 1, 2 when A2 < 0); without the swap
// every E_i changes sign, and so do the g_i and their sum: the quotients are the same bit for bit, so the setup is skipped here.
__device__ __forceinline__ void vs_barycentrics3(const int4& a, const int4& b, const int4& c, int px, int py, float& b0, float& b1, float& b2)
{
    const int Sx = 256 * px + 128, Sy = 256 * py + 128;
    // The sample lies inside the triangle (it is the fragment's own pixel), so every difference below is bounded by the
    // triangle's extent: if that is < 2^12 sub-pixel units (16 px) per axis, the products are < 2^25 and the edge functions
    // are the same integers in int32 arithmetic (2 IMAD + I2F each instead of 64-bit products and I2F.S64).
    const int ex = max(abs(b.x - a.x), max(abs(c.x - a.x), abs(c.x - b.x))), ey = max(abs(b.y - a.y), max(abs(c.y - a.y), abs(c.y - b.y)));
    float f0, f1, f2;
    if ((ex | ey) < 4096) {
        const int rx = Sx - a.x, ry = Sy - a.y;                        // sample relative to vertex a
        const int bx = b.x - a.x, by = b.y - a.y, cx = c.x - a.x, cy = c.y - a.y;
        const int E1 = cy * rx - cx * ry;                              // edge c -> a at S: (a - c) x (S - c) == c x r  (relative to a)
        const int E2 = bx * ry - by * rx;                              // edge a -> b at S
        const int A2 = bx * cy - cx * by;                              // E0 + E1 + E2 == A2 at every point
        f0 = __int2float_rn(A2 - E1 - E2); f1 = __int2float_rn(E1); f2 = __int2float_rn(E2);
    } else {
        f0 = __ll2float_rn(vs_edge(b.x, b.y, c.x, c.y, Sx, Sy)); f1 = __ll2float_rn(vs_edge(c.x, c.y, a.x, a.y, Sx, Sy));
        f2 = __ll2float_rn(vs_edge(a.x, a.y, b.x, b.y, Sx, Sy));
    }
    const float g0 = f0 * __int_as_float(a.z), g1 = f1 * __int_as_float(b.z), g2 = f2 * __int_as_float(c.z);
    const float inv = __fdividef(1.0f, g0 + g1 + g2);
    b0 = g0 * inv; b1 = g1 * inv; b2 = g2 * inv;
}
__device__ __forceinline__ void vs_barycentrics(const int4& a, const int4& b, const int4& c, int px, int py, float& b1, float& b2)
{
    float b0;
    vs_barycentrics3(a, b, c, px, py, b0, b1, b2);
}

// Normal of the fragment of triangle `lid` of layer l at pixel (px, py) for the transparency attenuation and the normal buffer
// (DESIGN.md §3.9): the unit face normal, or -- if the layer was given per-vertex normals (vs_scene_set_vertex_normals) -- the
// three vertex normals interpolated with the fragment's perspective-correct barycentrics and renormalised (0 if the sum vanishes).
__device__ __forceinline__ float4 vs_fragment_normal(const VsSceneDev& sc, const int4* __restrict__ vv, uint32_t l, uint32_t lid, int px, int py)
{
    if (!((sc.vnrm_mask >> l) & 1u)) return __ldg(&sc.tri_nrm[sc.tri_off[l] + lid]);
    const uint4 tri = __ldg(&sc.tris[sc.tri_off[l] + lid]);
    float b0, b1, b2;
    vs_barycentrics3(__ldg(&vv[tri.x]), __ldg(&vv[tri.y]), __ldg(&vv[tri.z]), px, py, b0, b1, b2);
    const float4 n0 = __ldg(&sc.vtx_nrm[tri.x]), n1 = __ldg(&sc.vtx_nrm[tri.y]), n2 = __ldg(&sc.vtx_nrm[tri.z]);
    const float x = b0 * n0.x + b1 * n1.x + b2 * n2.x, y = b0 * n0.y + b1 * n1.y + b2 * n2.y, z = b0 * n0.z + b1 * n1.z + b2 * n2.z;
    const float len2 = x * x + y * y + z * z;
    const float inv = len2 > 0.0f ? rsqrtf(len2) : 0.0f;
    return make_float4(x * inv, y * inv, z * inv, 0.0f);
}

// `tri` = index record of the winning triangle of layer l
__device__ __forceinline__ void vs_fragment_setup_tri(const VsSceneDev& sc, const int4* __restrict__ vv, uint32_t l,
                                                      const uint4 tri, int px, int py, VsFrag& f)
{
    const int4 a = __ldg(&vv[tri.x]), b = __ldg(&vv[tri.y]), c = __ldg(&vv[tri.z]);
    const float2 uv0 = __ldg(&sc.uvs[tri.x]), uv1 = __ldg(&sc.uvs[tri.y]), uv2 = __ldg(&sc.uvs[tri.z]);
    float b1, b2;
    vs_barycentrics(a, b, c, px, py, b1, b2);
    const int Wt = (int)sc.tex_w[l], Ht = (int)sc.tex_h[l];
    vs_texel_coord(uv0.x, b1 * (uv1.x - uv0.x) + b2 * (uv2.x - uv0.x), (float)Wt, Wt, f.cx0, f.cx1, f.a);
    vs_texel_coord(uv0.y, b1 * (uv1.y - uv0.y) + b2 * (uv2.y - uv0.y), (float)Ht, Ht, f.cy0, f.cy1, f.b);
}

__device__ __forceinline__ void vs_fragment_setup(const VsSceneDev& sc, const int4* __restrict__ vv, uint32_t l,
                                                  uint32_t local_tri, int px, int py, VsFrag& f)
{
    vs_fragment_setup_tri(sc, vv, l, __ldg(&sc.tris[sc.tri_off[l] + local_tri]), px, py, f);
}

// perspective-correct UV of the winning triangle at the pixel, as base + offset
__device__ __forceinline__ void vs_fragment_uv(const VsSceneDev& sc, const int4* __restrict__ vv, const uint4 tri, int px, int py,
                                               float& u0, float& du, float& v0, float& dv)
{
    const int4 a = __ldg(&vv[tri.x]), b = __ldg(&vv[tri.y]), c = __ldg(&vv[tri.z]);
    const float2 uva = __ldg(&sc.uvs[tri.x]), uv1 = __ldg(&sc.uvs[tri.y]), uv2 = __ldg(&sc.uvs[tri.z]);
    float b1, b2;
    vs_barycentrics(a, b, c, px, py, b1, b2);
    u0 = uva.x; du = b1 * (uv1.x - uva.x) + b2 * (uv2.x - uva.x);
    v0 = uva.y; dv = b1 * (uv1.y - uva.y) + b2 * (uv2.y - uva.y);
}

// ---- host-side launchers (vs_kernels_*.cu) ------------------------------------------------------
struct VsGradTex { float* p[VS_MAX_LAYERS]; };   // per layer [tex_h][tex_w][n_coef][4] fp32 gradient accumulators (API texture layout)

struct VsChunk {                 // one pass over `views` cameras
    uint32_t views;
    const VsCamDev* cams;        // DEVICE [views]
    int4* vtx;                   // DEVICE [views][v_total]
    uint32_t* tri_tiles;         // DEVICE [views][t_total] packed tile range of each triangle (count pass output)
    uint32_t* tile_count;        // DEVICE [views * tiles]   (count pass output)
    uint32_t* tile_off;          // DEVICE [views * tiles + 1] exclusive scan; [views*tiles] = total references
    uint32_t* tile_cursor;       // DEVICE [views * tiles]   scatter cursors
    uint32_t* tile_tris;         // DEVICE [ref_capacity]
    uint32_t ref_capacity;       // entries of tile_tris; references past it are dropped and flagged
    unsigned long long* counters;  // DEVICE [VS_CNT_N]
    uint32_t* ids;               // DEVICE [views][k][H][W] nearest triangle per (pixel, layer)
    int ids_is_output;           // ids is the caller's AOV: empty tiles must be filled with MISS too
    float* out_rgba;             // DEVICE [views][H][W][4]
    uint32_t* texel_bits;        // DEVICE [views][tex_bit_off[k] / 32] or nullptr (VS_FLAG_COUNT_TEXELS)
    const float* grad_out;       // DEVICE [views][H][W][4] upstream gradient: vs_render_backward runs k_backward instead of k_shade
    VsGradTex grad_tex;
    int count_fragments;         // banded scenes under VS_FLAG_COUNT_TEXELS: count shaded fragments only
    // direct (untiled) path: non-null keys selects it in vs_launch_shade
    unsigned long long* keys;    // DEVICE [views][k][H][W] max keys, zero between passes
    uint2* big_list;             // DEVICE [big_capacity] {view, global triangle} with very large boxes
    uint32_t* big_count;         // DEVICE entries appended this chunk (may exceed big_capacity: the rest was done in place)
    uint32_t big_capacity;
    uint32_t* tile_mask;         // DEVICE [views][tiles] layers whose triangles' boxes touch the 16x16 tile (zero on entry)
    const uint32_t* order;       // DEVICE [views * tiles] (view * tiles + tile) in shading order, or nullptr = screen order
};

cudaError_t vs_launch_transform(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st);
cudaError_t vs_launch_bin_count(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st);
cudaError_t vs_launch_bin_scan(const VsFrame& fr, const VsChunk& ch, cudaStream_t st);
cudaError_t vs_launch_bin_scatter(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st);
cudaError_t vs_launch_raster_direct(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st, uint32_t resident_ctas);
cudaError_t vs_launch_raster(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st);
cudaError_t vs_launch_shade(const VsSceneDev& sc, int tex_f16, const VsFrame& fr, const VsChunk& ch, cudaStream_t st);
cudaError_t vs_launch_order(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, uint32_t* order, uint32_t* work, cudaStream_t st);
cudaError_t vs_launch_bbox(const float* pos, uint32_t n_vertices, int* bb6, cudaStream_t st);
cudaError_t vs_launch_popcount(const uint32_t* words, size_t n, unsigned long long* counter, cudaStream_t st);
cudaError_t vs_launch_reference(const VsSceneDev& sc, int tex_f16, const VsFrame& fr, const VsChunk& ch, cudaStream_t st);

// scene construction helpers
cudaError_t vs_launch_pack_tris(const uint32_t* indices, const float* layer_positions, uint32_t num_tris, uint32_t num_vertices,
                                uint32_t vtx_off, uint32_t layer, uint4* out, float4* out_normals, uint32_t* error_flag, cudaStream_t st);
cudaError_t vs_launch_pack_band(const unsigned char* src, uint32_t n_texels, uint32_t band, unsigned char* dst, cudaStream_t st);
cudaError_t vs_launch_shade_banded(const VsSceneDev& sc, const VsFrame& fr, const struct VsChunk& ch, cudaStream_t st);
cudaError_t vs_launch_backward(const VsSceneDev& sc, int f16, const VsFrame& fr, const VsChunk& ch, cudaStream_t st);
cudaError_t vs_launch_shade_backward(const VsSceneDev& sc, int f16, const VsFrame& fr, const VsChunk& ch, cudaStream_t st);
cudaError_t vs_launch_layer_aov(const VsSceneDev& sc, int f16, const VsFrame& fr, uint32_t views, const VsCamDev* cams, const int4* vtx,
                                const uint32_t* ids, float* layer_rgba, float* layer_uv, float* layer_normal, cudaStream_t st);
cudaError_t vs_launch_check_finite(const float* v, size_t n, uint32_t* error_flag, cudaStream_t st);
cudaError_t vs_launch_pack_normals(const float* src, uint32_t n, float4* dst, cudaStream_t st);
cudaError_t vs_launch_pack_texture(const void* src, int f16, uint32_t n_texels, uint32_t n_coef, uint32_t np_pad, uint32_t frag_layout,
                                   uint4* dst, cudaStream_t st);

// Internal texel layout: [texel][ch = 0..3][np_pad] elements, channel-major, every channel row
// padded to np_pad = 16-byte vectors-per-channel (1, 2 or 4) * elements per vector coefficients.
// fp16 textures with np_pad == 16 (SH degree 2 and 3; VsSceneDev::frag_layout) permute the 64 halves of a texel into the
// A-fragment order of mma.sync.m16n8k16 instead, so that lane oi = 0..7 of an octet loads the four registers of its A
// fragment as ONE 16-byte vector: vector v = (ch & 1) * 4 + ((c & 7) >> 1), half ((c >> 3) * 2 + (ch >> 1)) * 2 + (c & 1)
// of that vector (A row = 2 f + (ch & 1) + 8 (ch >> 1) for the fragment f of the octet, A column = c).
__host__ __device__ inline uint32_t vs_frag_half_index(uint32_t c, uint32_t ch)
{
    return ((ch & 1u) * 4u + ((c & 7u) >> 1)) * 8u + ((c >> 3) * 2u + (ch >> 1)) * 2u + (c & 1u);
}
__host__ __device__ inline uint32_t vs_vecs_per_channel(int f16, uint32_t n_coef)
{
    const uint32_t epv = f16 ? 8u : 4u;
    const uint32_t v = (n_coef + epv - 1u) / epv;
    return v <= 1u ? 1u : (v == 2u ? 2u : 4u);
}

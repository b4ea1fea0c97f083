// vs_kernels_shade.cu -- S5 perspective-correct UV + bilinear texel fetch, S6 SH evaluation + sigmoid,
// S7 fixed-order front-to-back compositing.  DESIGN.md §1, §3.5-3.8, §6, §7.
//
// One CTA per (view, 16x16 tile), a warp owns an 8x4 pixel block, lane = pixel ("owner").
// Phase A: every owner turns the winning triangle of each layer (the id planes k_raster wrote) into
//   a packed fragment record (clamped texel column/row of the 2x2 footprint + the two bilinear
//   fractions) in shared memory.  The gather chain id -> triangle -> 3 vertices + 3 uvs is paid once
//   per tile, three layers at a time, instead of once per layer inside the shading loop.
// Phase B: per layer the warp re-maps itself to 4 fragments x 8 lanes.  Octet `o` streams the four
//   texels of the fragment of pixel row `o`, column `j`, as 16-byte vectors: the internal texel layout
//   is channel-major ([ch][coefficient]), so a lane's vector holds 8 (fp16) / 4 (fp32)
//   consecutive coefficients of ONE channel and an octet reads one full 128-byte line per texel at SH
//   degree 3 / fp16.  The loads of column j+1 are issued before the arithmetic of column j (software
//   pipeline).  A lane blends its coefficients with the bilinear weights and dots them with the pixel's
//   SH basis (staged once per pixel in shared memory, shared by all layers) using packed fp32 FMAs
//   (fma.rn.f32x2 -> FFMA2); the one or two lanes of a channel are summed with one shuffle and the
//   four channel logits go back to the owner through shared memory.  Owners apply the sigmoid and
//   composite front to back in registers.
#include "vs_common.cuh"

struct __align__(16) VsFragRec {
    uint32_t o00, o01, o10, o11;  // 16-byte-vector offsets of the four texels inside the layer texture
    float w00, w01, w10, w11;     // bilinear weights (all 0: no fragment)
};

#ifndef VS_SHADE_PREFETCH
#define VS_SHADE_PREFETCH 2   // 0: off, 1: left column of the footprint, 2: all four texels (screen order only), 3: all four, in surface order too
#endif
#ifndef VS_SHADE_PF_DIST
#define VS_SHADE_PF_DIST 1    // layers between the prefetch of a footprint and its use
#endif
__device__ __forceinline__ void vs_prefetch_l2(const void* p)
{
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}
#ifndef VS_SHADE_PFMODE
#define VS_SHADE_PFMODE 0     // 0: one prefetch.global.L2 per texel; 1: one bulk prefetch per footprint row; 2: same, 256-byte aligned blocks
#endif
__device__ __forceinline__ void vs_prefetch_l2_bulk(const void* p, uint32_t bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes));
}
__device__ __forceinline__ uint4 vs_ldg_tex(const char* base, uint32_t vec_off, int slot)
{
#ifdef VS_EXP_TEXMASK   // timing experiment only (wrong images): confine the texel addresses to a cache-resident window
    vec_off &= (uint32_t)VS_EXP_TEXMASK;
#endif
    const uint4* p = reinterpret_cast<const uint4*>(base + (unsigned long long)vec_off * 16ull) + slot;
#ifdef VS_SHADE_LD256
    uint4 r;
    asm volatile("ld.global.nc.L2::256B.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
#else
    return __ldg(p);
#endif
}

// element pair q (0..3 for fp16, 0..1 for fp32) of a 16-byte texel vector as packed fp32
template <int F16>
__device__ __forceinline__ f32x2 vs_pair(const uint4& t, int q)
{
    if (F16) {
        const uint32_t w = q == 0 ? t.x : q == 1 ? t.y : q == 2 ? t.z : t.w;
        const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&w));
        return vs_pack2(f.x, f.y);
    } else {
        return q == 0 ? vs_pack2(__uint_as_float(t.x), __uint_as_float(t.y)) : vs_pack2(__uint_as_float(t.z), __uint_as_float(t.w));
    }
}

// packed record: cx0 | (cx1 != cx0) << 15 | cy0 << 16 | (cy1 != cy0) << 31  (texture sides <= 32768)
__device__ __forceinline__ uint32_t vs_pack_frag(const VsFrag& f)
{
    return f.cx0 | ((f.cx1 != f.cx0) ? 0x8000u : 0u) | (f.cy0 << 16) | ((f.cy1 != f.cy0) ? 0x80000000u : 0u);
}

// compile-time shape of the octet mapping for a texture format (must agree with vs_vecs_per_channel)
template <int F16, int DEG>
struct VsShadeShape {
    static constexpr int NCOEF = (DEG + 1) * (DEG + 1);
    static constexpr int EPV = F16 ? 8 : 4;                            // elements per 16-byte vector
    static constexpr int VPC0 = (NCOEF + EPV - 1) / EPV;
    static constexpr int VPC = VPC0 <= 1 ? 1 : (VPC0 == 2 ? 2 : 4);     // vectors per channel row
    static constexpr int NVEC = 4 * VPC;                               // vectors per texel (== sc.texel_vecs)
    static constexpr int SLOTS = NVEC > 8 ? NVEC / 8 : 1;              // vectors per octet lane
    static constexpr int LPC = VPC / SLOTS;                            // lanes per channel (1 or 2)
    static constexpr int NACT = NVEC / SLOTS;                          // octet lanes that hold data (4 or 8)
    static constexpr int NE = SLOTS * EPV;                             // coefficients per lane (4 or 8)
    static constexpr int PPV = EPV / 2;                                // fp32 pairs per vector
    // fp16 texels of 16 (padded) coefficients: stored in mma A-fragment order (VsSceneDev::frag_layout) and contracted on
    // the tensor cores, 4 fragments x 4 channels x 16 coefficients per mma.sync.m16n8k16
#ifdef VS_SHADE_NO_MMA   // experiment switch: the packed-FFMA formulation on channel-major texels for every format (see vs_api.cu)
    static constexpr bool MMA = false;
#else
    static constexpr bool MMA = F16 && NCOEF > 8;
#endif
};

// D (16x8, fp32) = A (16x16, fp16, row) x B (16x8, fp16, col), C = 0
__device__ __forceinline__ void vs_mma_16816(float& d0, float& d1, float& d2, float& d3, const uint4& a, uint32_t b0, uint32_t b1)
{
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%10, %10, %10, %10};"
                 : "=f"(d0), "=f"(d1), "=f"(d2), "=f"(d3)
                 : "r"(a.x), "r"(a.y), "r"(a.z), "r"(a.w), "r"(b0), "r"(b1), "f"(0.0f));
}

// A CTA shades a 16-pixel-wide strip of VS_SHADE_WARPS / 2 warp rows (8x4-pixel warp blocks) of one 16x16 mask tile:
// 8 warps = the whole tile, 4 warps = its upper or lower half (smaller CTAs pack the register file more tightly).
#ifndef VS_SHADE_WARPS
#define VS_SHADE_WARPS 4
#endif
#ifndef VS_SHADE_MIN_CTAS
#define VS_SHADE_MIN_CTAS (24 / VS_SHADE_WARPS)
#endif
#ifndef VS_SHADE_DEPTH
#define VS_SHADE_DEPTH 3      // tensor-core path: register buffers of texel vectors per lane (one is being consumed); others: 2
#endif
#ifndef VS_SHADE_RING
#define VS_SHADE_RING 0       // experiment: > 0 = the tensor-core path stages its texel vectors through a shared-memory
#endif                        // ring of that many fragment columns filled by cp.async (LDGSTS) instead of register buffers
#define VS_SHADE_PIX (VS_SHADE_WARPS * 32)
#define VS_SHADE_WARP_BYTES (3584 + VS_SHADE_RING * 2048)   // shared memory per warp: SH basis 2048 + fragment records 2 x 512 + logits 512 (+ ring)
__device__ __forceinline__ void vs_cp_async16(void* smem_dst, const void* gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void vs_cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
// at most n copy groups of this thread may still be pending (n is a constant after unrolling)
__device__ __forceinline__ void vs_cp_async_wait(int n)
{
    switch (n) {
        case 0: asm volatile("cp.async.wait_group 0;" ::: "memory"); break;
        case 1: asm volatile("cp.async.wait_group 1;" ::: "memory"); break;
        case 2: asm volatile("cp.async.wait_group 2;" ::: "memory"); break;
        case 3: asm volatile("cp.async.wait_group 3;" ::: "memory"); break;
        case 4: asm volatile("cp.async.wait_group 4;" ::: "memory"); break;
        case 5: asm volatile("cp.async.wait_group 5;" ::: "memory"); break;
        default: asm volatile("cp.async.wait_group 6;" ::: "memory"); break;
    }
}
#define VS_SHADE_SUBTILES (8 / VS_SHADE_WARPS)
// BWD (vs_render_backward): the same forward pass, but instead of writing the image every owner keeps
// (rgb, sigma, T) of the layers it composited in shared memory, then walks them back to front with the recurrence
//   R_end = bg . g_rgb - g_a ;  dL/dA_l = T_l (rgb_l . g_rgb - R_l) ;  R_{l-1} = A_l (rgb_l . g_rgb) + (1 - A_l) R_l
// and the octets scatter w_q Y_c dL/ds_ch into the fp32 gradient textures ([texel][c][ch], the API layout): lane i of an
// octet adds the coefficients c = i and c = 8 + i (a float4 of the 4 channels each) of the four texels of its fragment with
// red.global.add.v4.f32, so that every reduction instruction covers whole 128-byte lines.
__device__ __forceinline__ void vs_red_add4(float4* p, float a, float b, float c, float d)
{
#ifdef VS_BW_EXP_NORED     // timing experiment only (wrong gradients): everything but the reductions
    if (a != 12345.678f) return;
#endif
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

template <int F16, int DEG, bool COUNT, bool PF, bool BWD>
__global__ void __launch_bounds__(VS_SHADE_PIX, BWD ? 4 : VS_SHADE_MIN_CTAS)
k_shade(const VsSceneDev sc, const VsFrame fr, const VsCamDev* __restrict__ cams, const int4* __restrict__ vtx,
        const uint32_t* __restrict__ tile_off, const uint32_t* __restrict__ ids, unsigned long long* __restrict__ keys,
        uint32_t* __restrict__ out_ids, float* __restrict__ out_rgba,
        uint32_t* __restrict__ texel_bits, unsigned long long* __restrict__ counters, const uint32_t* __restrict__ order,
        const float* __restrict__ grad_out, const __grid_constant__ VsGradTex gt)
{
    typedef VsShadeShape<F16, DEG> S;
    constexpr int SLOTS = S::SLOTS, LPC = S::LPC, NACT = S::NACT, NE = S::NE, PPV = S::PPV;

    extern __shared__ __align__(16) unsigned char smem[];
    // [k][pixels] packed texel coordinates, then [k][pixels] float2 fractions (a < 0: no fragment)
    uint32_t* rec_xy = reinterpret_cast<uint32_t*>(smem);
    float2* rec_ab = reinterpret_cast<float2*>(smem + (size_t)sc.k * VS_SHADE_PIX * 4);
    unsigned char* per_warp = smem + (size_t)sc.k * VS_SHADE_PIX * 12;  // per warp: 2 KB basis + 1 KB records + 512 B logits
    float* rec_aw = reinterpret_cast<float*>(per_warp + VS_SHADE_WARPS * VS_SHADE_WARP_BYTES);   // [k][pixels] attenuation weights (only if fr.attenuate; always reserved under BWD)
    float4* act = reinterpret_cast<float4*>(rec_aw + (size_t)sc.k * VS_SHADE_PIX);                // BWD: [k][pixels] {sigmoid rgb, sigmoid of the opacity logit}
    float* trans = reinterpret_cast<float*>(act + (size_t)sc.k * VS_SHADE_PIX);                   // BWD: [k][pixels] transmittance in front of the layer

    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t tiles = fr.tiles_x * fr.tiles_y;
    uint32_t tile = blockIdx.x / VS_SHADE_SUBTILES, view = blockIdx.y;
    const uint32_t sub = blockIdx.x % VS_SHADE_SUBTILES;
    if (order) {   // surface order (vs_kernels_order.cu): CTAs are dispatched in launch order, entry = linear CTA index
        const uint32_t e = __ldg(&order[view * tiles + tile]);
        view = e / tiles; tile = e - view * tiles;
    }
    const int W = (int)fr.width, H = (int)fr.height;
    // lane -> pixel of the warp's 8x4 block: column = lane & 7, row = lane >> 3
    const int lx = (int)(warp & 1) * 8 + (int)(lane & 7), ly = (int)(sub * (VS_SHADE_WARPS / 2) + (warp >> 1)) * 4 + (int)(lane >> 3);
    const int px = (int)(tile % fr.tiles_x) * VS_TILE_W + lx, py = (int)(tile / fr.tiles_x) * VS_TILE_H + ly;
    const bool inimg = px < W && py < H;
    const size_t pix = ((size_t)view * H + py) * W + px;

    // tiled path: tile_off = reference list offsets; direct path: tile_off = per-tile masks of the layers drawn into
    const uint32_t lmask = keys ? tile_off[view * tiles + tile] : 0xFFFFFFFFu;
    if (keys ? lmask == 0u : tile_off[view * tiles + tile] == tile_off[view * tiles + tile + 1]) {  // nothing drawn here: background
        if (BWD) return;   // no fragment, no gradient
        if (out_ids && inimg)
            for (uint32_t l = 0; l < sc.k; ++l) out_ids[((size_t)view * sc.k + l) * ((size_t)W * H) + (size_t)py * W + px] = VS_MISS;
        if (inimg) reinterpret_cast<float4*>(out_rgba)[pix] = make_float4(fr.bg[0], fr.bg[1], fr.bg[2], 0.0f);
        return;
    }
    const int4* __restrict__ vv = vtx + (size_t)view * sc.v_total;

    // ---------------- phase A: fragment records of all layers ----------------
    const size_t plane = (size_t)W * H;
    const size_t pix0 = (size_t)view * sc.k * plane + (size_t)py * W + px;
    const uint32_t* idp = ids + pix0;
    bool any_hit = false;
    {
        // The gather chain key/id -> index record -> 3 vertices + 3 uvs is walked level by level: all layers' keys
        // first, then all index records, then the vertices three layers at a time (5 dependent round trips per
        // tile instead of 3 per group of three layers).
        uint32_t id[VS_MAX_LAYERS];
        if (keys) {
            // direct path: the key image of k_raster_direct; what is read is cleared for the next pass over this buffer
            unsigned long long key[VS_MAX_LAYERS];
#pragma unroll
            for (int u = 0; u < VS_MAX_LAYERS; ++u)
                key[u] = (inimg && u < (int)sc.k && ((lmask >> u) & 1u)) ? vs_key_load(&keys[pix0 + (size_t)u * plane]) : 0ull;
#pragma unroll
            for (int u = 0; u < VS_MAX_LAYERS; ++u) {
                id[u] = key[u] ? 0xFFFFFFFFu - (uint32_t)key[u] : VS_MISS;
                if (key[u]) vs_key_clear(&keys[pix0 + (size_t)u * plane]);
                if (out_ids && inimg && u < (int)sc.k) out_ids[pix0 + (size_t)u * plane] = id[u];
            }
        } else {
#pragma unroll
            for (int u = 0; u < VS_MAX_LAYERS; ++u) id[u] = (inimg && u < (int)sc.k) ? __ldg(idp + (size_t)u * plane) : VS_MISS;
        }
        uint4 tri[VS_MAX_LAYERS];
#pragma unroll
        for (int u = 0; u < VS_MAX_LAYERS; ++u)
            tri[u] = id[u] != VS_MISS ? __ldg(&sc.tris[sc.tri_off[u] + id[u]]) : make_uint4(0, 0, 0, 0);
        if (fr.attenuate) {  // alpha_w of every layer's fragment: all of a pixel's fragments share its view direction
            float vx, vy, vz;
            vs_view_dir(cams[view], px, py, vx, vy, vz);
#pragma unroll
            for (int u = 0; u < VS_MAX_LAYERS; ++u)
                if (u < (int)sc.k && id[u] != VS_MISS)
                    rec_aw[u * VS_SHADE_PIX + tid] = vs_alpha_w(vx, vy, vz, vs_fragment_normal(sc, vv, u, id[u], px, py));
        }
#pragma unroll
        for (int u = 0; u < VS_MAX_LAYERS; ++u) {
            if (u < (int)sc.k) {
                uint32_t xy = 0;
                float2 ab = make_float2(-1.0f, 0.0f);
                if (id[u] != VS_MISS) {
                    VsFrag f;
                    vs_fragment_setup_tri(sc, vv, u, tri[u], px, py, f);
                    xy = vs_pack_frag(f);
                    ab = make_float2(f.a, f.b);
                    any_hit = true;
                }
                rec_xy[u * VS_SHADE_PIX + tid] = xy;
                rec_ab[u * VS_SHADE_PIX + tid] = ab;
            }
        }
    }
    // each thread reads back only its own records: no barrier needed
    // pull the footprint of this pixel in layer `ln` into L2 (issued VS_SHADE_PF_DIST layers ahead of its use)
    auto prefetch_layer = [&](uint32_t ln) {
#ifdef VS_EXP_TEXMASK
        return;
#endif
        const float2 abn = rec_ab[ln * VS_SHADE_PIX + tid];
        if (abn.x >= 0.0f) {
            const uint32_t xy = rec_xy[ln * VS_SHADE_PIX + tid];
            const uint32_t cx0 = xy & 0x7FFFu, cy0 = (xy >> 16) & 0x7FFFu, Wt = sc.tex_w[ln];
            const uint4* p0 = sc.tex[ln] + (size_t)(cy0 * Wt + cx0) * S::NVEC;
            const uint4* p1 = p0 + ((xy >> 31) ? (size_t)Wt * S::NVEC : (size_t)0);
            const uint32_t dx = ((xy >> 15) & 1u) * S::NVEC;
            if (VS_SHADE_PFMODE == 0) {
                vs_prefetch_l2(p0); vs_prefetch_l2(p1);
                if (VS_SHADE_PREFETCH != 1) { vs_prefetch_l2(p0 + dx); vs_prefetch_l2(p1 + dx); }
            } else if (VS_SHADE_PFMODE == 1) {
                const uint32_t bytes = (S::NVEC + dx) * 16u;
                vs_prefetch_l2_bulk(p0, bytes);
                if (xy >> 31) vs_prefetch_l2_bulk(p1, bytes);
            } else {
                // the 256-byte aligned blocks that hold the row's one or two texels (texture allocations are padded to 256 bytes)
                const unsigned long long a0 = (unsigned long long)p0, a1 = (unsigned long long)p1;
                const unsigned long long s0 = a0 & ~255ull, s1 = a1 & ~255ull;
                const uint32_t bytes = (uint32_t)(((a0 + (S::NVEC + dx) * 16u + 255ull) & ~255ull) - s0);
                vs_prefetch_l2_bulk((const void*)s0, bytes);
                if (xy >> 31) vs_prefetch_l2_bulk((const void*)s1, bytes);
            }
        }
    };
    // In surface order most texels are already in L2 (another view's tile has just used them) and the prefetches are pure issue
    // overhead: C4 step 23.55 ms without against 24.67 ms with them.  In screen order they pay (27.1 against 27.7 ms).
    // (PF is a template parameter: the prefetch code left in the kernel behind a run-time flag still costs 0.1 ms per launch)
    constexpr bool pf_on = PF;
    if (pf_on)
        for (uint32_t ln = 0; ln < VS_SHADE_PF_DIST && ln < sc.k; ++ln) prefetch_layer(ln);

    if (!__any_sync(0xFFFFFFFFu, any_hit)) {
        if (!BWD && inimg) reinterpret_cast<float4*>(out_rgba)[pix] = make_float4(fr.bg[0], fr.bg[1], fr.bg[2], 0.0f);
        return;
    }

    // ---------------- phase B: shade + composite ----------------
    const uint32_t oct = lane >> 3, oi = lane & 7;  // octet index (= pixel row) / lane within octet
    // SH basis of the warp's 32 pixels: pixel (row r, column c) owns the four 16-byte chunks of slot r * 8 + (c ^ (r & 1)) and
    // keeps chunk q at position (q + (r >> 1) + (c >> 1)) & 3 -- both the owners' stores (8 columns of a row per quarter warp)
    // and the octets' loads (2 chunks x the 4 rows of one column) then touch every bank group exactly once
    float4* ysm = reinterpret_cast<float4*>(per_warp + warp * VS_SHADE_WARP_BYTES);
    // record / logit slabs, one 16-byte chunk per pixel, pixel (row o, column j) at chunk 8 o + ((j + 2 o) & 7):
    // the owners' stores (8 columns of one row) and the octets' accesses (4 rows of one column) are both conflict free
    uint4* rec_o = reinterpret_cast<uint4*>(per_warp + warp * VS_SHADE_WARP_BYTES + 2048);    // texel offsets
    float4* rec_w = reinterpret_cast<float4*>(per_warp + warp * VS_SHADE_WARP_BYTES + 2560);  // bilinear weights
    float4* part = reinterpret_cast<float4*>(per_warp + warp * VS_SHADE_WARP_BYTES + 3072);   // 4 channel logits
    const uint32_t own_slot = (lane & 24u) + (((lane & 7u) + 2u * (lane >> 3)) & 7u);
    {
        // SH basis of the owner's pixel (layout: see ysm above)
        float Y[16];
#pragma unroll
        for (int c = 0; c < 16; ++c) Y[c] = 0.0f;
        float vx, vy, vz;
        vs_view_dir(cams[view], px, py, vx, vy, vz);
        vs_sh_basis<DEG>(vx, vy, vz, Y);
        const uint32_t yr = lane >> 3, yc = lane & 7;
        float4* row = ysm + (yr * 8 + (yc ^ (yr & 1))) * 4;
        if (S::MMA) {
            // B operand of the mma: Y_c = hi_c + lo_c in fp16 (|error| < 2^-22 |Y_c|), chunk i = hilo * 2 + (t >> 1) holds the
            // halves {x[2t], x[2t+1], x[2t+8], x[2t+9]} of t = 2 (i & 1) and t + 1: lane oi of an octet reads 8 bytes at 8 oi
            __half hi[16], lo[16];
#pragma unroll
            for (int c = 0; c < 16; ++c) {
                hi[c] = __float2half_rn(Y[c]);
                lo[c] = __float2half_rn(Y[c] - __half2float(hi[c]));
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const __half* x = (i >> 1) ? lo : hi;
                const int t0 = 2 * (i & 1);
                const __half2 h0 = __halves2half2(x[2 * t0], x[2 * t0 + 1]), h1 = __halves2half2(x[2 * t0 + 8], x[2 * t0 + 9]);
                const __half2 h2 = __halves2half2(x[2 * t0 + 2], x[2 * t0 + 3]), h3 = __halves2half2(x[2 * t0 + 10], x[2 * t0 + 11]);
                uint4 u;
                u.x = *reinterpret_cast<const uint32_t*>(&h0); u.y = *reinterpret_cast<const uint32_t*>(&h1);
                u.z = *reinterpret_cast<const uint32_t*>(&h2); u.w = *reinterpret_cast<const uint32_t*>(&h3);
                reinterpret_cast<uint4*>(row)[(i + (yr >> 1) + (yc >> 1)) & 3] = u;
            }
        } else {
#pragma unroll
            for (int q = 0; q < 4; ++q) row[(q + (yr >> 1) + (yc >> 1)) & 3] = make_float4(Y[4 * q], Y[4 * q + 1], Y[4 * q + 2], Y[4 * q + 3]);
        }
    }
    const uint32_t ychunk0 = ((oi % LPC) * NE) >> 2;   // first 16-byte chunk of this lane's coefficients
    const bool lane_on = oi < (uint32_t)NACT;
#ifndef VS_SHADE_BF_REGS
#define VS_SHADE_BF_REGS 1    // 1: the tensor-core path keeps the B fragments (SH basis) of its 8 columns in 16 registers for all layers
#endif
    uint2 bfr[8];
    if (S::MMA && VS_SHADE_BF_REGS) {
        __syncwarp();
#pragma unroll
        for (int j = 0; j < 8; ++j)
            bfr[j] = *reinterpret_cast<const uint2*>(reinterpret_cast<const unsigned char*>(ysm) +
                (oct * 8 + ((uint32_t)j ^ (oct & 1))) * 64 + ((((oi >> 2) * 2 + ((oi & 3) >> 1)) + (oct >> 1) + (j >> 1)) & 3) * 16 + (oi & 1) * 8);
    }

    float Tr = 1.0f, Cr = 0.0f, Cg = 0.0f, Cb = 0.0f;
    bool alive = true;
    uint32_t used = 0;   // BWD: layers this pixel composited (bit l)
    for (uint32_t l = 0; l < sc.k; ++l) {
        const float2 ab = rec_ab[l * VS_SHADE_PIX + tid];
        const bool shade = ab.x >= 0.0f && alive;
        const unsigned m = __ballot_sync(0xFFFFFFFFu, shade);
        if (m == 0) continue;  // warp-uniform
        VsFragRec r;
        r.o00 = r.o01 = r.o10 = r.o11 = 0; r.w00 = r.w01 = r.w10 = r.w11 = 0.0f;
        if (shade) {
            const uint32_t xy = rec_xy[l * VS_SHADE_PIX + tid];
            const uint32_t cx0 = xy & 0x7FFFu, cy0 = (xy >> 16) & 0x7FFFu;
            const uint32_t Wt = sc.tex_w[l], nv = (uint32_t)S::NVEC;
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
        // two 16-byte records per fragment (texel offsets, bilinear weights).  One packed record {offset 00 | flag, offset 10, a, b}
        // from which the octets rebuild the rest was measured: -22 % shared-memory wavefronts but +15 % instructions, 4.455 vs
        // 4.375 ms per 16-view launch under ncu, no gain under the power cap (profiles/r2_c4_summary.md)
        rec_o[own_slot] = make_uint4(r.o00, r.o01, r.o10, r.o11);
        rec_w[own_slot] = make_float4(r.w00, r.w01, r.w10, r.w11);
        __syncwarp();
        // address = per-lane base + 16 * (32-bit texel-vector offset): one IMAD.WIDE.U32 per load
        const char* __restrict__ tb = reinterpret_cast<const char*>(sc.tex[l] + SLOTS * oi);

        constexpr bool RING = S::MMA && VS_SHADE_RING > 0;
        constexpr int DEPTH = RING ? VS_SHADE_RING : (S::MMA ? VS_SHADE_DEPTH : 2);
        // RING: [stage][texel][lane] 16-byte slots of this warp; a lane reads back only what it copied itself
        uint4* ring = reinterpret_cast<uint4*>(per_warp + warp * VS_SHADE_WARP_BYTES + 3584);
        uint4 tv[RING ? 1 : DEPTH][SLOTS][4];   // ring of texel vectors: columns j .. j + VS_SHADE_DEPTH - 2 are in flight
        auto issue = [&](int j, int b) {
            const uint4 o = rec_o[8 * oct + ((j + 2 * oct) & 7)];
            if (RING) {
                const uint32_t off4[4] = {o.x, o.y, o.z, o.w};
#pragma unroll
                for (int q = 0; q < 4; ++q) vs_cp_async16(ring + (b * 4 + q) * 32 + lane, tb + (unsigned long long)off4[q] * 16ull);
                vs_cp_async_commit();
                return;
            }
#pragma unroll
            for (int s = 0; s < SLOTS; ++s) {
                if (lane_on) {
                    tv[b][s][0] = vs_ldg_tex(tb, o.x, s); tv[b][s][1] = vs_ldg_tex(tb, o.y, s);
                    tv[b][s][2] = vs_ldg_tex(tb, o.z, s); tv[b][s][3] = vs_ldg_tex(tb, o.w, s);
                } else {
                    tv[b][s][0] = tv[b][s][1] = tv[b][s][2] = tv[b][s][3] = make_uint4(0, 0, 0, 0);
                }
            }
        };
#pragma unroll
        for (int j = 0; j < DEPTH - 1; ++j) issue(j, j);
        if (pf_on && l + VS_SHADE_PF_DIST < sc.k && alive) prefetch_layer(l + VS_SHADE_PF_DIST);
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            if (j + DEPTH - 1 < 8) issue(j + DEPTH - 1, (j + DEPTH - 1) % DEPTH);
            const int b = j % DEPTH;
            const int tb_i = RING ? 0 : b;
            if (RING) {   // the copies of column j have landed (at most the younger groups are still pending)
                vs_cp_async_wait((7 - j) < (DEPTH - 2) ? (7 - j) : (DEPTH - 2));
#pragma unroll
                for (int q = 0; q < 4; ++q) tv[0][0][q] = ring[(b * 4 + q) * 32 + lane];
            }
            const uint32_t slot = 8 * oct + ((j + 2 * oct) & 7);
            const float4 w = rec_w[slot];
            if (S::MMA) {
                // rows of A = (fragment f = octet, channel), columns of B = (fragment, hi | lo): lane (g = lane >> 2, t = lane & 3)
                // gets D[g][2t .. 2t+1] and D[g+8][..]; the entries of its OWN fragment are those of t == f
                const uint2 bf = VS_SHADE_BF_REGS ? bfr[j] : *reinterpret_cast<const uint2*>(reinterpret_cast<const unsigned char*>(ysm) +
                    (oct * 8 + ((uint32_t)j ^ (oct & 1))) * 64 + ((((oi >> 2) * 2 + ((oi & 3) >> 1)) + (oct >> 1) + (j >> 1)) & 3) * 16 + (oi & 1) * 8);
                float d0, d1, d2, d3, sa, sb;
                vs_mma_16816(d0, d1, d2, d3, tv[tb_i][0][0], bf.x, bf.y);
                sa = w.x * (d0 + d1); sb = w.x * (d2 + d3);
                vs_mma_16816(d0, d1, d2, d3, tv[tb_i][0][1], bf.x, bf.y);
                sa = fmaf(w.y, d0 + d1, sa); sb = fmaf(w.y, d2 + d3, sb);
                vs_mma_16816(d0, d1, d2, d3, tv[tb_i][0][2], bf.x, bf.y);
                sa = fmaf(w.z, d0 + d1, sa); sb = fmaf(w.z, d2 + d3, sb);
                vs_mma_16816(d0, d1, d2, d3, tv[tb_i][0][3], bf.x, bf.y);
                sa = fmaf(w.w, d0 + d1, sa); sb = fmaf(w.w, d2 + d3, sb);
                // lane (g, t == f) holds channels g & 1 (sa) and (g & 1) + 2 (sb) of its fragment: part = {ch0, ch2, ch1, ch3}
                if ((lane & 3u) == oct) reinterpret_cast<float2*>(part)[slot * 2 + ((lane >> 2) & 1u)] = make_float2(sa, sb);
            } else {
            const f32x2 W00 = vs_pack2(w.x, w.x), W01 = vs_pack2(w.y, w.y), W10 = vs_pack2(w.z, w.z), W11 = vs_pack2(w.w, w.w);
            const float4* yrow = ysm + (oct * 8 + ((uint32_t)j ^ (oct & 1))) * 4;
            f32x2 acc2 = 0ull;
#ifdef VS_EXP_NOMATH   // timing experiment only (wrong images): keep the loads, drop conversions + bilinear + SH arithmetic
            {
                uint32_t x = 0;
#pragma unroll
                for (int s = 0; s < SLOTS; ++s)
#pragma unroll
                    for (int q4 = 0; q4 < 4; ++q4) x ^= tv[b][s][q4].x ^ tv[b][s][q4].y ^ tv[b][s][q4].z ^ tv[b][s][q4].w;
                acc2 = vs_pack2(__uint_as_float(x & 0x3F800000u) * w.x, yrow[ychunk0 & 3].x);
            }
#else
#pragma unroll
            for (int s = 0; s < SLOTS; ++s) {
#pragma unroll
                for (int h = 0; h < PPV / 2; ++h) {   // 16-byte chunk of 4 basis values <-> 2 element pairs
                    const int e = s * PPV + 2 * h;    // element pair index within the lane's coefficients
                    const float4 y = yrow[(ychunk0 + (e >> 1) + (oct >> 1) + (j >> 1)) & 3];
#pragma unroll
                    for (int g = 0; g < 2; ++g) {
                        const int q = 2 * h + g;
                        f32x2 v = vs_mul2(W00, vs_pair<F16>(tv[b][s][0], q));
                        v = vs_fma2(W01, vs_pair<F16>(tv[b][s][1], q), v);
                        v = vs_fma2(W10, vs_pair<F16>(tv[b][s][2], q), v);
                        v = vs_fma2(W11, vs_pair<F16>(tv[b][s][3], q), v);
                        acc2 = vs_fma2(g == 0 ? vs_pack2(y.x, y.y) : vs_pack2(y.z, y.w), v, acc2);
                    }
                }
            }
#endif
            float a0, a1;
            vs_unpack2(acc2, a0, a1);
            float acc = a0 + a1;
            if (LPC == 2) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, 1);
            if (lane_on && (oi % LPC) == 0) reinterpret_cast<float*>(part)[slot * 4 + oi / LPC] = acc;
            }
        }
        __syncwarp();
        if (shade) {
            float4 s4 = part[own_slot];
            if (S::MMA) { const float t = s4.y; s4.y = s4.z; s4.z = t; }   // stored as {ch0, ch2, ch1, ch3}
            float A = vs_sigmoid(s4.w);
            if (BWD) {
                act[l * VS_SHADE_PIX + tid] = make_float4(vs_sigmoid(s4.x), vs_sigmoid(s4.y), vs_sigmoid(s4.z), A);
                trans[l * VS_SHADE_PIX + tid] = Tr;
                used |= 1u << l;
            }
            if (fr.attenuate) A *= rec_aw[l * VS_SHADE_PIX + tid];
            const float TA = Tr * A;
            if (!BWD) { Cr += TA * vs_sigmoid(s4.x); Cg += TA * vs_sigmoid(s4.y); Cb += TA * vs_sigmoid(s4.z); }
            Tr *= (1.0f - A);
            if (Tr < fr.t_min) alive = false;
        }
    }
    if (BWD) {
        // ---------------- backward: recurrence in the owner, octet scatter (every slab below belongs to this warp) ----------------
        // fp32 SH basis over the fp16 B operand: pixel (row r, column c) at slot c * 4 + r, coefficient i at (i + 8 (r >> 1)) & 15,
        // so that the four octets' reads of one column (8 consecutive coefficients each) touch every bank once
        float* y32 = reinterpret_cast<float*>(ysm);
        float4* rec_d = part;   // dL/ds of the four channels, slot mapping of rec_o / rec_w
        __syncwarp();
        {
            float Y[16];
#pragma unroll
            for (int c = 0; c < 16; ++c) Y[c] = 0.0f;
            float vx, vy, vz;
            vs_view_dir(cams[view], px, py, vx, vy, vz);
            vs_sh_basis<DEG>(vx, vy, vz, Y);
            const uint32_t yr = lane >> 3, yc = lane & 7;
            float4* row = reinterpret_cast<float4*>(y32 + (yc * 4 + yr) * 16);
#pragma unroll
            for (int q = 0; q < 4; ++q) row[(q + 2 * (yr >> 1)) & 3] = make_float4(Y[4 * q], Y[4 * q + 1], Y[4 * q + 2], Y[4 * q + 3]);
        }
        float4 g = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (inimg) g = __ldg(reinterpret_cast<const float4*>(grad_out) + pix);
        float R = fr.bg[0] * g.x + fr.bg[1] * g.y + fr.bg[2] * g.z - g.w;
        constexpr uint32_t NC = (uint32_t)S::NCOEF;   // float4s per gradient texel
        for (int l = (int)sc.k - 1; l >= 0; --l) {
            const bool on = (used >> l) & 1u;
            if (__ballot_sync(0xFFFFFFFFu, on) == 0u) continue;   // warp-uniform
            uint4 ro = make_uint4(0, 0, 0, 0);
            float4 rw = make_float4(0.0f, 0.0f, 0.0f, 0.0f), rd = rw;
            if (on) {
                const float4 a4 = act[l * VS_SHADE_PIX + tid];
                const float Tl = trans[l * VS_SHADE_PIX + tid];
                const float aw = fr.attenuate ? rec_aw[l * VS_SHADE_PIX + tid] : 1.0f;
                const float A = a4.w * aw;
                const float cg = a4.x * g.x + a4.y * g.y + a4.z * g.z;
                const float TA = Tl * A;
                rd.x = TA * g.x * a4.x * (1.0f - a4.x);
                rd.y = TA * g.y * a4.y * (1.0f - a4.y);
                rd.z = TA * g.z * a4.z * (1.0f - a4.z);
                rd.w = Tl * (cg - R) * aw * a4.w * (1.0f - a4.w);
                R = A * cg + (1.0f - A) * R;
                const float2 ab = rec_ab[l * VS_SHADE_PIX + tid];
                const uint32_t xy = rec_xy[l * VS_SHADE_PIX + tid];
                const uint32_t cx0 = xy & 0x7FFFu, cy0 = (xy >> 16) & 0x7FFFu, Wt = sc.tex_w[l];
                const uint32_t row0 = cy0 * Wt, row1 = row0 + ((xy >> 31) ? Wt : 0u), cx1 = cx0 + ((xy >> 15) & 1u);
                ro = make_uint4((row0 + cx0) * NC, (row0 + cx1) * NC, (row1 + cx0) * NC, (row1 + cx1) * NC);   // < 2^32: checked at scene creation
                rw = make_float4((1.0f - ab.x) * (1.0f - ab.y), ab.x * (1.0f - ab.y), (1.0f - ab.x) * ab.y, ab.x * ab.y);
            }
            rec_o[own_slot] = ro; rec_w[own_slot] = rw; rec_d[own_slot] = rd;
            // Magnified textures (close-ups; the fitting regime of PAPER.md:L441-443, where many pixels fall into one texel
            // cell): neighbouring pixels of a row then have the SAME 2x2 footprint, and the octet, which walks its row from
            // left to right, sums such a run in registers and issues the reductions once per run instead of once per pixel.
            // Taken only by warps in which some pixel shares its footprint with its left neighbour (warp-uniform).
            bool merge;
            {
                const uint32_t lx0 = __shfl_up_sync(0xFFFFFFFFu, ro.x, 1), ly0 = __shfl_up_sync(0xFFFFFFFFu, ro.y, 1);
                const uint32_t lz0 = __shfl_up_sync(0xFFFFFFFFu, ro.z, 1), lw0 = __shfl_up_sync(0xFFFFFFFFu, ro.w, 1);
                const int lon = __shfl_up_sync(0xFFFFFFFFu, (int)on, 1);
                merge = __any_sync(0xFFFFFFFFu, on && lon && (lane & 7u) != 0u && lx0 == ro.x && ly0 == ro.y && lz0 == ro.z && lw0 == ro.w);
            }
            __syncwarp();
            float4* __restrict__ gl = reinterpret_cast<float4*>(gt.p[l]);
#ifdef VS_BW_NO_MERGE   // experiment switch: always one set of reductions per pixel
            merge = false;
#endif
            if (merge) {
                float4 acc[2][4];
                uint4 cur = make_uint4(0, 0, 0, 0);
                bool have = false;
                auto flush = [&]() {
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const uint32_t c = oi + 8 * h;
                        if (c >= NC) continue;
                        vs_red_add4(gl + cur.x + c, acc[h][0].x, acc[h][0].y, acc[h][0].z, acc[h][0].w);
                        vs_red_add4(gl + cur.y + c, acc[h][1].x, acc[h][1].y, acc[h][1].z, acc[h][1].w);
                        vs_red_add4(gl + cur.z + c, acc[h][2].x, acc[h][2].y, acc[h][2].z, acc[h][2].w);
                        vs_red_add4(gl + cur.w + c, acc[h][3].x, acc[h][3].y, acc[h][3].z, acc[h][3].w);
                    }
                };
#pragma unroll 1
                for (int j = 0; j < 8; ++j) {
                    const uint32_t slot = 8 * oct + ((j + 2 * oct) & 7);
                    const float4 w = rec_w[slot];
                    if (w.x == 0.0f && w.y == 0.0f && w.z == 0.0f && w.w == 0.0f) continue;   // (does not end a run)
                    const uint4 o = rec_o[slot];
                    const float4 d = rec_d[slot];
                    if (!(have && o.x == cur.x && o.y == cur.y && o.z == cur.z && o.w == cur.w)) {   // octet-uniform
                        if (have) flush();
                        cur = o; have = true;
#pragma unroll
                        for (int h = 0; h < 2; ++h)
#pragma unroll
                            for (int q = 0; q < 4; ++q) acc[h][q] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                    }
                    const float wq[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const uint32_t c = oi + 8 * h;
                        if (c >= NC) continue;
                        const float y = y32[(j * 4 + oct) * 16 + ((c + 8 * (oct >> 1)) & 15)];
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            const float wy = wq[q] * y;
                            acc[h][q].x = fmaf(wy, d.x, acc[h][q].x); acc[h][q].y = fmaf(wy, d.y, acc[h][q].y);
                            acc[h][q].z = fmaf(wy, d.z, acc[h][q].z); acc[h][q].w = fmaf(wy, d.w, acc[h][q].w);
                        }
                    }
                }
                if (have) flush();
            } else {
#pragma unroll 2
            for (int j = 0; j < 8; ++j) {
                const uint32_t slot = 8 * oct + ((j + 2 * oct) & 7);   // fragment of pixel row oct, column j
                const float4 w = rec_w[slot];
                if (w.x == 0.0f && w.y == 0.0f && w.z == 0.0f && w.w == 0.0f) continue;
                const uint4 o = rec_o[slot];
                const float4 d = rec_d[slot];
#pragma unroll
#ifdef VS_BW_EXP_HALF   // timing experiment only (wrong gradients): half of the reductions
                for (int h = 0; h < 1; ++h) {
#else
                for (int h = 0; h < 2; ++h) {
#endif
                    const uint32_t c = oi + 8 * h;
                    if (c >= NC) continue;
                    const float y = y32[(j * 4 + oct) * 16 + ((c + 8 * (oct >> 1)) & 15)];
                    float wy = w.x * y; vs_red_add4(gl + o.x + c, wy * d.x, wy * d.y, wy * d.z, wy * d.w);
                    wy = w.y * y;       vs_red_add4(gl + o.y + c, wy * d.x, wy * d.y, wy * d.z, wy * d.w);
                    wy = w.z * y;       vs_red_add4(gl + o.z + c, wy * d.x, wy * d.y, wy * d.z, wy * d.w);
                    wy = w.w * y;       vs_red_add4(gl + o.w + c, wy * d.x, wy * d.y, wy * d.z, wy * d.w);
                }
            }
            }
            __syncwarp();
        }
        return;
    }
    if (inimg) {
        const float4 o4 = make_float4(Cr + Tr * fr.bg[0], Cg + Tr * fr.bg[1], Cb + Tr * fr.bg[2], 1.0f - Tr);
#if VS_KEYS_STREAM >= 2
        __stcs(reinterpret_cast<float4*>(out_rgba) + pix, o4);
#else
        reinterpret_cast<float4*>(out_rgba)[pix] = o4;
#endif
    }
}

template <int F16, int DEG, bool COUNT>
static cudaError_t launch_sh2(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    if (sc.texel_vecs != (uint32_t)VsShadeShape<F16, DEG>::NVEC) return cudaErrorInvalidValue;
    const size_t smem = (size_t)sc.k * VS_SHADE_PIX * (fr.attenuate ? 16 : 12) + VS_SHADE_WARPS * VS_SHADE_WARP_BYTES;
    const bool pf = VS_SHADE_PREFETCH && (VS_SHADE_PREFETCH >= 3 || ch.order == nullptr);
    auto kern = pf ? k_shade<F16, DEG, COUNT, true, false> : k_shade<F16, DEG, COUNT, false, false>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
#ifdef VS_SHADE_CARVEOUT
    e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, VS_SHADE_CARVEOUT);
    if (e != cudaSuccess) return e;
#endif
    dim3 grid(fr.tiles_x * fr.tiles_y * VS_SHADE_SUBTILES, ch.views);
    if (ch.keys)
        kern<<<grid, VS_SHADE_PIX, smem, st>>>(sc, fr, ch.cams, ch.vtx, ch.tile_mask, nullptr, ch.keys, ch.ids_is_output ? ch.ids : nullptr,
                                      ch.out_rgba, ch.texel_bits, ch.counters, ch.order, nullptr, VsGradTex{});
    else
        kern<<<grid, VS_SHADE_PIX, smem, st>>>(sc, fr, ch.cams, ch.vtx, ch.tile_off, ch.ids, nullptr, nullptr, ch.out_rgba, ch.texel_bits,
                                      ch.counters, nullptr, nullptr, VsGradTex{});
    return cudaGetLastError();
}

// vs_render_backward on the direct path: k_shade<BWD> in place of k_shade (consumes and clears the same key image)
template <int F16, int DEG>
static cudaError_t launch_bwd(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    if (sc.texel_vecs != (uint32_t)VsShadeShape<F16, DEG>::NVEC || !ch.keys) return cudaErrorInvalidValue;
    // fragment records 12 B + attenuation weights 4 B + kept activations 20 B per pixel and layer, and the per-warp slabs
    const size_t smem = (size_t)sc.k * VS_SHADE_PIX * 36 + VS_SHADE_WARPS * VS_SHADE_WARP_BYTES;
    auto kern = k_shade<F16, DEG, false, false, true>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid(fr.tiles_x * fr.tiles_y * VS_SHADE_SUBTILES, ch.views);
    kern<<<grid, VS_SHADE_PIX, smem, st>>>(sc, fr, ch.cams, ch.vtx, ch.tile_mask, nullptr, ch.keys, nullptr, nullptr, nullptr, ch.counters,
                                           ch.order, ch.grad_out, ch.grad_tex);
    return cudaGetLastError();
}

cudaError_t vs_launch_shade_backward(const VsSceneDev& sc, int f16, const VsFrame& fr, const VsChunk& ch, cudaStream_t st)
{
    switch ((f16 ? 4 : 0) + (int)sc.sh_degree) {
        case 0: return launch_bwd<0, 0>(sc, fr, ch, st);
        case 1: return launch_bwd<0, 1>(sc, fr, ch, st);
        case 2: return launch_bwd<0, 2>(sc, fr, ch, st);
        case 3: return launch_bwd<0, 3>(sc, fr, ch, st);
        case 4: return launch_bwd<1, 0>(sc, fr, ch, st);
        case 5: return launch_bwd<1, 1>(sc, fr, ch, st);
        case 6: return launch_bwd<1, 2>(sc, fr, ch, st);
        case 7: return launch_bwd<1, 3>(sc, fr, ch, st);
    }
    return cudaErrorInvalidValue;
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

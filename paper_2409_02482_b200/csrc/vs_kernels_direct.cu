// vs_kernels_direct.cu -- S2 + S4 without screen tiles: triangle-parallel coverage and per-layer
// nearest-fragment resolve straight into a 64-bit key image in HBM/L2.  DESIGN.md §1, §3.2-3.4, §7.
//
// The paper-shaped scenes consist of triangles of a few pixels (C4: ~6 px each, 2.7 M per view).  For
// those, binning every triangle into 16x16 tiles and re-gathering it per tile costs more than the
// rasterisation itself, so this path visits every triangle exactly once:
//   phase 1, lane = triangle: coalesced index record, three vertex gathers, integer setup, sample
//     bounding box clipped to the screen.  A triangle whose box fits 8x8 samples gets its coverage mask
//     from three biased int32 edge functions stepped with exact adds (same arithmetic as k_raster).
//   phase 2, lane = triangle: every lane walks the set bits of its own mask: fp32-exact depth key (IEEE
//     division, the reciprocal of the triangle's area hoisted out of the loop) and one fire-and-forget
//     64-bit max (RED.MAX.U64) on keys[view][layer][y][x] per covered sample.  The maximum is order
//     independent, so the key image is the same whatever the scheduling (reading Q18).  (Until round 2's
//     last session the covered samples of a warp were compacted into a shared-memory queue so that all 32
//     lanes had one sample each; measured: 5.6 iterations of 48 instructions + 141 for the compaction
//     against 7.4 iterations of ~27 -- the warp's largest mask is only 1.7x its mean.)
//   larger triangles are broadcast one at a time and the warp maps its lanes to 8x4 pixel chunks of the
//     box; triangles whose box exceeds VS_BIG_SAMPLES samples are appended to a list that k_raster_big
//     spreads over the whole grid.
// The key image must be zero on entry; k_shade reads it (id = ~low word) and clears what it read.
// tile_mask[view][tile] (zero on entry) receives the layers whose triangles' boxes touch the tile.
#include "vs_common.cuh"
#include "vs_div.cuh"
#include <type_traits>

#define VS_BIG_SAMPLES 4096   // clipped-box samples above which a triangle goes to the big list

__device__ __forceinline__ void vs_key_red(unsigned long long* slot, unsigned long long key)
{
    asm volatile("red.global.max.u64 [%0], %1;" ::"l"(slot), "l"(key) : "memory");
}

__device__ __forceinline__ float vs_depth_div(float f0, float f1, float f2, float q0, float q1, float q2, float fA)
{
    const float num = __fmaf_rn(f2, q2, __fmaf_rn(f1, q1, __fmul_rn(f0, q0)));
    return __fdiv_rn(num, fA);
}

// Whole warp, lane = pixel of an 8x4 chunk of the box [i0,i1] x [j0,j1]; chunks c = first, first+stride, ...
// LINEAR: lane = sample 32 c + lane of the box in row-major order instead (boxes of a few hundred samples, where
// 8x4 chunks would leave most lanes outside the box).
template <typename I, bool LINEAR>
__device__ __forceinline__ void vs_direct_large(int X0, int Y0, int X1, int Y1, int X2, int Y2, float q0, float q1, float q2,
                                                float fA, int i0, int i1, int j0, int j1, int W,
                                                unsigned long long* __restrict__ plane, uint32_t lid, uint32_t lane,
                                                uint32_t first, uint32_t stride)
{
    const int dx0 = X2 - X1, dy0 = Y2 - Y1, dx1 = X0 - X2, dy1 = Y0 - Y2, dx2 = X1 - X0, dy2 = Y1 - Y0;
    const int m0 = ((dy0 < 0) || (dy0 == 0 && dx0 > 0)) ? 0 : 1;
    const int m1 = ((dy1 < 0) || (dy1 == 0 && dx1 > 0)) ? 0 : 1;
    const int m2 = ((dy2 < 0) || (dy2 == 0 && dx2 > 0)) ? 0 : 1;
    const uint32_t bw = (uint32_t)(i1 - i0 + 1), bh = (uint32_t)(j1 - j0 + 1);
    const uint32_t ncx = (bw + 7) >> 3, ncy = (bh + 3) >> 2;
    const uint32_t nchunks = LINEAR ? (bw * bh + 31) >> 5 : ncx * ncy;
    const float inv_bw = 1.0f / (float)bw;
    for (uint32_t c = first; c < nchunks; c += stride) {
        int i, j;
        if (LINEAR) {
            // row = floor((s + 0.5) / bw): s + 0.5 is never within 0.5 / bw of a multiple of bw, so fp32 is exact here (s < 2^13)
            const uint32_t sidx = 32u * c + lane;
            const uint32_t row = (uint32_t)__float2int_rd(((float)sidx + 0.5f) * inv_bw);
            i = i0 + (int)(sidx - row * bw); j = j0 + (int)row;
        } else {
            i = i0 + (int)(c % ncx) * 8 + (int)(lane & 7); j = j0 + (int)(c / ncx) * 4 + (int)(lane >> 3);
        }
        if (i > i1 || j > j1) continue;
        const int Sx = 256 * i + 128, Sy = 256 * j + 128;
        const I e0 = (I)dx0 * (I)(Sy - Y1) - (I)dy0 * (I)(Sx - X1);
        const I e1 = (I)dx1 * (I)(Sy - Y2) - (I)dy1 * (I)(Sx - X2);
        const I e2 = (I)dx2 * (I)(Sy - Y0) - (I)dy2 * (I)(Sx - X0);
        if (e0 >= (I)m0 && e1 >= (I)m1 && e2 >= (I)m2) {
            float f0, f1, f2;
            if (sizeof(I) == 4) { f0 = __int2float_rn((int)e0); f1 = __int2float_rn((int)e1); f2 = __int2float_rn((int)e2); }
            else { f0 = __ll2float_rn((long long)e0); f1 = __ll2float_rn((long long)e1); f2 = __ll2float_rn((long long)e2); }
            const float qp = vs_depth_div(f0, f1, f2, q0, q1, q2, fA);
            vs_key_red(&plane[(size_t)j * W + i], vs_make_key(qp, lid));
        }
    }
}

#ifndef VS_RD_THREADS
#define VS_RD_THREADS 128
#endif
#ifndef VS_RD_MIN_CTAS
#define VS_RD_MIN_CTAS (1024 / VS_RD_THREADS)
#endif
template <bool RESIDENT>
__global__ void __launch_bounds__(VS_RD_THREADS, VS_RD_MIN_CTAS)
k_raster_direct(const VsSceneDev sc, const VsFrame fr, const int4* __restrict__ vtx, unsigned long long* __restrict__ keys,
                uint32_t* __restrict__ tile_mask, uint2* __restrict__ big_list, uint32_t* __restrict__ big_count, uint32_t big_capacity,
                unsigned long long* __restrict__ counters, uint32_t blocks_per_view, uint32_t total_blocks, uint32_t view_major)
{
    const uint32_t tid = threadIdx.x, lane = tid & 31;
    const int W = (int)fr.width, H = (int)fr.height;
    const size_t plane_px = (size_t)W * H;
    // work item = (view, block of VS_RD_THREADS consecutive triangles).  The grid has one CTA per item (x = block, y = view)
    // or, RESIDENT (the kernel runs beside the previous chunk's k_shade), a few CTAs per SM that stride over the items
    for (uint32_t item = RESIDENT ? blockIdx.x : 0u; item < (RESIDENT ? total_blocks : 1u); item += gridDim.x) {
    // 2-D grid: x = view, y = block of triangles when the block count fits gridDim.y (view_major), else x = block, y = view.
    // View-major, CTAs that are dispatched together read the SAME index records for different views: the 16 bytes per
    // triangle come from L2 instead of HBM for all views but one, and a warp's first load returns sooner.
    const uint32_t view = RESIDENT ? item / blocks_per_view : (view_major ? blockIdx.x : blockIdx.y);
    const uint32_t gt = (RESIDENT ? item - view * blocks_per_view : (view_major ? blockIdx.y : blockIdx.x)) * (uint32_t)VS_RD_THREADS + tid;
    const int4* __restrict__ vv = vtx + (size_t)view * sc.v_total;
    unsigned long long* __restrict__ vkeys = keys + (size_t)view * sc.k * plane_px;

    // ---------------- phase 1: lane = triangle ----------------
    VsTri T;
    int i0 = 0, i1 = -1, j0 = 0, j1 = -1, status = -1;
    uint32_t layer = 0, lid = 0;
    bool narrow = false, valid = false, large = false;
    if (gt < sc.t_total) {
        const uint4 tri = __ldg(&sc.tris[gt]);
        const int4 a = __ldg(&vv[tri.x]), b = __ldg(&vv[tri.y]), c = __ldg(&vv[tri.z]);
        status = vs_setup_tri(a, b, c, T);
        if (status == 0) {
            const int minX = min(T.X0, min(T.X1, T.X2)), maxX = max(T.X0, max(T.X1, T.X2));
            const int minY = min(T.Y0, min(T.Y1, T.Y2)), maxY = max(T.Y0, max(T.Y1, T.Y2));
            i0 = max((minX + 127) >> 8, 0); i1 = min((maxX - 128) >> 8, W - 1);
            j0 = max((minY + 127) >> 8, 0); j1 = min((maxY - 128) >> 8, H - 1);
            layer = vs_tri_layer(tri.w); lid = vs_tri_lid(tri.w);
            narrow = maxX - minX < 8192 && maxY - minY < 8192;  // every int32 intermediate < 2^28
            valid = i0 <= i1 && j0 <= j1;
            large = valid && !(narrow && i1 - i0 < 8 && j1 - j0 < 8);
        }
    }
#ifndef VS_EXP_NOMASK
    {
        // layer bit of every 16x16 tile the box touches: k_shade skips the tiles and layers nothing was drawn into.  The mask
        // only has to be a SUPERSET (a set bit costs k_shade a read of zero keys, nothing else).  A warp's 32 consecutive
        // triangles form a compact patch, so the warp marks the tiles of the bounding box of its boxes with the union of its
        // layer bits: five warp reductions and at most one atomic per lane.  Warps whose patch is spread over more than 32
        // tiles (a mesh whose index order jumps) fall back to exact per-triangle marks.
        uint32_t* __restrict__ tm = tile_mask + (size_t)view * fr.tiles_x * fr.tiles_y;
        const int tx0 = i0 / VS_TILE_W, tx1 = i1 / VS_TILE_W, ty0 = j0 / VS_TILE_H, ty1 = j1 / VS_TILE_H;
        const int wx0 = __reduce_min_sync(0xFFFFFFFFu, valid ? tx0 : 0x7FFFFFFF), wx1 = __reduce_max_sync(0xFFFFFFFFu, valid ? tx1 : -1);
        const int wy0 = __reduce_min_sync(0xFFFFFFFFu, valid ? ty0 : 0x7FFFFFFF), wy1 = __reduce_max_sync(0xFFFFFFFFu, valid ? ty1 : -1);
        const uint32_t wl = __reduce_or_sync(0xFFFFFFFFu, valid ? (1u << layer) : 0u);
        const int nx = wx1 - wx0 + 1, nt = nx * (wy1 - wy0 + 1);
        if (wl != 0u && nt <= 32) {
            for (int ty = wy0; ty <= wy1; ++ty)   // (warp-uniform trip count; lanes = tile columns: no integer division)
                if ((int)lane < nx) atomicOr(&tm[(size_t)ty * fr.tiles_x + (wx0 + (int)lane)], wl);
        } else if (wl != 0u) {
#pragma unroll
            for (int c = 0; c < 4; ++c) {  // the four corner tiles; a box of at most 8x8 samples touches no other
                const int tx = (c & 1) ? tx1 : tx0, ty = (c & 2) ? ty1 : ty0;
                const bool fresh = valid && !((c & 1) && tx1 == tx0) && !((c & 2) && ty1 == ty0);
                const uint32_t tile = (uint32_t)ty * fr.tiles_x + (uint32_t)tx;
                const uint32_t key = fresh ? tile * 16u + layer : 0xFFFFFFFFu;
                const uint32_t peers = __match_any_sync(0xFFFFFFFFu, key);
                if (fresh && (uint32_t)(__ffs(peers) - 1) == lane) atomicOr(&tm[tile], 1u << layer);
            }
            if (large && (tx1 - tx0 > 1 || ty1 - ty0 > 1))  // the tiles between the corners
                for (int ty = ty0; ty <= ty1; ++ty)
                    for (int tx = tx0; tx <= tx1; ++tx) atomicOr(&tm[(size_t)ty * fr.tiles_x + tx], 1u << layer);
        }
    }
#endif
    if (__any_sync(0xFFFFFFFFu, status > 0)) {   // rare: dropped (near plane / guard band) or zero-area triangles in this warp
        const unsigned dropped = __popc(__ballot_sync(0xFFFFFFFFu, status == 1));
        const unsigned degen = __popc(__ballot_sync(0xFFFFFFFFu, status == 2));
        if (lane == 0) {
            if (dropped) atomicAdd(&counters[VS_CNT_DROPPED], (unsigned long long)dropped);
            if (degen) atomicAdd(&counters[VS_CNT_DEGENERATE], (unsigned long long)degen);
        }
    }
    uint32_t mlo = 0, mhi = 0;  // coverage of the clipped box, sample (r, c) -> bit 8r + c of mhi:mlo
    int E0 = 0, E1 = 0, E2 = 0, sx0 = 0, sx1 = 0, sx2 = 0, sy0 = 0, sy1 = 0, sy2 = 0, E0u = 0, E1u = 0;
    const bool small = valid && !large;
    // The coverage loop below runs max-over-lanes(rows) x max-over-lanes(columns) steps for the whole warp.  A lane whose box is
    // taller than wide transposes it (loop row = image column): every lane then has rows <= columns, and a warp that holds a
    // 2x7 and a 7x2 box loops 2x7 times instead of 7x7.  
    const bool transposed = small && (j1 - j0) > (i1 - i0);
    if (small) {
        // edge e_i runs (i+1) -> (i+2) and weights vertex i; sample (i0, j0)
        const int dx0 = T.X2 - T.X1, dy0 = T.Y2 - T.Y1, dx1 = T.X0 - T.X2, dy1 = T.Y0 - T.Y2;
        const int dx2 = T.X1 - T.X0, dy2 = T.Y1 - T.Y0;
        const int Sx = 256 * i0 + 128, Sy = 256 * j0 + 128;
        E0 = dx0 * (Sy - T.Y1) - dy0 * (Sx - T.X1);
        E1 = dx1 * (Sy - T.Y2) - dy1 * (Sx - T.X2);
        E2 = dx2 * (Sy - T.Y0) - dy2 * (Sx - T.X0);
        sx0 = -256 * dy0; sx1 = -256 * dy1; sx2 = -256 * dy2;  // one step along a loop row: one pixel in +x ...
        sy0 = 256 * dx0; sy1 = 256 * dx1; sy2 = 256 * dx2;     // one loop row further: one pixel in +y ...
        if (transposed) {                                       // ... or the other way round
            int t;
            t = sx0; sx0 = sy0; sy0 = t; t = sx1; sx1 = sy1; sy1 = t; t = sx2; sx2 = sy2; sy2 = t;
        }
        E0u = E0; E1u = E1;   // the unbiased values at sample (i0, j0): the depth key interpolates with these
        // covered <=> E_e > 0 || (E_e == 0 && topleft_e) <=> F_e := E_e - (topleft_e ? 0 : 1) >= 0
        E0 -= ((dy0 < 0) || (dy0 == 0 && dx0 > 0)) ? 0 : 1;
        E1 -= ((dy1 < 0) || (dy1 == 0 && dx1 > 0)) ? 0 : 1;
        E2 -= ((dy2 < 0) || (dy2 == 0 && dx2 > 0)) ? 0 : 1;
    }
    const int nr = small ? (transposed ? i1 - i0 : j1 - j0) + 1 : 0, nc = small ? (transposed ? j1 - j0 : i1 - i0) + 1 : 0;
    {
        // rows of up to 8 samples, row and column counts uniform over the warp (the lanes' boxes are alike);
        // samples of a row are visited from column cols-1 down to 0 so that each funnel shift pushes the next lower bit
        const int rows = __reduce_max_sync(0xFFFFFFFFu, nr);
        const int cols = __reduce_max_sync(0xFFFFFFFFu, nc);
        int a0 = E0 + (cols - 1) * sx0, a1 = E1 + (cols - 1) * sx1, a2 = E2 + (cols - 1) * sx2;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            if (r < rows) {
                uint32_t bits = 0;
                int c0 = a0, c1 = a1, c2 = a2;
                // exactly `cols` steps (warp-uniform): enter the unrolled sequence at the right step instead of predicating
                // all eight (the predicated-off steps of a 4-column warp still cost their issue slots)
#define VS_RD_STEP bits = __funnelshift_l((uint32_t)(c0 | c1 | c2), bits, 1); c0 -= sx0; c1 -= sx1; c2 -= sx2;
                switch (cols) {
                    case 8: VS_RD_STEP  // fall through
                    case 7: VS_RD_STEP  // fall through
                    case 6: VS_RD_STEP  // fall through
                    case 5: VS_RD_STEP  // fall through
                    case 4: VS_RD_STEP  // fall through
                    case 3: VS_RD_STEP  // fall through
                    case 2: VS_RD_STEP  // fall through
                    case 1: bits = __funnelshift_l((uint32_t)(c0 | c1 | c2), bits, 1);
                    default: break;
                }
#undef VS_RD_STEP
                bits = ~bits & 0xFFu;
                if (r < 4) mlo |= bits << (8 * r); else mhi |= bits << (8 * (r - 4));
                a0 += sy0; a1 += sy1; a2 += sy2;
            }
        }
        const uint32_t colm = 0x01010101u * ((1u << nc) - 1u);
        mlo &= colm & (nr >= 4 ? 0xFFFFFFFFu : ((1u << (8 * nr)) - 1u));
        mhi &= colm & (nr >= 8 ? 0xFFFFFFFFu : (nr > 4 ? ((1u << (8 * (nr - 4))) - 1u) : 0u));
    }
#ifndef VS_RD_NO_DEMOTE
    {
        // phase 2 runs as many rounds as the warp's LARGEST mask has bits.  A lane whose mask is far above the warp's mean (a few
        // big triangles among small ones: close-ups, silhouettes) would keep the other 31 waiting: it hands its triangle to the
        // warp-cooperative path below instead (every lane one sample of the box per round).
        const uint32_t cnt = (uint32_t)(__popc(mlo) + __popc(mhi));
        const uint32_t tot = __reduce_add_sync(0xFFFFFFFFu, cnt);
        if (cnt > max(12u, (3u * tot) >> 5)) { large = true; mlo = 0u; mhi = 0u; }
    }
#endif
    // ---------------- phase 2: lane = triangle, one covered sample of every lane's own mask per round ----------------
    if (__any_sync(0xFFFFFFFFu, (mlo | mhi) != 0u)) {
        // (a small triangle's A2 < 2^24: its box has at most 8x8 samples, so A2 and the edge values are exact in fp32)
        const int A2 = (int)T.A2;
        const float fA = __int2float_rn(A2);
        const float rA = vs_rcp_seed(fA);
        // the seeded division is __fdiv_rn's own in-range path; operands near the ends of the exponent range (a scene at
        // w ~ 1e20 or 1e-20) take the library division instead
        const float qlo = fminf(T.q0, fminf(T.q1, T.q2)), qhi = fmaxf(T.q0, fmaxf(T.q1, T.q2));
        const bool seeded = __all_sync(0xFFFFFFFFu, (mlo | mhi) == 0u || (qlo > 1e-20f && qhi < 1e20f));   // warp-uniform
        const int str_r = transposed ? 1 : W, str_c = transposed ? W : 1;   // a transposed box: loop row = image column
        const uint32_t koff = (uint32_t)(layer * plane_px) + (uint32_t)(j0 * W + i0);   // < 2^32: checked by the launcher
        const uint32_t klo = 0xFFFFFFFFu - lid;
        auto resolve = [&](int r, int c, auto seeded_tag) {
            const int e0 = E0u + r * sy0 + c * sx0;
            const int e1 = E1u + r * sy1 + c * sx1;
            const int e2 = A2 - e0 - e1;  // E0 + E1 + E2 == A2 at every point
            const float num = __fmaf_rn(__int2float_rn(e2), T.q2, __fmaf_rn(__int2float_rn(e1), T.q1, __fmul_rn(__int2float_rn(e0), T.q0)));
            const float qp = decltype(seeded_tag)::value ? vs_div_seeded(num, fA, rA) : __fdiv_rn(num, fA);
            const uint32_t idx = koff + (uint32_t)(r * str_r + c * str_c);
            unsigned long long* slot;   // one IMAD.WIDE.U32: 64-bit base + 8 * 32-bit index
            asm("mad.wide.u32 %0, %1, 8, %2;" : "=l"(slot) : "r"(idx), "l"(vkeys));
            vs_key_red(slot, ((unsigned long long)__float_as_uint(qp) << 32) | klo);
        };
        auto walk = [&](auto seeded_tag) {
            for (uint32_t m = mlo; m; m &= m - 1) {
                const int bit = __ffs(m) - 1;
                resolve(bit >> 3, bit & 7, seeded_tag);
            }
            for (uint32_t m = mhi; m; m &= m - 1) {   // (rows 4..7: empty for most warps now that rows <= columns)
                const int bit = __ffs(m) - 1;
                resolve(4 + (bit >> 3), bit & 7, seeded_tag);
            }
        };
        if (seeded) walk(std::true_type{}); else walk(std::false_type{});
    }
    // ---------------- large triangles ----------------
    bool big = false;
    if (large) {
        const unsigned long long samples = (unsigned long long)(i1 - i0 + 1) * (unsigned long long)(j1 - j0 + 1);
        if (samples > VS_BIG_SAMPLES) {
            const uint32_t slot = atomicAdd(big_count, 1u);
            if (slot < big_capacity) { big_list[slot] = make_uint2(view, gt); big = true; }
        }
    }
    uint32_t lm = __ballot_sync(0xFFFFFFFFu, large && !big);
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
        unsigned long long* plane = vkeys + blayer * plane_px;
        const float fA = __ll2float_rn(A2);
        // (only a box that did not fit the big list can be larger than VS_BIG_SAMPLES here)
        const bool lin = (unsigned long long)(bi1 - bi0 + 1) * (unsigned long long)(bj1 - bj0 + 1) <= VS_BIG_SAMPLES;
        if (bnarrow) vs_direct_large<int, true>(X0, Y0, X1, Y1, X2, Y2, q0, q1, q2, fA, bi0, bi1, bj0, bj1, W, plane, blid, lane, 0u, 1u);
        else if (lin) vs_direct_large<long long, true>(X0, Y0, X1, Y1, X2, Y2, q0, q1, q2, fA, bi0, bi1, bj0, bj1, W, plane, blid, lane, 0u, 1u);
        else vs_direct_large<long long, false>(X0, Y0, X1, Y1, X2, Y2, q0, q1, q2, fA, bi0, bi1, bj0, bj1, W, plane, blid, lane, 0u, 1u);
    }
    }   // items
}

// Triangles with very large clipped boxes (full-screen quads, close-ups of coarse meshes): every entry of
// the list is rasterised by ALL warps of the grid, warp w taking the 8x4 chunks w, w + warps, ...
__global__ void __launch_bounds__(256)
k_raster_big(const VsSceneDev sc, const VsFrame fr, const int4* __restrict__ vtx, unsigned long long* __restrict__ keys,
             const uint2* __restrict__ big_list, const uint32_t* __restrict__ big_count, uint32_t big_capacity)
{
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t gw = blockIdx.x * 8u + (threadIdx.x >> 5), warps = gridDim.x * 8u;
    const uint32_t n = min(*big_count, big_capacity);
    const int W = (int)fr.width, H = (int)fr.height;
    const size_t plane_px = (size_t)W * H;
    for (uint32_t e = 0; e < n; ++e) {
        const uint2 ent = __ldg(&big_list[e]);
        const uint4 tri = __ldg(&sc.tris[ent.y]);
        const int4* __restrict__ vv = vtx + (size_t)ent.x * sc.v_total;
        VsTri T;
        if (vs_setup_tri(__ldg(&vv[tri.x]), __ldg(&vv[tri.y]), __ldg(&vv[tri.z]), T) != 0) continue;
        int i0, i1, j0, j1;
        if (!vs_tri_pixel_bbox(T, W, H, i0, i1, j0, j1)) continue;
        const int minX = min(T.X0, min(T.X1, T.X2)), maxX = max(T.X0, max(T.X1, T.X2));
        const int minY = min(T.Y0, min(T.Y1, T.Y2)), maxY = max(T.Y0, max(T.Y1, T.Y2));
        const bool narrow = maxX - minX < 8192 && maxY - minY < 8192;
        unsigned long long* plane = keys + ((size_t)ent.x * sc.k + vs_tri_layer(tri.w)) * plane_px;
        const uint32_t lid = vs_tri_lid(tri.w);
        if (narrow) vs_direct_large<int, false>(T.X0, T.Y0, T.X1, T.Y1, T.X2, T.Y2, T.q0, T.q1, T.q2, __ll2float_rn(T.A2), i0, i1, j0, j1, W, plane, lid, lane, gw, warps);
        else vs_direct_large<long long, false>(T.X0, T.Y0, T.X1, T.Y1, T.X2, T.Y2, T.q0, T.q1, T.q2, __ll2float_rn(T.A2), i0, i1, j0, j1, W, plane, lid, lane, gw, warps);
    }
}

cudaError_t vs_launch_raster_direct(const VsSceneDev& sc, const VsFrame& fr, const VsChunk& ch, cudaStream_t st, uint32_t resident_ctas)
{
    if (sc.t_total == 0) return cudaSuccess;
    // key offsets inside one view are carried as uint32
    if ((unsigned long long)sc.k * fr.width * fr.height >= (1ull << 32)) return cudaErrorInvalidValue;
    const uint32_t bpv = (sc.t_total + VS_RD_THREADS - 1) / VS_RD_THREADS;
    const unsigned long long total = (unsigned long long)bpv * ch.views;
    if (total >= (1ull << 31)) return cudaErrorInvalidValue;
    // resident_ctas != 0: that many CTAs stride over the work items (the kernel shares the SMs with another one)
    if (resident_ctas && resident_ctas < total)
        k_raster_direct<true><<<resident_ctas, VS_RD_THREADS, 0, st>>>(sc, fr, ch.vtx, ch.keys, ch.tile_mask, ch.big_list, ch.big_count,
                                                                       ch.big_capacity, ch.counters, bpv, (uint32_t)total, 0u);
    else {
#ifdef VS_RD_BLOCK_MAJOR   // experiment switch: the grid order of the earlier versions
        const bool view_major = false;
#else
        const bool view_major = bpv <= 65535u;
#endif
        k_raster_direct<false><<<view_major ? dim3(ch.views, bpv) : dim3(bpv, ch.views), VS_RD_THREADS, 0, st>>>(
            sc, fr, ch.vtx, ch.keys, ch.tile_mask, ch.big_list, ch.big_count, ch.big_capacity, ch.counters, bpv, (uint32_t)total, view_major ? 1u : 0u);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    k_raster_big<<<resident_ctas ? 148 : 148 * 4, 256, 0, st>>>(sc, fr, ch.vtx, ch.keys, ch.big_list, ch.big_count, ch.big_capacity);
    return cudaGetLastError();
}

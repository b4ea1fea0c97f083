/*
 * vs_oracle.c -- CPU ORACLE for the k-shell rasterise-and-composite path of "Volumetric Surfaces"
 * (arXiv 2409.02482).  TEST INFRASTRUCTURE ONLY: it may be imported / linked / executed by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs, never by the product
 * path.  It shares no code with paper_2409_02482_b200/csrc (only the seeded input generators in
 * paper_2409_02482_b200/synth.py serve both sides).
 *
 * What it computes (the plain definition):
 *   For each pixel and each layer l = 0..k-1 INDEPENDENTLY, among the layer's triangles whose
 *   projection covers the pixel centre (top-left fill rule) take the one nearest the camera
 *   ("only sampling the first intersection with each surface", Fig. "sampling" c;
 *   per-layer buffers).  At that fragment interpolate UV perspective-correctly,
 *   sample the layer's SH-coefficient texture bilinearly at texel centres (PAPER.md:L339-346 Fig.
 *   "neural_textures", L441-442 §4.5), decode RGBA with the view direction (§4.5),
 *   and blend the layers in FIXED order outermost -> innermost, no sorting (§4.2
 *   "Surface Blending"; order L25, L52; no sort L121).
 *
 * Precision: everything that decides an integer (coverage, nearest triangle, tie-break) follows the
 * fixed fp32 / integer sequence of DESIGN.md §3 (= SURVEY.md Appendix A.1-A.4) so that triangle IDs are
 * bit-comparable; everything after the ID is decided (A.5-A.8) is IEEE double.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fno-fast-math -fopenmp -shared -fPIC  (oracle/build.py)
 * No tiles, no bins, no SIMD, no blocking beyond "loop the pixels of a triangle's bounding box".
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): closed-form full-screen quad; hand-counted top-left
 * fixtures (tests/golden/); double-precision ray-triangle brute force; scipy sph_harm; torch
 * grid_sample; numpy float16; SPEC.md:L478 blend example; analytic constant-layer compositing;
 * depth-sorted blend equivalence; attenuation: SPEC.md:L468-470 values, tanh(5x), closed-form tilted quads; per-vertex
 * normals: radial normals of a sphere mesh (n = the hit point's direction exactly), flat-quad coincidence with the face normal;
 * banded 8-bit format: SPEC.md:L361-378 values, grid_sample per band, float-twin renders, affine mixed-resolution
 * bands; render buffers: closed-form quad, sphere normals; backward: central finite differences of the forward;
 * footprint census (vso_count_footprints): hand-counted texels of pixel-aligned quads, early-exit and clamp cases.
 * "Parity unpinned" by the paper (readings): the sigmoid on the colour channels (Q2), the SH sign
 * convention (Q3), which normal the transparency attenuation uses (Q13: the geometric face normal) and the raw
 * (unencoded) form of the render buffers (Q13b) -- each is pinned only against its own stated definition.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define VSO_MISS 0xFFFFFFFFu
#define VSO_MAX_LAYERS 9
#define VSO_MAX_COEF 16

typedef struct {
    const float* positions;   /* [V][3] */
    const float* uvs;         /* [V][2] */
    const uint32_t* indices;  /* [T][3] */
    const void* texture;      /* [tex_h][tex_w][n][4], float or IEEE half */
    uint32_t num_vertices, num_triangles, tex_w, tex_h;
    const float* normals;     /* [V][3] per-vertex normals (need not be unit) or NULL: the geometric face normal is used */
} vso_layer;

/* camera = fx fy cx cy R[9] t[3]  (x_cam = R x_world + t; +x right, +y down, +z forward) */
enum { CAM_FX = 0, CAM_FY = 1, CAM_CX = 2, CAM_CY = 3, CAM_R = 4, CAM_T = 13 };

typedef struct {
    int32_t X, Y; /* 24.8 fixed point screen position */
    float q;      /* 1/w */
    int bad;      /* 1 = behind near plane, 2 = off the +-16384 px grid */
} vso_vtx;

typedef struct {
    int32_t X[3], Y[3];
    float q[3];
    uint32_t vi[3]; /* vertex indices after the orientation swap */
    int64_t A2;
} vso_tri;

/* ---- A.1 vertex transform (fp32-exact).  "hardware-accelerated rasterization"
 *       leaves this to the GPU; the op order is fixed here so both sides agree. ---- */
void vso_transform_vertex(const float* cam, float near_plane, const float* p, int32_t* X, int32_t* Y,
                          float* q_out, int32_t* bad)
{
    const float* R = cam + CAM_R;
    const float* t = cam + CAM_T;
    float xc = fmaf(R[0], p[0], fmaf(R[1], p[1], fmaf(R[2], p[2], t[0])));
    float yc = fmaf(R[3], p[0], fmaf(R[4], p[1], fmaf(R[5], p[2], t[1])));
    float w = fmaf(R[6], p[0], fmaf(R[7], p[1], fmaf(R[8], p[2], t[2])));
    int b = 0;
    if (!(w >= near_plane)) b = 1;
    float q = 1.0f / w;
    float xq = xc * q;
    float yq = yc * q;
    float xs = fmaf(cam[CAM_FX], xq, cam[CAM_CX]);
    float ys = fmaf(cam[CAM_FY], yq, cam[CAM_CY]);
    if (!b && !(fabsf(xs) < 16384.0f && fabsf(ys) < 16384.0f)) b = 2;
    if (b) {
        *X = 0; *Y = 0;
    } else {
        *X = (int32_t)rintf(xs * 256.0f); /* round-half-even in the default rounding mode */
        *Y = (int32_t)rintf(ys * 256.0f);
    }
    *q_out = q;
    *bad = b;
}

/* ---- A.2 triangle setup (integer-exact).  Returns 0 ok, 1 dropped (behind/offgrid), 2 zero area. */
static int vso_setup(const vso_vtx* vtx, const uint32_t* idx, vso_tri* t)
{
    for (int i = 0; i < 3; ++i) {
        const vso_vtx* v = &vtx[idx[i]];
        if (v->bad) return 1;
        t->X[i] = v->X; t->Y[i] = v->Y; t->q[i] = v->q; t->vi[i] = idx[i];
    }
    int64_t A2 = (int64_t)(t->X[1] - t->X[0]) * (int64_t)(t->Y[2] - t->Y[0])
               - (int64_t)(t->X[2] - t->X[0]) * (int64_t)(t->Y[1] - t->Y[0]);
    if (A2 == 0) return 2;
    if (A2 < 0) { /* swap vertices 1 and 2: no culling, both orientations rasterise */
        int32_t xi = t->X[1]; t->X[1] = t->X[2]; t->X[2] = xi;
        int32_t yi = t->Y[1]; t->Y[1] = t->Y[2]; t->Y[2] = yi;
        float qi = t->q[1]; t->q[1] = t->q[2]; t->q[2] = qi;
        uint32_t vi = t->vi[1]; t->vi[1] = t->vi[2]; t->vi[2] = vi;
        A2 = -A2;
    }
    t->A2 = A2;
    return 0;
}

/* ---- A.3 coverage (integer-exact).  Edge e_i runs from vertex (i+1)%3 to (i+2)%3 and weights
 *      vertex i.  Sample point of pixel (i,j) = (256 i + 128, 256 j + 128).  Top-left rule. ---- */
static int vso_covers(const vso_tri* t, int px, int py, int64_t E[3])
{
    int64_t Sx = 256 * (int64_t)px + 128, Sy = 256 * (int64_t)py + 128;
    for (int e = 0; e < 3; ++e) {
        int a = (e + 1) % 3, b = (e + 2) % 3;
        int64_t dx = (int64_t)t->X[b] - t->X[a], dy = (int64_t)t->Y[b] - t->Y[a];
        int64_t Ev = dx * (Sy - t->Y[a]) - dy * (Sx - t->X[a]);
        int topleft = (dy < 0) || (dy == 0 && dx > 0);
        E[e] = Ev;
        if (!(Ev > 0 || (Ev == 0 && topleft))) return 0;
    }
    return 1;
}

/* ---- A.4 depth key (fp32-exact): interpolated 1/w at the sample; larger = nearer. ---- */
static float vso_depth_q(const vso_tri* t, const int64_t E[3])
{
    float f0 = (float)E[0], f1 = (float)E[1], f2 = (float)E[2];
    float fA = (float)t->A2;
    float m = f0 * t->q[0];
    float num = fmaf(f2, t->q[2], fmaf(f1, t->q[1], m));
    return num / fA;
}

static inline uint32_t f32_bits(float f) { uint32_t u; memcpy(&u, &f, 4); return u; }
static inline float bits_f32(uint32_t u) { float f; memcpy(&f, &u, 4); return f; }

static inline int64_t floor_div(int64_t a, int64_t b) /* b > 0 */
{
    int64_t q = a / b, r = a % b;
    return (r != 0 && r < 0) ? q - 1 : q;
}

/* IEEE binary16 -> double, exact (pinned against numpy on all 65536 patterns). */
double vso_half_to_double(uint16_t h)
{
    int s = (h >> 15) & 1, e = (h >> 10) & 31, m = h & 1023;
    double v;
    if (e == 0) v = ldexp((double)m, -24);
    else if (e == 31) v = m ? NAN : INFINITY;
    else v = ldexp((double)(m + 1024), e - 25);
    return s ? -v : v;
}

/* ---- A.7 real orthonormal SH basis, index c = l^2 + l + m, no Condon-Shortley sign
 *      (band sizes c = {1,3,5,7}; "decoded with view direction v", L438). ---- */
void vso_sh_basis(int degree, const double* v, double* Y)
{
    const double PI = 3.14159265358979323846;
    double x = v[0], y = v[1], z = v[2];
    Y[0] = 0.5 * sqrt(1.0 / PI);
    if (degree < 1) return;
    double c1 = sqrt(3.0 / (4.0 * PI));
    Y[1] = c1 * y; Y[2] = c1 * z; Y[3] = c1 * x;
    if (degree < 2) return;
    double c2a = 0.5 * sqrt(15.0 / PI), c2b = 0.25 * sqrt(5.0 / PI), c2c = 0.25 * sqrt(15.0 / PI);
    Y[4] = c2a * x * y; Y[5] = c2a * y * z; Y[6] = c2b * (3.0 * z * z - 1.0);
    Y[7] = c2a * x * z; Y[8] = c2c * (x * x - y * y);
    if (degree < 3) return;
    double c3a = 0.25 * sqrt(35.0 / (2.0 * PI)), c3b = 0.5 * sqrt(105.0 / PI),
           c3c = 0.25 * sqrt(21.0 / (2.0 * PI)), c3d = 0.25 * sqrt(7.0 / PI), c3e = 0.25 * sqrt(105.0 / PI);
    Y[9] = c3a * y * (3.0 * x * x - y * y);
    Y[10] = c3b * x * y * z;
    Y[11] = c3c * y * (5.0 * z * z - 1.0);
    Y[12] = c3d * z * (5.0 * z * z - 3.0);
    Y[13] = c3c * x * (5.0 * z * z - 1.0);
    Y[14] = c3e * z * (x * x - y * y);
    Y[15] = c3a * x * (x * x - 3.0 * y * y);
}

static inline double tex_fetch(const void* tex, int dtype, uint32_t W, uint32_t n, int64_t ix, int64_t iy, uint32_t e)
{
    size_t o = (((size_t)iy * W + (size_t)ix) * n) * 4 + e;
    if (dtype == 2) return (double)((const uint8_t*)tex)[o]; /* stored byte t = 255 q, 0..255 (banded format below) */
    return dtype == 0 ? (double)((const float*)tex)[o] : vso_half_to_double(((const uint16_t*)tex)[o]);
}

static inline int64_t clampi(int64_t v, int64_t lo, int64_t hi) { return v < lo ? lo : (v > hi ? hi : v); }

/* ---- A.6 bilinear sample at texel centres, clamp-to-edge (PAPER.md:L339-346, L441-442:
 *      "bilinear interpolation of predictions at neighboring texels centers ... mimics how OpenGL
 *      fragment shaders access and interpolate texture values").  out[4n], layout [c][ch]. ---- */
void vso_sample_bilinear(const void* tex, int dtype, uint32_t W, uint32_t H, uint32_t n, double u, double v, double* out)
{
    double x = u * (double)W - 0.5, y = v * (double)H - 0.5;
    double x0 = floor(x), y0 = floor(y);
    double a = x - x0, b = y - y0;
    int64_t ix0 = clampi((int64_t)x0, 0, (int64_t)W - 1), ix1 = clampi((int64_t)x0 + 1, 0, (int64_t)W - 1);
    int64_t iy0 = clampi((int64_t)y0, 0, (int64_t)H - 1), iy1 = clampi((int64_t)y0 + 1, 0, (int64_t)H - 1);
    for (uint32_t e = 0; e < 4 * n; ++e) {
        double t00 = tex_fetch(tex, dtype, W, n, ix0, iy0, e), t01 = tex_fetch(tex, dtype, W, n, ix1, iy0, e);
        double t10 = tex_fetch(tex, dtype, W, n, ix0, iy1, e), t11 = tex_fetch(tex, dtype, W, n, ix1, iy1, e);
        out[e] = (1.0 - b) * ((1.0 - a) * t00 + a * t01) + b * ((1.0 - a) * t10 + a * t11);
    }
}

/* ---- The paper's baked texture format (§4.5 "Mixed resolutions", "Squeezing and quantization";
 *      SURVEY.md §8(f) NEXT-1): one 8-bit image set per SH band b = 0..deg, band b holding its 2b+1 coefficients x 4
 *      channels at its OWN resolution ("scaling texture resolution proportionally to the SH coefficient degree: the
 *      base color at the highest resolution (2048^2), the highest SH degree at the lowest (256^2)").  A stored byte t
 *      is 255 q(sh^) with q(x) = round(255 x)/255; "before rendering, we re-scale value to a hyper-parameters
 *      controlled range": sh = v_min + (v_max - v_min) q.  Each band is sampled bilinearly at its own texel centres
 *      (the stored values are what the texture unit interpolates; the affine re-scale follows), and the bands are
 *      "concatenated over the coefficient dimension" (L438) into coef[c][ch], c = b^2 .. b^2 + 2b. ---- */
typedef struct {
    const uint8_t* tex[4]; /* band b: [h[b]][w[b]][2b+1][4] */
    uint32_t w[4], h[4];
} vso_bands;

double vso_quantize(double x) /* q(x) = round(255 x) / 255, x in [0,1]; halves round away from zero (C round()) */
{
    return round(255.0 * x) / 255.0;
}

double vso_rescale(double q, double v_min, double v_max) /* sh = v_min + (v_max - v_min) q */
{
    return v_min + (v_max - v_min) * q;
}

void vso_sample_banded(const vso_bands* B, uint32_t degree, double v_min, double v_max, double u, double v, double* coef)
{
    double t[4 * 7];
    for (uint32_t b = 0; b <= degree; ++b) {
        uint32_t nb = 2 * b + 1;
        vso_sample_bilinear(B->tex[b], 2, B->w[b], B->h[b], nb, u, v, t);
        for (uint32_t e = 0; e < 4 * nb; ++e) coef[4 * (b * b) + e] = vso_rescale(t[e] / 255.0, v_min, v_max);
    }
}

/* ---- A.7 decode: s_ch = sum_c Y_c coef[c][ch]; RGBA = sigmoid(s)  (reading Q2). ---- */
void vso_decode_rgba(uint32_t n, const double* coef, const double* Y, double* rgba)
{
    for (int ch = 0; ch < 4; ++ch) {
        double s = 0.0;
        for (uint32_t c = 0; c < n; ++c) s += Y[c] * coef[4 * c + ch];
        rgba[ch] = 1.0 / (1.0 + exp(-s));
    }
}

/* ---- A.8 fixed-order front-to-back blend (with the transmittance product taken
 *      over j < i: reading Q1 in DESIGN.md).  hit[l]=0 layers contribute nothing. */
void vso_blend(uint32_t k, const double* layer_rgba, const int32_t* hit, double t_min, const double* bg, double* out)
{
    double T = 1.0, C[3] = {0.0, 0.0, 0.0};
    for (uint32_t l = 0; l < k; ++l) {
        if (!hit[l]) continue;
        const double* c = layer_rgba + 4 * l;
        double A = c[3];
        for (int i = 0; i < 3; ++i) C[i] += T * A * c[i];
        T *= (1.0 - A);
        if (T < t_min) break;
    }
    for (int i = 0; i < 3; ++i) out[i] = C[i] + T * bg[i];
    out[3] = 1.0 - T;
}

/* ---- Transparency attenuation (§4.2 "Transparency Attenuation":
 *      "multiplying predicted transparencies with a weight alpha_w that depends on the angle between the
 *      view direction and the surface normal", alpha_w = 2 Sigmoid(10 |v . n|) - 1  (= tanh(5 |v . n|));
 *      SPEC.md:L462-470).  v, n: unit vectors; n = 0 (degenerate triangle) gives 0. ---- */
double vso_alpha_attenuation(const double* v, const double* n)
{
    double d = fabs(v[0] * n[0] + v[1] * n[1] + v[2] * n[2]);
    return 2.0 * (1.0 / (1.0 + exp(-10.0 * d))) - 1.0;
}

/* Surface normal of a fragment = unit geometric normal of its triangle in world space (the paper does not
 * say where the baked renderer takes n from: reading Q13 in DESIGN.md).  Sign is irrelevant (|v . n|).
 * Zero-area triangle -> n = 0. */
void vso_face_normal(const float* p0, const float* p1, const float* p2, double* n)
{
    double a[3], b[3];
    for (int c = 0; c < 3; ++c) { a[c] = (double)p1[c] - (double)p0[c]; b[c] = (double)p2[c] - (double)p0[c]; }
    n[0] = a[1] * b[2] - a[2] * b[1];
    n[1] = a[2] * b[0] - a[0] * b[2];
    n[2] = a[0] * b[1] - a[1] * b[0];
    double len = sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
    for (int c = 0; c < 3; ++c) n[c] = len > 0.0 ? n[c] / len : 0.0;
}

/* Surface normal of a fragment when the mesh carries per-vertex normals (SURVEY.md §8(f) NEXT-2 "optional per-vertex normals";
 * PAPER.md:L279-286 "the angle between the view direction and the surface normal"): the three vertex normals are
 * interpolated with the fragment's perspective-correct barycentrics b'_i (A.5) and the sum is renormalised; a vanishing sum
 * gives n = 0 (alpha_w = 0), like a zero-area triangle does for the face normal.  nv = the three vertex normals in the order of
 * the weights b. */
void vso_interp_normal(const double* b, const float* n0, const float* n1, const float* n2, double* n)
{
    for (int c = 0; c < 3; ++c) n[c] = b[0] * (double)n0[c] + b[1] * (double)n1[c] + b[2] * (double)n2[c];
    double len = sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
    for (int c = 0; c < 3; ++c) n[c] = len > 0.0 ? n[c] / len : 0.0;
}

/* view direction of pixel (i,j): camera -> scene, world frame, unit (reading Q4) */
static void view_dir(const float* cam, int px, int py, double* v)
{
    double dx = ((double)px + 0.5 - (double)cam[CAM_CX]) / (double)cam[CAM_FX];
    double dy = ((double)py + 0.5 - (double)cam[CAM_CY]) / (double)cam[CAM_FY];
    double dz = 1.0;
    const float* R = cam + CAM_R;
    double w[3];
    for (int c = 0; c < 3; ++c) w[c] = (double)R[0 + c] * dx + (double)R[3 + c] * dy + (double)R[6 + c] * dz;
    double nrm = sqrt(w[0] * w[0] + w[1] * w[1] + w[2] * w[2]);
    for (int c = 0; c < 3; ++c) v[c] = w[c] / nrm;
}

/*
 * Render ONE view.
 *   out_rgba  [H][W][4] double                      (required)
 *   out_ids   [k][H][W] uint32, miss = 0xFFFFFFFF   (required)
 *   out_qp    [k][H][W] float, interpolated 1/w of the winning fragment, 0 on miss   (optional)
 *   out_layer_rgba [k][H][W][4] double, decoded per-layer RGBA, 0 on miss            (optional)
 *   out_layer_uv   [k][H][W][2] double, interpolated UV, 0 on miss                   (optional)
 *   stats[0] += triangles dropped (near plane / guard band), stats[1] += zero-area triangles
 *   out_layer_normal [k][H][W][3] double, unit normal of the winning fragment (the face normal of its triangle, or the
 *                   interpolated vertex normal if the layer has `normals`; world space), signed so that it faces the viewer
 *                   (v . n <= 0), 0 on miss or when the normal vanishes                                 (optional, last argument)
 *   attenuate != 0: every fragment's opacity is multiplied by alpha_w(v, that normal) before blending
 *                   (PAPER.md:L279-286); the alpha of out_layer_rgba is the attenuated one
 * Returns 0, or -1 on bad arguments / allocation failure.
 */
static int render_impl(const vso_layer* layers, const vso_bands* btex, double v_min, double v_max, uint32_t k,
                       uint32_t sh_degree, int tex_dtype, const float* cam,
                       uint32_t width, uint32_t height, float near_plane, double t_min, const double* bg,
                       double* out_rgba, uint32_t* out_ids, float* out_qp, double* out_layer_rgba,
                       double* out_layer_uv, uint64_t* stats, int num_threads, int attenuate, double* out_layer_normal)
{
    if (!layers || k < 1 || k > VSO_MAX_LAYERS || sh_degree > 3 || !cam || !out_rgba || !out_ids || !(near_plane > 0.0f))
        return -1;
    const uint32_t n = (sh_degree + 1) * (sh_degree + 1);
    const size_t P = (size_t)width * height;
#ifdef _OPENMP
    if (num_threads < 1) num_threads = omp_get_max_threads();
#else
    num_threads = 1;
#endif
    uint64_t* keys = (uint64_t*)calloc(P * k, sizeof(uint64_t));
    vso_vtx** vtx = (vso_vtx**)calloc(k, sizeof(vso_vtx*));
    if (!keys || !vtx) { free(keys); free(vtx); return -1; }
    uint64_t dropped = 0, degenerate = 0;

    /* S1: transform every vertex of every layer */
    for (uint32_t l = 0; l < k; ++l) {
        vtx[l] = (vso_vtx*)malloc(sizeof(vso_vtx) * (layers[l].num_vertices ? layers[l].num_vertices : 1));
        if (!vtx[l]) return -1;
#pragma omp parallel for num_threads(num_threads) schedule(static)
        for (int64_t i = 0; i < (int64_t)layers[l].num_vertices; ++i) {
            vso_vtx* o = &vtx[l][i];
            int32_t bad;
            vso_transform_vertex(cam, near_plane, layers[l].positions + 3 * i, &o->X, &o->Y, &o->q, &bad);
            o->bad = bad;
        }
    }

    /* S2-S4: per layer, per triangle, per pixel of its bounding box: coverage + nearest resolve.
     * Work items = (layer, band of rows); each writes a disjoint part of the key buffer. */
    int bands = (num_threads + (int)k - 1) / (int)k;
    if (bands < 1) bands = 1;
    if ((uint32_t)bands > height) bands = (int)height ? (int)height : 1;
    int items = (int)k * bands;
#pragma omp parallel for num_threads(num_threads) schedule(dynamic, 1) reduction(+ : dropped, degenerate)
    for (int it = 0; it < items; ++it) {
        uint32_t l = (uint32_t)(it / bands);
        int band = it % bands;
        int64_t row0 = (int64_t)height * band / bands, row1 = (int64_t)height * (band + 1) / bands;
        uint64_t* kb = keys + (size_t)l * P;
        const vso_layer* L = &layers[l];
        for (uint32_t t = 0; t < L->num_triangles; ++t) {
            vso_tri tri;
            int r = vso_setup(vtx[l], L->indices + 3 * (size_t)t, &tri);
            if (r) { if (band == 0) { if (r == 1) dropped++; else degenerate++; } continue; }
            int32_t minX = tri.X[0], maxX = tri.X[0], minY = tri.Y[0], maxY = tri.Y[0];
            for (int i = 1; i < 3; ++i) {
                if (tri.X[i] < minX) minX = tri.X[i];
                if (tri.X[i] > maxX) maxX = tri.X[i];
                if (tri.Y[i] < minY) minY = tri.Y[i];
                if (tri.Y[i] > maxY) maxY = tri.Y[i];
            }
            /* pixels whose sample point 256 i + 128 lies in [min, max] */
            int64_t i0 = -floor_div(-((int64_t)minX - 128), 256), i1 = floor_div((int64_t)maxX - 128, 256);
            int64_t j0 = -floor_div(-((int64_t)minY - 128), 256), j1 = floor_div((int64_t)maxY - 128, 256);
            if (i0 < 0) i0 = 0;
            if (i1 > (int64_t)width - 1) i1 = (int64_t)width - 1;
            if (j0 < row0) j0 = row0;
            if (j1 > row1 - 1) j1 = row1 - 1;
            for (int64_t j = j0; j <= j1; ++j)
                for (int64_t i = i0; i <= i1; ++i) {
                    int64_t E[3];
                    if (!vso_covers(&tri, (int)i, (int)j, E)) continue;
                    float qp = vso_depth_q(&tri, E);
                    uint64_t key = ((uint64_t)f32_bits(qp) << 32) | (uint64_t)(0xFFFFFFFFu - t);
                    uint64_t* slot = &kb[(size_t)j * width + (size_t)i];
                    if (key > *slot) *slot = key; /* nearer wins; equal depth -> lowest triangle index */
                }
        }
    }
    if (stats) { stats[0] += dropped; stats[1] += degenerate; }

    for (uint32_t l = 0; l < k; ++l)
        for (size_t p = 0; p < P; ++p) {
            uint64_t key = keys[(size_t)l * P + p];
            out_ids[(size_t)l * P + p] = key ? (0xFFFFFFFFu - (uint32_t)(key & 0xFFFFFFFFu)) : VSO_MISS;
            if (out_qp) out_qp[(size_t)l * P + p] = key ? bits_f32((uint32_t)(key >> 32)) : 0.0f;
        }
    if (out_layer_rgba) memset(out_layer_rgba, 0, sizeof(double) * P * k * 4);
    if (out_layer_uv) memset(out_layer_uv, 0, sizeof(double) * P * k * 2);
    if (out_layer_normal) memset(out_layer_normal, 0, sizeof(double) * P * k * 3);

    /* S5-S7: shade and composite, per pixel, in double */
#pragma omp parallel for num_threads(num_threads) schedule(dynamic, 4)
    for (int64_t j = 0; j < (int64_t)height; ++j) {
        double coef[4 * VSO_MAX_COEF];
        for (int64_t i = 0; i < (int64_t)width; ++i) {
            size_t p = (size_t)j * width + (size_t)i;
            double v[3], Y[VSO_MAX_COEF];
            view_dir(cam, (int)i, (int)j, v);
            vso_sh_basis((int)sh_degree, v, Y);
            double lrgba[4 * VSO_MAX_LAYERS];
            int32_t hit[VSO_MAX_LAYERS];
            for (uint32_t l = 0; l < k; ++l) {
                uint32_t id = out_ids[(size_t)l * P + p];
                hit[l] = (id != VSO_MISS);
                if (!hit[l]) continue;
                const vso_layer* L = &layers[l];
                vso_tri tri;
                int64_t E[3];
                vso_setup(vtx[l], L->indices + 3 * (size_t)id, &tri);
                vso_covers(&tri, (int)i, (int)j, E);
                /* A.5 perspective-correct barycentrics: b'_i proportional to E_i q_i */
                double g[3], gs = 0.0;
                for (int c = 0; c < 3; ++c) { g[c] = (double)E[c] * (double)tri.q[c]; gs += g[c]; }
                double uu = 0.0, vv = 0.0, bw[3];
                for (int c = 0; c < 3; ++c) {
                    double b = g[c] / gs;
                    bw[c] = b;
                    uu += b * (double)L->uvs[2 * (size_t)tri.vi[c] + 0];
                    vv += b * (double)L->uvs[2 * (size_t)tri.vi[c] + 1];
                }
                if (btex) vso_sample_banded(&btex[l], sh_degree, v_min, v_max, uu, vv, coef);
                else vso_sample_bilinear(L->texture, tex_dtype, L->tex_w, L->tex_h, n, uu, vv, coef);
                vso_decode_rgba(n, coef, Y, lrgba + 4 * l);
                if (attenuate || out_layer_normal) {
                    const uint32_t* ix = L->indices + 3 * (size_t)id;
                    double nrm[3];
                    if (L->normals)
                        vso_interp_normal(bw, L->normals + 3 * (size_t)tri.vi[0], L->normals + 3 * (size_t)tri.vi[1],
                                          L->normals + 3 * (size_t)tri.vi[2], nrm);
                    else
                        vso_face_normal(L->positions + 3 * (size_t)ix[0], L->positions + 3 * (size_t)ix[1],
                                        L->positions + 3 * (size_t)ix[2], nrm);
                    if (attenuate) lrgba[4 * l + 3] *= vso_alpha_attenuation(v, nrm);
                    if (out_layer_normal) { /* "Surface normals" buffer: oriented towards the viewer */
                        double sgn = (v[0] * nrm[0] + v[1] * nrm[1] + v[2] * nrm[2]) > 0.0 ? -1.0 : 1.0;
                        for (int c = 0; c < 3; ++c) out_layer_normal[((size_t)l * P + p) * 3 + c] = sgn * nrm[c];
                    }
                }
                if (out_layer_rgba) memcpy(out_layer_rgba + ((size_t)l * P + p) * 4, lrgba + 4 * l, 4 * sizeof(double));
                if (out_layer_uv) { out_layer_uv[((size_t)l * P + p) * 2] = uu; out_layer_uv[((size_t)l * P + p) * 2 + 1] = vv; }
            }
            /* A.8: the t_min early exit lives in vso_blend (layers past it are shaded but unused) */
            vso_blend(k, lrgba, hit, t_min, bg, out_rgba + p * 4);
        }
    }

    for (uint32_t l = 0; l < k; ++l) free(vtx[l]);
    free(vtx);
    free(keys);
    return 0;
}

int vso_render(const vso_layer* layers, uint32_t k, uint32_t sh_degree, int tex_dtype, const float* cam,
               uint32_t width, uint32_t height, float near_plane, double t_min, const double* bg,
               double* out_rgba, uint32_t* out_ids, float* out_qp, double* out_layer_rgba,
               double* out_layer_uv, uint64_t* stats, int num_threads, int attenuate, double* out_layer_normal)
{
    return render_impl(layers, NULL, 0.0, 0.0, k, sh_degree, tex_dtype, cam, width, height, near_plane, t_min, bg, out_rgba,
                       out_ids, out_qp, out_layer_rgba, out_layer_uv, stats, num_threads, attenuate, out_layer_normal);
}

/* The same render with the paper's banded 8-bit textures (layers[l].texture is ignored; bands[l] is used). */
int vso_render_banded(const vso_layer* layers, const vso_bands* bands, double v_min, double v_max, uint32_t k,
                      uint32_t sh_degree, const float* cam, uint32_t width, uint32_t height, float near_plane,
                      double t_min, const double* bg, double* out_rgba, uint32_t* out_ids, float* out_qp,
                      double* out_layer_rgba, double* out_layer_uv, uint64_t* stats, int num_threads, int attenuate,
                      double* out_layer_normal)
{
    if (!bands) return -1;
    for (uint32_t l = 0; l < k && l < VSO_MAX_LAYERS; ++l)
        for (uint32_t b = 0; b <= sh_degree && b < 4; ++b)
            if (!bands[l].tex[b] || bands[l].w[b] == 0 || bands[l].h[b] == 0) return -1;
    return render_impl(layers, bands, v_min, v_max, k, sh_degree, 2, cam, width, height, near_plane, t_min, bg, out_rgba,
                       out_ids, out_qp, out_layer_rgba, out_layer_uv, stats, num_threads, attenuate, out_layer_normal);
}

/*
 * Backward pass to the texels (§4.5: the baked textures are optimised through
 * the same bilinear lookup "such that when displayed in our real-time renderer, images match ... those synthesized by our
 * differentiable renderer").  Given the triangle ids of a forward render of the SAME view and settings
 * (`ids` [k][H][W], as written by vso_render) and an upstream gradient g = dL/d(out_rgba) [H][W][4], ACCUMULATES
 * dL/d(texture of layer l) into grad_tex[l] ([tex_h][tex_w][n][4] double, same layout as the texture), by the chain rule
 * through A.8 blend -> A.7 sigmoid / SH dot -> A.6 bilinear weights (and alpha_w, a constant factor, if `attenuate`):
 *   out_rgb = sum_l T_l A_l rgb_l + T_end bg,  out_a = 1 - T_end,  T_{l+1} = T_l (1 - A_l)
 *   R_end = bg . g_rgb - g_a ;  R_{l-1} = A_l (rgb_l . g_rgb) + (1 - A_l) R_l       (what lies behind layer l, per unit T)
 *   dL/dA_l = T_l (rgb_l . g_rgb - R_l) ;  dL/drgb_l = T_l A_l g_rgb
 *   dL/ds_ch = dL/drgb_ch rgb_ch (1 - rgb_ch) ;  dL/ds_3 = dL/dA alpha_w sigma(s_3) (1 - sigma(s_3))
 *   dL/dtex[q][c][ch] += w_q Y_c dL/ds_ch           for the four texels q of the footprint
 * The early exit is a constant of the differentiation (layers behind it get no gradient); coverage and UVs do not depend
 * on the textures.  Float textures only (dtype 0 / 1).  grad_tex[l] == NULL: the gradient of layer l is not wanted (a full-size
 * fp64 gradient texture is 2 GB per layer; the tests take the layers one at a time).  Returns 0, or -1 on bad arguments.
 */
int vso_render_backward(const vso_layer* layers, uint32_t k, uint32_t sh_degree, int tex_dtype, const float* cam,
                        uint32_t width, uint32_t height, float near_plane, double t_min, const double* bg,
                        const uint32_t* ids, const double* grad_out, double* const* grad_tex, int attenuate, int num_threads)
{
    if (!layers || k < 1 || k > VSO_MAX_LAYERS || sh_degree > 3 || !cam || !ids || !grad_out || !grad_tex || tex_dtype > 1)
        return -1;
    const uint32_t n = (sh_degree + 1) * (sh_degree + 1);
    const size_t P = (size_t)width * height;
#ifdef _OPENMP
    if (num_threads < 1) num_threads = omp_get_max_threads();
#else
    num_threads = 1;
#endif
    vso_vtx** vtx = (vso_vtx**)calloc(k, sizeof(vso_vtx*));
    if (!vtx) return -1;
    for (uint32_t l = 0; l < k; ++l) {
        vtx[l] = (vso_vtx*)malloc(sizeof(vso_vtx) * (layers[l].num_vertices ? layers[l].num_vertices : 1));
        if (!vtx[l]) return -1;
        for (int64_t i = 0; i < (int64_t)layers[l].num_vertices; ++i) {
            int32_t bad;
            vso_transform_vertex(cam, near_plane, layers[l].positions + 3 * i, &vtx[l][i].X, &vtx[l][i].Y, &vtx[l][i].q, &bad);
            vtx[l][i].bad = bad;
        }
    }
#pragma omp parallel for num_threads(num_threads) schedule(dynamic, 4)
    for (int64_t j = 0; j < (int64_t)height; ++j) {
        for (int64_t i = 0; i < (int64_t)width; ++i) {
            size_t p = (size_t)j * width + (size_t)i;
            double v[3], Y[VSO_MAX_COEF];
            view_dir(cam, (int)i, (int)j, v);
            vso_sh_basis((int)sh_degree, v, Y);
            /* forward, keeping what the backward needs */
            double rgb[VSO_MAX_LAYERS][3], sig3[VSO_MAX_LAYERS], aw[VSO_MAX_LAYERS], A[VSO_MAX_LAYERS], Tl[VSO_MAX_LAYERS];
            double wq[VSO_MAX_LAYERS][4];
            int64_t tx[VSO_MAX_LAYERS][4], ty[VSO_MAX_LAYERS][4];
            int order[VSO_MAX_LAYERS], cnt = 0;
            double T = 1.0;
            for (uint32_t l = 0; l < k; ++l) {
                uint32_t id = ids[(size_t)l * P + p];
                if (id == VSO_MISS) continue;
                const vso_layer* L = &layers[l];
                vso_tri tri;
                int64_t E[3];
                vso_setup(vtx[l], L->indices + 3 * (size_t)id, &tri);
                vso_covers(&tri, (int)i, (int)j, E);
                double g[3], gs = 0.0, uu = 0.0, vv = 0.0, bw[3];
                for (int c = 0; c < 3; ++c) { g[c] = (double)E[c] * (double)tri.q[c]; gs += g[c]; }
                for (int c = 0; c < 3; ++c) {
                    double b = g[c] / gs;
                    bw[c] = b;
                    uu += b * (double)L->uvs[2 * (size_t)tri.vi[c] + 0];
                    vv += b * (double)L->uvs[2 * (size_t)tri.vi[c] + 1];
                }
                /* A.6 footprint and weights */
                double x = uu * (double)L->tex_w - 0.5, y = vv * (double)L->tex_h - 0.5;
                double x0 = floor(x), y0 = floor(y), a = x - x0, b = y - y0;
                int64_t ix0 = clampi((int64_t)x0, 0, (int64_t)L->tex_w - 1), ix1 = clampi((int64_t)x0 + 1, 0, (int64_t)L->tex_w - 1);
                int64_t iy0 = clampi((int64_t)y0, 0, (int64_t)L->tex_h - 1), iy1 = clampi((int64_t)y0 + 1, 0, (int64_t)L->tex_h - 1);
                tx[l][0] = ix0; ty[l][0] = iy0; wq[l][0] = (1.0 - b) * (1.0 - a);
                tx[l][1] = ix1; ty[l][1] = iy0; wq[l][1] = (1.0 - b) * a;
                tx[l][2] = ix0; ty[l][2] = iy1; wq[l][2] = b * (1.0 - a);
                tx[l][3] = ix1; ty[l][3] = iy1; wq[l][3] = b * a;
                double sch[4] = {0.0, 0.0, 0.0, 0.0};
                for (uint32_t c = 0; c < n; ++c)
                    for (int ch = 0; ch < 4; ++ch) {
                        double t = 0.0;
                        for (int q = 0; q < 4; ++q) t += wq[l][q] * tex_fetch(L->texture, tex_dtype, L->tex_w, n, tx[l][q], ty[l][q], 4 * c + ch);
                        sch[ch] += Y[c] * t;
                    }
                for (int ch = 0; ch < 3; ++ch) rgb[l][ch] = 1.0 / (1.0 + exp(-sch[ch]));
                sig3[l] = 1.0 / (1.0 + exp(-sch[3]));
                aw[l] = 1.0;
                if (attenuate) {
                    const uint32_t* ix = L->indices + 3 * (size_t)id;
                    double nrm[3];
                    if (L->normals)
                        vso_interp_normal(bw, L->normals + 3 * (size_t)tri.vi[0], L->normals + 3 * (size_t)tri.vi[1],
                                          L->normals + 3 * (size_t)tri.vi[2], nrm);
                    else
                        vso_face_normal(L->positions + 3 * (size_t)ix[0], L->positions + 3 * (size_t)ix[1], L->positions + 3 * (size_t)ix[2], nrm);
                    aw[l] = vso_alpha_attenuation(v, nrm);
                }
                A[l] = sig3[l] * aw[l];
                Tl[l] = T;
                order[cnt++] = (int)l;
                T *= (1.0 - A[l]);
                if (T < t_min) break;
            }
            /* backward */
            const double* go = grad_out + p * 4;
            double R = bg[0] * go[0] + bg[1] * go[1] + bg[2] * go[2] - go[3];
            for (int o = cnt - 1; o >= 0; --o) {
                int l = order[o];
                double cg = rgb[l][0] * go[0] + rgb[l][1] * go[1] + rgb[l][2] * go[2];
                double ds[4];
                for (int ch = 0; ch < 3; ++ch) ds[ch] = Tl[l] * A[l] * go[ch] * rgb[l][ch] * (1.0 - rgb[l][ch]);
                ds[3] = Tl[l] * (cg - R) * aw[l] * sig3[l] * (1.0 - sig3[l]);
                R = A[l] * cg + (1.0 - A[l]) * R;
                const vso_layer* L = &layers[l];
                if (!grad_tex[l]) continue;
                for (int q = 0; q < 4; ++q)
                    for (uint32_t c = 0; c < n; ++c)
                        for (int ch = 0; ch < 4; ++ch) {
                            double* slot = grad_tex[l] + (((size_t)ty[l][q] * L->tex_w + (size_t)tx[l][q]) * n + c) * 4 + ch;
                            double add = wq[l][q] * Y[c] * ds[ch];
#pragma omp atomic
                            *slot += add;
                        }
            }
        }
    }
    for (uint32_t l = 0; l < k; ++l) free(vtx[l]);
    free(vtx);
    return 0;
}

/*
 * Footprint census of ONE rendered view -- the numerator of the roofline (B_tex = "unique texels referenced by
 * the 2x2 footprints of *shaded* fragments ... counted, not assumed: an instrumented pass or the oracle").
 * Inputs are what vso_render produced for the view: ids [k][H][W], layer_rgba [k][H][W][4] (alpha = the blend weight A of
 * A.8, after alpha_w if it was enabled) and layer_uv [k][H][W][2].  Per pixel, the layers are walked in blend order with the
 * A.8 recurrence (T *= 1 - A; stop once T < t_min): every hit layer reached before the stop -- the stopping layer included --
 * is a COMPOSITED fragment.  Each composited fragment marks the four texels of its A.6 footprint (x = u W - 0.5, floor,
 * clamp-to-edge; texels of weight 0 count: they are fetched) in marks[l] ([tex_h][tex_w] bytes, set to 1, never cleared
 * here, so several views may be accumulated).  out[0] += composited fragments, out[1] += texels newly marked by this call.
 * Returns 0, or -1 on bad arguments.
 */
int vso_count_footprints(const vso_layer* layers, uint32_t k, uint32_t width, uint32_t height, double t_min,
                         const uint32_t* ids, const double* layer_rgba, const double* layer_uv, uint8_t* const* marks,
                         uint64_t* out)
{
    if (!layers || k < 1 || k > VSO_MAX_LAYERS || !ids || !layer_rgba || !layer_uv || !marks || !out) return -1;
    const size_t P = (size_t)width * height;
    uint64_t frags = 0, fresh = 0;
    for (size_t p = 0; p < P; ++p) {
        double T = 1.0;
        for (uint32_t l = 0; l < k; ++l) {
            if (ids[(size_t)l * P + p] == VSO_MISS) continue;
            const vso_layer* L = &layers[l];
            frags++;
            double u = layer_uv[((size_t)l * P + p) * 2], v = layer_uv[((size_t)l * P + p) * 2 + 1];
            double x0 = floor(u * (double)L->tex_w - 0.5), y0 = floor(v * (double)L->tex_h - 0.5);
            int64_t ix[2] = {clampi((int64_t)x0, 0, (int64_t)L->tex_w - 1), clampi((int64_t)x0 + 1, 0, (int64_t)L->tex_w - 1)};
            int64_t iy[2] = {clampi((int64_t)y0, 0, (int64_t)L->tex_h - 1), clampi((int64_t)y0 + 1, 0, (int64_t)L->tex_h - 1)};
            for (int b = 0; b < 2; ++b)
                for (int a = 0; a < 2; ++a) {
                    uint8_t* m = &marks[l][(size_t)iy[b] * L->tex_w + (size_t)ix[a]];
                    if (!*m) { *m = 1; fresh++; }
                }
            T *= (1.0 - layer_rgba[((size_t)l * P + p) * 4 + 3]);
            if (T < t_min) break;
        }
    }
    out[0] += frags;
    out[1] += fresh;
    return 0;
}

int vso_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * c_abi_smoke.c -- a plain C99 caller of include/vs.h (the boundary is a C ABI, not a Python binding).
 * Compiled by tests/test_c_abi.py with `gcc -std=c99 -pedantic -Wall -Werror -Iinclude` and linked against libvs_b200.so and
 * the CUDA runtime; the header must therefore be valid C99 on its own.
 *
 * Scene: one layer, one viewport-filling quad (two triangles) at depth 2 whose 2x2 fp32 texture holds only band-0
 * coefficients, given as HOST arrays.  Closed form: every pixel is sigmoid(Y00 * coefficient) per channel,
 * composited over a black background: rgb = A * sigmoid(.), alpha = A.  Checks argument validation, vs_scene_create,
 * vs_render (asynchronous: the stream is synchronised here), the triangle-id AOV of the two pixels on either side of the
 * diagonal, vs_render_host, vs_query_last_render and vs_scene_destroy.  Exit code 0 = pass.
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <cuda_runtime_api.h>

#include "vs.h"

#define W 16
#define H 12
#define CHECK(cond, msg)                                                       \
    do {                                                                       \
        if (!(cond)) {                                                         \
            fprintf(stderr, "FAIL %s:%d: %s (%s)\n", __FILE__, __LINE__, msg, vs_last_error()); \
            return 1;                                                          \
        }                                                                      \
    } while (0)

int main(void)
{
    const float f = 64.0f, d = 2.0f;
    const float hx = (W / 2.0f) * d / f, hy = (H / 2.0f) * d / f;
    float positions[4][3] = {{-hx, -hy, d}, {hx, -hy, d}, {hx, hy, d}, {-hx, hy, d}};
    float uvs[4][2] = {{0, 0}, {1, 0}, {1, 1}, {0, 1}};
    uint32_t indices[2][3] = {{0, 1, 2}, {0, 2, 3}};
    const double Y00 = 0.28209479177387814;
    const double logits[4] = {0.7, -0.4, 0.2, 1.1};
    float texture[2][2][1][4];
    double want[4];
    vs_layer_desc layer;
    vs_scene_desc desc;
    vs_scene* scene = NULL;
    vs_camera cam;
    vs_render_params params;
    vs_render_stats stats;
    float *d_rgba = NULL, *h_rgba = NULL, *h_rgba2 = NULL;
    uint32_t *d_ids = NULL, *h_ids = NULL;
    cudaStream_t stream;
    int i, j, c;

    for (i = 0; i < 2; ++i)
        for (j = 0; j < 2; ++j)
            for (c = 0; c < 4; ++c) texture[i][j][0][c] = (float)(logits[c] / Y00);
    for (c = 0; c < 4; ++c) want[c] = 1.0 / (1.0 + exp(-(double)texture[0][0][0][c] * Y00));

    /* argument validation happens before any CUDA work */
    CHECK(vs_scene_create(NULL, NULL, &scene) == VS_ERR_INVALID_ARG && scene == NULL, "NULL descriptor must be rejected");
    CHECK(strlen(vs_last_error()) > 0, "vs_last_error must describe the failure");
    CHECK(strstr(vs_version(), "sm_100a") != NULL, "version string");

    memset(&layer, 0, sizeof layer);
    layer.positions = &positions[0][0]; layer.uvs = &uvs[0][0]; layer.num_vertices = 4;
    layer.indices = &indices[0][0]; layer.num_triangles = 2;
    layer.texture = texture; layer.tex_w = 2; layer.tex_h = 2;
    memset(&desc, 0, sizeof desc);
    desc.num_layers = 1; desc.sh_degree = 0; desc.tex_dtype = VS_F32; desc.memory = VS_MEM_HOST; desc.layers = &layer;

    CHECK(cudaStreamCreate(&stream) == cudaSuccess, "cudaStreamCreate");
    CHECK(vs_scene_create(&desc, stream, &scene) == VS_OK && scene != NULL, "vs_scene_create");

    memset(&cam, 0, sizeof cam);
    cam.fx = f; cam.fy = f; cam.cx = W / 2.0f; cam.cy = H / 2.0f;
    cam.R[0] = cam.R[4] = cam.R[8] = 1.0f;
    memset(&params, 0, sizeof params);
    params.width = W; params.height = H; params.near_plane = 0.05f; params.t_min = 1.0f / 16384.0f;

    CHECK(cudaMalloc((void**)&d_rgba, sizeof(float) * W * H * 4) == cudaSuccess, "cudaMalloc");
    CHECK(cudaMalloc((void**)&d_ids, sizeof(uint32_t) * W * H) == cudaSuccess, "cudaMalloc");
    h_rgba = (float*)malloc(sizeof(float) * W * H * 4);
    h_rgba2 = (float*)malloc(sizeof(float) * W * H * 4);
    h_ids = (uint32_t*)malloc(sizeof(uint32_t) * W * H);
    CHECK(h_rgba && h_rgba2 && h_ids, "malloc");

    params.width = 0;
    CHECK(vs_render(scene, &cam, 1, &params, d_rgba, d_ids, stream) == VS_ERR_INVALID_ARG, "empty image must be rejected");
    params.width = W;
    CHECK(vs_render(scene, &cam, 1, &params, d_rgba, d_ids, stream) == VS_OK, "vs_render");
    /* the call is asynchronous: the outputs are complete once the stream has drained */
    CHECK(cudaMemcpyAsync(h_rgba, d_rgba, sizeof(float) * W * H * 4, cudaMemcpyDeviceToHost, stream) == cudaSuccess, "copy");
    CHECK(cudaMemcpyAsync(h_ids, d_ids, sizeof(uint32_t) * W * H, cudaMemcpyDeviceToHost, stream) == cudaSuccess, "copy");
    CHECK(cudaStreamSynchronize(stream) == cudaSuccess, "sync");

    for (j = 0; j < H; ++j)
        for (i = 0; i < W; ++i) {
            const float* px = h_rgba + ((size_t)j * W + i) * 4;
            for (c = 0; c < 3; ++c) CHECK(fabs(px[c] - want[3] * want[c]) <= 1e-4, "colour differs from the closed form");
            CHECK(fabs(px[3] - want[3]) <= 1e-4, "alpha differs from the closed form");
            CHECK(h_ids[(size_t)j * W + i] <= 1u, "every pixel is covered by one of the two triangles");
        }
    /* the diagonal runs from the top-left to the bottom-right corner: triangle 0 (0,1,2) owns the upper right half */
    CHECK(h_ids[(size_t)0 * W + (W - 1)] == 0u && h_ids[(size_t)(H - 1) * W + 0] == 1u, "triangle ids of the two halves");

    CHECK(vs_query_last_render(scene, &stats) == VS_OK, "vs_query_last_render");
    CHECK(stats.kernel_launches > 0 && stats.dropped_triangles == 0 && stats.degenerate_triangles == 0, "stats");

    CHECK(vs_render_host(scene, &cam, 1, &params, h_rgba2, NULL, stream) == VS_OK, "vs_render_host");
    CHECK(memcmp(h_rgba, h_rgba2, sizeof(float) * W * H * 4) == 0, "vs_render_host must give the same image bit for bit");

    vs_scene_destroy(scene);
    vs_scene_destroy(NULL);
    cudaFree(d_rgba); cudaFree(d_ids); cudaStreamDestroy(stream);
    free(h_rgba); free(h_rgba2); free(h_ids);
    printf("c_abi_smoke ok: %dx%d quad, rgba = (%.6f %.6f %.6f %.6f)\n", W, H, want[3] * want[0], want[3] * want[1], want[3] * want[2], want[3]);
    return 0;
}

// vs_internal.cuh -- the few things of vs_api.cu that another translation unit of the library may use (vs_noalloc.cu).
// The scene's internals stay private to vs_api.cu.
#pragma once
#include "../../include/vs.h"
#include "vs_common.cuh"

// Argument checks of vs_render (clears the thread's error text first).
vs_status vs_internal_validate_render(const vs_scene* scene, const vs_camera* cams, uint32_t n, const vs_render_params* p,
                                      const void* out_rgba);
// The immutable device-side description of a scene, its texture element type and its device ordinal.
void vs_internal_scene_view(const vs_scene* scene, const VsSceneDev** dev, int* tex_f16, int* device);
// Sets the calling thread's vs_last_error() text and returns `s`.
vs_status vs_internal_fail(vs_status s, const char* message);

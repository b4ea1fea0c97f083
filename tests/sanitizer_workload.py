#!/usr/bin/env python
"""Workload for `compute-sanitizer --tool memcheck|racecheck|initcheck python tests/sanitizer_workload.py`:
every render entry point of the C-ABI on C1 and on a reduced C2 (fp16 SH-2: the tensor-core path of k_shade) and a reduced
C4 (fp16 SH-3), on both raster paths, plus the banded format, the per-layer buffers, the backward pass, the texel census,
VS_FLAG_ATTENUATION, VS_FLAG_OVERLAP and the host-output call.  Sizes are small because the tools slow kernels down by
10-100x.  Prints one line per case; the tool's own summary is what profiles/r2_sanitizer.md records."""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2409_02482_b200 import binding as b, synth  # noqa: E402


def run(sc, tag):
    r = b.Renderer(sc)
    W, H, B, k = sc.width, sc.height, len(sc.cameras), sc.k
    banded = sc.layers[0].band_textures is not None
    out = torch.empty((B, H, W, 4), dtype=torch.float32, device="cuda")
    ids = torch.empty((B, k, H, W), dtype=torch.int32, device="cuda")
    for name, flags, chunk in (("direct", 0, 0), ("direct, 1 view per chunk", 0, 1), ("tiled", b.VS_FLAG_TILED_PATH, 0),
                               ("overlap", b.VS_FLAG_OVERLAP, 1), ("attenuation", b.VS_FLAG_ATTENUATION, 0),
                               ("census", b.VS_FLAG_COUNT_TEXELS, 0), ("timing", b.VS_FLAG_KERNEL_TIMING, 0)):
        p = b.make_params(W, H, sc.near_plane, sc.t_min, sc.background, flags, chunk)
        b.vs_render(r.handle, sc.cameras, p, out, ids)
        b.vs_render(r.handle, sc.cameras, p, out)          # second call: the read-and-clear key image is reused
        torch.cuda.synchronize()
        st = r.stats()
        print("%s | vs_render %s: ok, %d launches" % (tag, name, st["kernel_launches"]), flush=True)
    p = b.make_params(W, H, sc.near_plane, sc.t_min, sc.background)
    lr = torch.empty((B, k, H, W, 4), dtype=torch.float32, device="cuda")
    luv = torch.empty((B, k, H, W, 2), dtype=torch.float32, device="cuda")
    ln = torch.empty((B, k, H, W, 3), dtype=torch.float32, device="cuda")
    for flags in (0, b.VS_FLAG_TILED_PATH):
        pa = b.make_params(W, H, sc.near_plane, sc.t_min, sc.background, flags)
        b.vs_render_aov(r.handle, sc.cameras, pa, out, None, lr, luv, ln)
        b.vs_render_aov(r.handle, sc.cameras, pa, out, ids, lr, luv, ln)
    torch.cuda.synchronize()
    print("%s | vs_render_aov: ok" % tag, flush=True)
    host = np.empty((B, H, W, 4), np.float32)
    hids = np.empty((B, k, H, W), np.uint32)
    b.vs_render_host(r.handle, sc.cameras, b.make_params(W, H, sc.near_plane, sc.t_min, sc.background, 0, 1), host, hids)
    print("%s | vs_render_host: ok" % tag, flush=True)
    if not banded:
        g = torch.ones((B, H, W, 4), dtype=torch.float32, device="cuda")
        grads = [torch.zeros(ly.texture.shape, dtype=torch.float32, device="cuda") for ly in sc.layers]
        b.vs_render_backward(r.handle, sc.cameras, p, g, grads)
        torch.cuda.synchronize()
        print("%s | vs_render_backward: ok" % tag, flush=True)
    r.close()


def main():
    b.load_library()
    run(synth.make_config(1, width=96, height=80, num_cameras=2), "C1-reduced")
    run(synth.make_config(2, mesh_n=16, width=112, height=96, tex_size=64, num_cameras=2), "C2-reduced (fp16 SH2)")
    run(synth.make_config(4, mesh_n=12, width=100, height=52, tex_size=64, num_cameras=2, k=9), "C4-reduced (fp16 SH3)")
    run(synth.make_config(4, mesh_n=12, width=100, height=52, tex_size=64, num_cameras=2, k=4, banded=True), "C4-reduced banded")
    print("sanitizer workload finished")


if __name__ == "__main__":
    main()

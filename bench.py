#!/usr/bin/env python
"""bench.py -- headline measurement of the k-shell render path (BASELINE.json metric: megapixels/s and
fps rendering k layers at 1080p; achieved HBM GB/s vs peak).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one vs_render call = one pass of the whole hot path (S1-S7) over one batch of cameras of
the chosen configuration (default C4, the headline roofline config: k=9, ~300k triangles per layer,
1920x1080, 64 views per call, SH-3 fp16 2048^2 textures).  Prints ONE JSON line on rank 0.
`--impl reference` times the CPU oracle (as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2409_02482_b200 import dist as vsdist  # noqa: E402
from paper_2409_02482_b200 import synth  # noqa: E402

METRIC = "megapixels_per_sec_rendering_k_layers"
UNIT = "MP/s"
# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel from the committed `ncu --set full` captures:
# profiles/ncu_traffic.json holds, per configuration, the bytes per view of the captured launch together with the commit
# and the SHA-256 of the kernel sources the capture was taken from.  `roofline.traffic` is reported only while those
# sources are unchanged (else null: a capture of other code is not evidence about this run).
TRAFFIC_FILE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "profiles", "ncu_traffic.json")
TRAFFIC_SOURCES = ("vs_kernels_shade.cu", "vs_kernels_order.cu", "vs_common.cuh")


def kernel_source_hashes():
    import hashlib
    d = os.path.join(os.path.dirname(os.path.abspath(__file__)), "paper_2409_02482_b200", "csrc")
    return {f: hashlib.sha256(open(os.path.join(d, f), "rb").read()).hexdigest() for f in TRAFFIC_SOURCES}


def ncu_traffic_bytes_per_view(config_key, views_per_launch=None):
    """(bytes per view, provenance) of the committed capture of this configuration, or (None, why not).  In surface order the
    views of a launch share texels through L2, so a capture only speaks for launches of the same number of views."""
    try:
        table = json.load(open(TRAFFIC_FILE))
    except Exception:
        return None, "no profiles/ncu_traffic.json"
    ent = table.get(str(config_key))
    if not ent:
        return None, "no committed ncu capture of this configuration"
    if ent.get("source_sha256") != kernel_source_hashes():
        return None, "kernel sources changed since the capture of commit %s" % ent.get("commit")
    if views_per_launch is not None and ent.get("views_per_launch") not in (None, int(round(views_per_launch))):
        return None, "the committed capture is of a %s-view launch, this run launched %g views at a time" % (
            ent.get("views_per_launch"), views_per_launch)
    return float(ent["dram_bytes_per_view"]), "ncu --set full capture of commit %s (%s)" % (ent.get("commit"), ent.get("summary"))


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def geometry_bytes_per_view(sc):
    return sum(ly.positions.shape[0] * 20 + ly.indices.shape[0] * 12 for ly in sc.layers)


class ClockSampler:
    FIELDS = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.path = tempfile.mktemp(suffix=".csv")
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self, t0=None, t1=None):
        """Median SM clock, maximum clock, power and throttle reasons of the samples taken between the wall-clock times
        t0 and t1 (the timed region); the sampler is started before the warm-up so that it is already running then."""
        import datetime
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        rows = []
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    ts = datetime.datetime.strptime(f[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                except ValueError:
                    ts = None
                try:
                    rows.append((ts, float(f[1]), float(f[2]), float(f[3]), f[5:9]))
                except ValueError:
                    continue
            os.unlink(self.path)
        except Exception:
            pass
        inside = [r for r in rows if t0 is not None and r[0] is not None and t0 - 0.02 <= r[0] <= t1 + 0.02]
        window = "timed region" if inside else "warm-up + timed region"
        sm, mx, reasons, power = [], [], set(), []
        for _, a_sm, a_mx, a_pw, flags in (inside or rows):
            sm.append(a_sm); mx.append(a_mx); power.append(a_pw)
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), flags):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if sm:
            out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                   "samples": len(sm), "window": window, "power_w_max": max(power) if power else None}
        return out


def build_scene(cfg, rank, world, args):
    kw = {}
    if args.views:
        kw["num_cameras"] = args.views
    if getattr(args, "banded", False):
        kw["banded"] = True
    if getattr(args, "tex_size", 0):
        kw["tex_size"] = args.tex_size
    if getattr(args, "camera_subset", None):
        kw["camera_subset"] = args.camera_subset
    if getattr(args, "strong", False):
        # strong scaling: ONE batch (rank 0's cameras), split evenly over the ranks; every rank renders its slice
        sc = synth.make_config(cfg, **kw)
        mine = vsdist.shard_views(len(sc.cameras), rank, world)
        sc.name += " [strong scaling: views %d..%d of the %d-view batch on rank %d]" % (mine.start, mine.stop - 1, len(sc.cameras), rank)
        sc.cameras = np.ascontiguousarray(sc.cameras[mine.start:mine.stop])
        return sc
    return synth.make_config(cfg, camera_rotate=vsdist.rank_camera_rotation(rank, world), **kw)


def time_oracle(sc, views, threads=0):
    import oracle
    t0 = time.perf_counter()
    for v in views:
        oracle.render_view(sc.layers, sc.sh_degree, sc.cameras[v], sc.width, sc.height, near_plane=sc.near_plane,
                           t_min=sc.t_min, background=sc.background, num_threads=threads, v_range=sc.v_range)
    return time.perf_counter() - t0


def run_reference(args):
    rank, local, world = vsdist.env_rank()
    if rank != 0:
        return 0
    import oracle
    sc = build_scene(args.config, 0, 1, args)
    sample_views = 1
    px = sc.width * sc.height * sample_views
    for _ in range(args.warmup):
        time_oracle(sc, [0])
    t = 0.0
    for s in range(args.steps):
        t += time_oracle(sc, [(s * sample_views + i) % len(sc.cameras) for i in range(sample_views)])
    value = px * args.steps / t / 1e6
    cores = oracle.max_threads()
    sample = "%d view(s) per step of %s (bounded sample of the %d-view batch)" % (sample_views, sc.name, len(sc.cameras))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "fps": sample_views * args.steps / t,
            "config": {"workload": sc.name, "k": sc.k, "width": sc.width, "height": sc.height,
                       "views_per_step": sample_views, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_ours(args):
    import torch
    from paper_2409_02482_b200 import binding
    rank, local, world = vsdist.env_rank()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    vsdist.init_process_group("nccl")
    if args.lib:            # a variant build of the same sources (python -m paper_2409_02482_b200.build --lib PATH -D...)
        binding.LIB_PATH = os.path.abspath(args.lib)
        binding.load_library(build_if_missing=False)
    else:
        binding.load_library()

    sc = build_scene(args.config, rank, world, args)
    B, W, H = len(sc.cameras), sc.width, sc.height
    renderer = binding.Renderer(sc, dev)
    path_flag = ((binding.VS_FLAG_TILED_PATH if args.tiled else 0) | (binding.VS_FLAG_ATTENUATION if args.attenuation else 0) |
                 (binding.VS_FLAG_OVERLAP if args.overlap else 0) | (binding.VS_FLAG_SCREEN_ORDER if args.screen_order else 0) |
                 (binding.VS_FLAG_PLAIN_BACKWARD if args.plain_backward else 0))
    flags = binding.VS_FLAG_KERNEL_TIMING | path_flag
    params = binding.make_params(W, H, sc.near_plane, sc.t_min, sc.background, flags, args.chunk)
    out = torch.empty((B, H, W, 4), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream()

    # untimed: count the algorithmic texture bytes (unique texels per view) of this batch
    cparams = binding.make_params(W, H, sc.near_plane, sc.t_min, sc.background, binding.VS_FLAG_COUNT_TEXELS | path_flag, args.chunk)
    binding.vs_render(renderer.handle, sc.cameras, cparams, out)
    cstats = renderer.stats()
    banded = sc.layers[0].band_textures is not None
    texel_bytes = 0 if banded else 16 * ((sc.n_coef * 4 * sc.layers[0].texture.dtype.itemsize + 15) // 16)
    b_tex = cstats["unique_texels"] * texel_bytes      # banded scenes: not counted (ALU-bound path, see below)
    b_geom = geometry_bytes_per_view(sc) * B
    b_fb = W * H * 16 * B
    alg_bytes_step = b_tex + b_geom + b_fb

    if args.backward:
        # step = one vs_render_backward call (S1-S4 + k_shade<BWD>, or k_backward with --plain-backward) over the batch; the fp32 gradient textures are
        # accumulated into across steps (zeroed once, outside the timed region)
        gen = torch.Generator(device=dev).manual_seed(1234)
        gout = torch.randn((B, H, W, 4), dtype=torch.float32, device=dev, generator=gen)
        grads = [torch.zeros(ly.texture.shape, dtype=torch.float32, device=dev) for ly in sc.layers]
        b_grad = cstats["unique_texels"] * sc.n_coef * 16 * 2          # fp32 gradient texel read + written once per view
        b_fb = W * H * 16 * B                                           # the upstream gradient is read instead of an image written
        alg_bytes_step = b_tex + b_grad + b_geom + b_fb

        def run_step():
            binding.vs_render_backward(renderer.handle, sc.cameras, params, gout, grads)
    else:
        b_grad = 0

        def run_step():
            binding.vs_render(renderer.handle, sc.cameras, params, out)

    sampler = ClockSampler(local) if rank == 0 else None   # started before the warm-up: nvidia-smi takes a moment to come up
    for _ in range(max(args.warmup, 0)):
        run_step()
    torch.cuda.synchronize()
    renderer.stats()        # resets the accumulated kernel timings: what the next query returns belongs to the timed steps

    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    vsdist.barrier()
    torch.cuda.synchronize()
    wall0 = time.time()
    ev0.record(stream)
    for _ in range(args.steps):
        run_step()          # asynchronous: no host synchronisation between the steps
    ev1.record(stream)
    torch.cuda.synchronize()
    vsdist.barrier()
    st = renderer.stats()   # per-kernel CUDA-event times (recorded on the render stream) and launch counts of the K steps
    shade_ms, raster_ms, bin_ms, xf_ms = st["ms_shade"], st["ms_raster"], st["ms_binning"], st["ms_transform"]
    shade_launches, launches = st["shade_launches"], st["kernel_launches"]
    secs = ev0.elapsed_time(ev1) / 1e3
    clocks = sampler.stop(wall0, time.time()) if sampler else None
    secs_max = vsdist.max_over_ranks(secs, dev)
    pixels_all = vsdist.sum_over_ranks(float(B * W * H * args.steps), dev)
    value = pixels_all / secs_max / 1e6
    fps = vsdist.sum_over_ranks(float(B * args.steps), dev) / secs_max

    # end to end through the C-ABI with HOST buffers: camera upload + image download every step
    e2e_steps = max(1, min(args.steps, 5))
    host_out = torch.empty((B, H, W, 4), dtype=torch.float32).pin_memory()
    eparams = binding.make_params(W, H, sc.near_plane, sc.t_min, sc.background, path_flag, args.chunk)
    binding.vs_render_host(renderer.handle, sc.cameras, eparams, host_out)
    vsdist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        binding.vs_render_host(renderer.handle, sc.cameras, eparams, host_out)
    torch.cuda.synchronize()
    e2e_secs = vsdist.max_over_ranks(time.perf_counter() - t0, dev)
    e2e_value = vsdist.sum_over_ranks(float(B * W * H * e2e_steps), dev) / e2e_secs / 1e6

    if rank != 0:
        renderer.close()
        return 0

    peak, peak_src = load_peaks()
    # dominant kernel = k_shade: it moves the texture bytes and writes the framebuffer; its algorithmic
    # bytes are B_tex + B_fb of the views one launch processes (B_geom belongs to the geometry kernels
    # and is counted in `whole_step`, which divides ALL algorithmic bytes by the whole step's time).
    per_launch_ms = shade_ms / max(shade_launches, 1)
    bytes_per_launch = (b_tex + b_grad + b_fb) * args.steps / max(shade_launches, 1)
    achieved = bytes_per_launch / (per_launch_ms * 1e-3) / 1e9 if per_launch_ms > 0 else 0.0
    step_achieved = alg_bytes_step * world / (secs_max / args.steps) / 1e9
    views_per_launch = B * args.steps / max(shade_launches, 1)
    traffic_key = "%d%s%s" % (args.config, "-" + args.camera_subset if args.camera_subset else "", "-backward" if args.backward else "")
    plain = not (args.tiled or args.attenuation or args.overlap or args.screen_order or args.views or banded or args.lib or args.plain_backward or args.tex_size)
    traffic_per_view, traffic_src = ncu_traffic_bytes_per_view(traffic_key, views_per_launch) if plain else (None, "not the captured launch configuration")
    # the three candidate bounds of SURVEY.md §8(d), per view: HBM (algorithmic bytes), L1 gather (4 texels per fragment through
    # the 128 B/clk/SM data pipe), FP32 issue (algorithmic lane-ops: 4 x 4n bilinear + SH FMAs, 4 x 4n half->float conversions
    # for fp16 texels, ~40 for sigmoids and blend; 128 lanes per SM) -- the largest one binds
    sm_clock_hz = 1965.0e6
    frags_view = cstats["shaded_fragments"] / B
    t_hbm = alg_bytes_step / B / (peak * 1e9) * 1e3
    t_l1 = frags_view * 4 * texel_bytes / (148 * 128 * sm_clock_hz) * 1e3
    lane_ops = 16 * sc.n_coef + (16 * sc.n_coef if (not banded and sc.layers[0].texture.dtype == np.float16) or banded else 0) + 40
    t_fp32 = frags_view * lane_ops / (148 * 128 * sm_clock_hz) * 1e3
    cand = {"hbm": t_hbm, "l1_gather": t_l1, "fp32_issue": t_fp32}
    bounds = {"ms_per_view": cand, "binding": max(cand, key=cand.get), "measured_ms_per_view": 1e3 * secs_max / args.steps / B,
              "lane_ops_per_fragment": lane_ops, "note": "148 SMs x 128 B/clk resp. 128 lanes at 1965 MHz; HBM at the measured copy peak"}
    roofline = {"bound": "hbm", "kernel": ("k_backward" if args.plain_backward else "k_shade<BWD>") if args.backward else "k_shade", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic_per_view * views_per_launch if traffic_per_view else None,
                "traffic_source": traffic_src, "bounds": bounds,
                "peak_source": peak_src, "algorithmic_bytes_per_launch": bytes_per_launch,
                "launch_ms": per_launch_ms, "views_per_launch": B * args.steps / max(shade_launches, 1),
                "kernel_share_of_step": shade_ms / (secs * 1e3),
                "bytes_per_view": {"texels_unique": b_tex / B, "geometry": b_geom / B, "framebuffer": b_fb / B},
                "whole_step": {"achieved": step_achieved / world, "frac": step_achieved / world / peak,
                               "algorithmic_bytes_per_step": alg_bytes_step},
                "stage_ms_per_step": {"transform": xf_ms / args.steps, "binning": bin_ms / args.steps,
                                      "raster": raster_ms / args.steps, "shade": shade_ms / args.steps}}

    if roofline["traffic"]:
        # < 1 in surface order: the views of a launch share texels through L2, while the algorithmic bytes
        # charge every view its unique texels once.  `frac` then measures speed against a view-by-view renderer running at the
        # HBM peak, not DRAM utilisation
        roofline["traffic_over_algorithmic"] = roofline["traffic"] / bytes_per_launch
        if roofline["traffic_over_algorithmic"] < 1.0:
            roofline["note"] = ("DRAM traffic is below the per-view algorithmic bytes: the views of a launch share texels through L2 "
                                "(surface-ordered shading); frac is against a view-by-view renderer at the HBM peak, the kernel "
                                "itself is bound by SM-side work (L1 data pipe), see DESIGN.md 7-8")
    if banded:
        # The banded 8-bit path is bound by the plain FP32/ALU pipes: algorithmic lane-ops per shaded
        # fragment at degree d = 4 texels x 4(d+1)^2 byte->float conversions + as many bilinear FMAs + 4(d+1)^2 SH FMAs
        # (576 at degree 3); peak = 148 SMs x 128 FP32 lanes x the maximum SM clock.
        n4 = 4 * sc.n_coef
        ops_per_frag = 4 * n4 + 4 * n4 + n4
        frags_per_launch = cstats["shaded_fragments"] * args.steps / max(shade_launches, 1)
        alu_achieved = frags_per_launch * ops_per_frag / (per_launch_ms * 1e-3) / 1e12 if per_launch_ms > 0 else 0.0
        alu_peak = 148 * 128 * ((clocks or {}).get("sm_max_mhz") or 1965.0) * 1e6 / 1e12
        roofline = {"bound": "alu", "kernel": "k_shade_banded", "achieved": alu_achieved, "peak": alu_peak, "unit": "Tlane-op/s",
                    "frac": alu_achieved / alu_peak, "traffic": None,
                    "peak_source": "derived: 148 SMs x 128 FP32 lanes x max SM clock (B200_PROFILING.md unit counts)",
                    "lane_ops_per_fragment": ops_per_frag, "launch_ms": per_launch_ms,
                    "views_per_launch": B * args.steps / max(shade_launches, 1),
                    "kernel_share_of_step": shade_ms / (secs * 1e3),
                    "stage_ms_per_step": roofline["stage_ms_per_step"]}

    cpu_baseline = None
    if world == 1 and not args.no_cpu:
        import oracle
        nviews, t = 0, 0.0
        while nviews < B and (t < args.cpu_seconds or nviews < 1):   # bounded sample: ~10 s of oracle work
            t += time_oracle(sc, [nviews])
            nviews += 1
        cpu_baseline = {"value": nviews * W * H / t / 1e6, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
                        "sample": "first %d of %d views of %s, %.1f s" % (nviews, B, sc.name, t)}
        # "reported for 1 thread and for all host cores" -- one view on one thread, if it fits the budget
        est = t / nviews * oracle.max_threads()
        if est <= args.cpu_1thread_seconds:
            t1 = time_oracle(sc, [0], threads=1)
            cpu_baseline["one_thread"] = {"value": W * H / t1 / 1e6, "unit": UNIT, "cores": 1, "sample": "view 0, %.1f s" % t1}
        else:
            cpu_baseline["one_thread"] = {"value": None, "skipped": "estimated %.0f s for one view > --cpu-1thread-seconds %.0f" % (est, args.cpu_1thread_seconds)}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * secs_max / args.steps, "higher_is_better": True, "scaling": "strong" if args.strong else "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic", "fps": fps,
            "config": {"workload": sc.name, "k": sc.k, "triangles_per_layer": int(sc.layers[0].indices.shape[0]),
                       "width": W, "height": H, "views_per_step": B, "sh_degree": sc.sh_degree,
                       "texture": ("uint8 banded " + " ".join("%dx%d" % (t.shape[1], t.shape[0]) for t in sc.layers[0].band_textures)
                                   + " range [%g, %g]" % sc.v_range) if banded else
                                  "%s %dx%d" % (sc.layers[0].texture.dtype, sc.layers[0].texture.shape[1], sc.layers[0].texture.shape[0]),
                       "raster_path": "tiled (binning + per-tile shared-memory keys)" if args.tiled
                       else "direct (triangle-parallel, 64-bit max keys in HBM/L2)",
                       "attenuation": bool(args.attenuation), "overlap": bool(args.overlap), "shading_order": "screen" if (args.screen_order or args.tiled or banded) else "surface", "library": args.lib or "libvs_b200.so",
                       "timed_loop": "K asynchronous vs_render calls, one stream synchronisation at the end; kernel times from CUDA events on the render stream",
                       "pass": "backward to texels (vs_render_backward)" if args.backward else "forward (vs_render)",
                       "parallelism": "views sharded, scene replicated (dp%d)" % world,
                       "l2": "no flush: %.2f GiB of textures streamed per step >> 126 MB L2" % (
                           sum(sum(t.nbytes for t in ly.band_textures) if banded else ly.texture.nbytes for ly in sc.layers) / 2 ** 30),
                       "shaded_fragments_per_view": cstats["shaded_fragments"] / B,
                       "tile_refs_per_view": cstats["tile_refs"] / B},
            "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu_baseline,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(sc.cameras.nbytes),
                    "d2h_bytes_per_step": int(host_out.numel() * 4), "steps": e2e_steps,
                    "pass": "forward (vs_render_host)"},
            "gpu_launches": int(launches)}
    print(json.dumps(line))
    renderer.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--views", type=int, default=0, help="override the number of views per step")
    ap.add_argument("--chunk", type=int, default=0, help="views per internal pass (0 = automatic)")
    ap.add_argument("--cpu-seconds", type=float, default=10.0, help="oracle work of the cpu_baseline sample (whole views)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--backward", action="store_true", help="time vs_render_backward (gradients to the texels, PAPER.md:L441-443) instead of vs_render (not the headline workload)")
    ap.add_argument("--banded", action="store_true", help="the paper's 8-bit mixed-resolution textures on the same geometry (PAPER.md:L445-459; not the headline workload)")
    ap.add_argument("--attenuation", action="store_true", help="render with VS_FLAG_ATTENUATION (PAPER.md:L279-286; not the headline workload)")
    ap.add_argument("--tiled", action="store_true", help="time the per-tile raster path (VS_FLAG_TILED_PATH) instead of the default direct one")
    ap.add_argument("--tex-size", type=int, default=0, help="override the texture side (e.g. 512 on C4: magnified texels, the fitting regime of PAPER.md:L441-443; not the headline workload)")
    ap.add_argument("--plain-backward", action="store_true", help="with --backward: VS_FLAG_PLAIN_BACKWARD, the plain per-lane k_backward instead of k_shade<BWD> (A/B)")
    ap.add_argument("--screen-order", action="store_true", help="VS_FLAG_SCREEN_ORDER: shade view by view instead of in surface order (A/B, DESIGN.md §7)")
    ap.add_argument("--overlap", action="store_true", help="VS_FLAG_OVERLAP: S1-S4 of the next chunk beside S5-S7 of the current one (experiment, DESIGN.md §7)")
    ap.add_argument("--camera-subset", choices=["far", "close"], default=None,
                    help="every other camera of the set: on C5 the r=3 orbit cameras resp. the r=1.6 close-ups (SURVEY.md §8(d))")
    ap.add_argument("--strong", action="store_true", help="multi-GPU: split ONE camera batch evenly over the ranks (strong scaling) instead of one batch per rank")
    ap.add_argument("--lib", default=None, help="load this build of the library (an experiment variant made by `python -m paper_2409_02482_b200.build --lib PATH -D...`)")
    ap.add_argument("--record-traffic", nargs=5, metavar=("KEY", "DRAM_BYTES_PER_VIEW", "VIEWS_PER_LAUNCH", "COMMIT", "SUMMARY"), default=None,
                    help="no benchmark: store the dram__bytes_read+write per view of an `ncu --set full` capture of configuration KEY "
                         "(e.g. 4, 5-close) in profiles/ncu_traffic.json together with the hashes of the kernel sources as they are now")
    ap.add_argument("--cpu-1thread-seconds", type=float, default=30.0, help="budget of the 1-thread oracle sample (one whole view); skipped if a view would take longer")
    args = ap.parse_args()
    if args.record_traffic:
        key, nbytes, vpl, commit, summary = args.record_traffic
        try:
            table = json.load(open(TRAFFIC_FILE))
        except Exception:
            table = {}
        table[key] = {"kernel": "k_shade<BWD>" if key.endswith("-backward") else "k_shade", "dram_bytes_per_view": float(nbytes), "views_per_launch": int(vpl), "commit": commit,
                      "summary": summary, "source_sha256": kernel_source_hashes()}
        json.dump(table, open(TRAFFIC_FILE, "w"), indent=1, sort_keys=True)
        print("recorded", key, "in", TRAFFIC_FILE)
        return 0
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())

"""Multi-process host logic of the sharded path: views shard across ranks, the scene is
replicated, there is NO data-path collective -- only the barrier and the max/sum reductions of the timing.
World size 2 over `gloo` on CPU; the ranks' work is the oracle on tiny views (test infrastructure), the
product renderer needs a GPU and is not called here."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2409_02482_b200 import dist as vsdist  # noqa: E402


def test_shard_views_partitions_the_batch():
    for n in (0, 1, 2, 7, 64, 65):
        for world in (1, 2, 3, 8):
            shards = [list(vsdist.shard_views(n, r, world)) for r in range(world)]
            assert sorted(v for s in shards for v in s) == list(range(n))          # every view exactly once
            assert max(len(s) for s in shards) - min(len(s) for s in shards) <= 1  # balanced
            assert all(s == sorted(s) for s in shards)


def test_rank_camera_rotation_distinct_views():
    assert vsdist.rank_camera_rotation(0, 1) == 0.0
    rots = [vsdist.rank_camera_rotation(r, 8) for r in range(8)]
    assert len(set(rots)) == 8 and rots[0] == 0.0
    from paper_2409_02482_b200 import synth
    small = dict(mesh_n=4, tex_size=16, width=32, height=32, num_cameras=4)   # reduced C2: Fibonacci-lattice cameras
    a = synth.make_config(2, camera_rotate=rots[0], **small).cameras
    b = synth.make_config(2, camera_rotate=rots[1], **small).cameras
    assert a.shape == b.shape and not np.allclose(a, b)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import torch.distributed as dist
    import oracle
    from paper_2409_02482_b200 import synth
    r, w = vsdist.init_process_group("gloo")
    assert (r, w) == (rank, world)
    sc = synth.make_config(1)                       # 4 views of 128x128, k = 3
    mine = list(vsdist.shard_views(len(sc.cameras), rank, world))
    checksum = 0.0
    for v in mine:                                  # each rank renders only its own views
        res = oracle.render_view(sc.layers, sc.sh_degree, sc.cameras[v], sc.width, sc.height,
                                 near_plane=sc.near_plane, t_min=sc.t_min, background=sc.background, num_threads=1)
        checksum += float(np.asarray(res["rgba"], dtype=np.float64).sum())
    # bench.py --strong builds its per-rank scene with the same split: this rank's slice of ONE batch
    import types
    import bench
    mine_sc = bench.build_scene(1, rank, world, types.SimpleNamespace(views=0, banded=False, camera_subset=None, strong=True))
    assert np.array_equal(mine_sc.cameras, sc.cameras[mine]) and "strong scaling" in mine_sc.name
    weak_sc = bench.build_scene(1, rank, world, types.SimpleNamespace(views=0, banded=False, camera_subset=None, strong=False))
    assert len(weak_sc.cameras) == len(sc.cameras)   # weak scaling: a whole batch per rank
    vsdist.barrier()
    secs = 1.0 + rank                               # synthetic per-rank device times: the job time is the max
    out = {"rank": rank, "views": mine, "checksum": checksum,
           "max": vsdist.max_over_ranks(secs), "sum": vsdist.sum_over_ranks(float(len(mine))),
           "thr": vsdist.whole_job_throughput(float(len(mine)), secs),
           "total_checksum": vsdist.sum_over_ranks(checksum)}
    vsdist.barrier()
    dist.destroy_process_group()
    q.put(out)


@pytest.mark.timeout(300)
def test_world_size_2_gloo_sharded_render():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=240) for _ in procs), key=lambda d: d["rank"])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0]["views"] == [0, 1] and res[1]["views"] == [2, 3]
    for d in res:
        assert d["max"] == 2.0                      # max over ranks of (1.0, 2.0)
        assert d["sum"] == 4.0                      # all four views rendered exactly once
        assert d["thr"] == 2.0                      # 4 views / 2.0 s
    # single-process render of the whole batch gives the same images as the two shards together
    import oracle
    from paper_2409_02482_b200 import synth
    sc = synth.make_config(1)
    total = 0.0
    for v in range(len(sc.cameras)):
        one = oracle.render_view(sc.layers, sc.sh_degree, sc.cameras[v], sc.width, sc.height,
                                 near_plane=sc.near_plane, t_min=sc.t_min, background=sc.background, num_threads=1)
        total += float(np.asarray(one["rgba"], dtype=np.float64).sum())
    assert abs(res[0]["total_checksum"] - total) <= 1e-9 * max(1.0, abs(total))
    assert abs(res[0]["checksum"] + res[1]["checksum"] - total) <= 1e-9 * max(1.0, abs(total))

"""The N > 1 path of bench.py on CPU (gloo, world_size 2): replicas only -- every rank renders its own views
of a replicated scene, there is no data-path collective; the only exchange is the max-over-ranks of the step
time, and the job value counts the views of all ranks."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank: int, world: int, port: int, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        views = [bench.view_of_step(i, rank, 8) for i in range(16)]
        ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist)           # rank 1 is the slow one
        gathered = [None] * world
        dist.all_gather_object(gathered, views)
        if rank == 0:
            out.put((ms, gathered))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
    import bench
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    ms, views = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert ms == 15.0                                                  # the max over ranks, on every rank
    # in every step the two ranks render different views, and each rank cycles through all 8
    assert all(a != b for a, b in zip(views[0], views[1]))
    assert set(views[0]) == set(views[1]) == set(range(8))
    # whole-job value: both ranks' pixels over the slowest rank's time
    assert bench.job_value(1297 * 840, 2, ms) == 2 * 1297 * 840 / 1e6 / (ms / 1e3)


def test_single_rank_is_identity():
    import bench
    assert bench.max_over_ranks(3.5, None) == 3.5
    assert [bench.view_of_step(i, 0, 8) for i in range(9)] == [0, 1, 2, 3, 4, 5, 6, 7, 0]


def test_bench_gpus_2_spawns_two_ranks():
    """`python bench.py --gpus 2` with no launcher around it starts two ranks by itself (torchrun, 127.0.0.1) and
    rank 0 prints one line for the whole job; --dry-run keeps it on the CPU (gloo, a stand-in step)."""
    import json
    import subprocess
    env = dict(os.environ)
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT"):
        env.pop(k, None)
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "16", "--dry-run"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                   # one line, from rank 0
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["scaling"] == "weak"
    assert out["ms_per_step"] == 1.5                         # max over ranks (rank 1 is the slow one)
    assert out["value"] == 2 * 1297 * 840 / 1e6 / 1.5e-3     # both ranks' pixels over the slowest rank's time
    v0, v1 = out["views_per_rank"]
    assert all(a != b for a, b in zip(v0, v1)) and set(v0) == set(v1) == set(range(8))

"""Host-side logic of bench.py that needs no GPU: the N > 1 ("replicas only") view
sharding and max-over-ranks aggregation, run as a world_size-2 gloo group on CPU, and the reference arm's
JSON contract on a tiny scene."""
import json
import os
import subprocess
import sys
from pathlib import Path

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))
import bench  # noqa: E402


def _worker(rank, world, port, steps, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    views = [bench.views_for_rank(i, rank, world, 32) for i in range(steps)]
    secs = torch.tensor([0.010 * (rank + 1)], dtype=torch.float64)       # rank 1 is the slow one
    dist.all_reduce(secs, op=dist.ReduceOp.MAX)
    gathered = [None] * world
    dist.all_gather_object(gathered, views)
    if rank == 0:
        q.put((gathered, bench.aggregate_fps(steps, world, float(secs.item()))))
    dist.barrier()
    dist.destroy_process_group()


def test_view_sharding_and_max_over_ranks_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    steps, world, port = 16, 2, 29533
    procs = [ctx.Process(target=_worker, args=(r, world, port, steps, q)) for r in range(world)]
    for p in procs:
        p.start()
    gathered, fps = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    all_views = [v for per_rank in gathered for v in per_rank]
    assert sorted(all_views) == list(range(32))                           # disjoint, and together they cover the orbit
    assert gathered[0][:3] == [0, 2, 4] and gathered[1][:3] == [1, 3, 5]
    assert abs(fps - steps * world / 0.020) < 1e-6                        # whole-job frames / slowest rank's time


def test_single_rank_views_walk_the_orbit():
    assert [bench.views_for_rank(i, 0, 1, 32) for i in (0, 1, 31, 32, 33)] == [0, 1, 31, 0, 1]


def test_reference_arm_prints_the_contract_line():
    out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--steps", "2", "--warmup", "1",
                          "--n", "20000"], capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "frames/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["value"] == line["value"]
    assert line["higher_is_better"] is True and line["steps"] == 2

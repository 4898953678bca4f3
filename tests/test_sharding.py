"""Multi-GPU story: independent KEM instances are sharded over
ranks with no data-path collective; the only communication is the timing/summary
reduction bench.py does.  Covered here with world_size-2 gloo on CPU."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_01211_b200 import workloads as W


def test_shard_instances_partitions_exactly():
    for batch in (1, 2, 31, 32, 33, 64):
        for ws in (1, 2, 3, 4, 8):
            parts = [W.shard_instances(batch, r, ws) for r in range(ws)]
            flat = [i for p in parts for i in p]
            assert flat == list(range(batch))
            sizes = [len(p) for p in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        W.shard_instances(4, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    mine = W.shard_instances(32, rank, world)
    # each rank "times" its own shard; bench's reduction = max time, sum of units
    ms, units = bench.reduce_over_ranks(10.0 + rank, len(mine))
    out[rank] = (ms, units, list(mine)[0], list(mine)[-1])
    dist.destroy_process_group()


def test_world_size_2_gloo_reduction_and_disjoint_shards():
    world = 2
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == 11.0                  # max over ranks
    assert res[0][1] == res[1][1] == 32                    # all instances counted once
    assert (res[0][2], res[0][3]) == (0, 15) and (res[1][2], res[1][3]) == (16, 31)


def test_bench_spawns_its_own_ranks_for_gpus_2_dry_run():
    """`python bench.py --gpus 2` started as a PLAIN process (no torchrun, no WORLD_SIZE) must produce the two ranks
    itself.  --dry-run runs that launch path and the rank plumbing (instance-id assignment, barrier, max / sum
    reduction, one JSON line from rank 0) on CPU/gloo; it prints no measurement."""
    import json
    import subprocess
    import sys
    from pathlib import Path
    root = Path(__file__).resolve().parent.parent
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, str(root / "bench.py"), "--gpus", "2", "--dry-run", "--steps", "3", "--warmup", "1"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout                           # rank 0 alone prints
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["dry_run"] is True and line["value"] is None
    assert line["ms_per_step"] == 11.0                         # max over ranks of (10 + rank)
    assert line["units_per_step"] == 64                        # 32 instances per rank, summed
    ids = line["instance_ids_first_3_steps"]
    spans = sorted(tuple(x) for rank_ids in ids for x in rank_ids)
    assert spans == [(32 * i, 32 * i + 31) for i in range(6)]  # disjoint over ranks and steps, nothing skipped

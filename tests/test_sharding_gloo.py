"""N > 1 path on CPU (world_size 2, gloo): the partition of a batch of patch groups over ranks, the independence
of the shards (each rank steps its shard with the ORACLE — the CUDA path needs a GPU — and the concatenation must
equal the unsharded result bit for bit) and the max-over-ranks timing reduction bench.py reports."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import mhm_oracle as O
from paper_1007_3818_b200 import sharding
from harness import workloads as wl


def test_shard_range_partitions_every_batch():
    for n in (0, 1, 2, 7, 8, 148, 32768, 32769):
        for world in (1, 2, 3, 4, 8):
            r = [sharding.shard_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.shard_range(4, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, tmp):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        g = wl.random_groups(5, seed=321, N=8, ghost=2)
        a, b = sharding.shard_range(g.shape[0], rank, world)
        r = O.step_groups(g[a:b], 8, 2, 2e-3, 1.0 / 8, wl.GAMMA, 1, n_threads=1)
        np.save(os.path.join(tmp, "out%d.npy" % rank), r.U_out)
        np.save(os.path.join(tmp, "bf%d.npy" % rank), r.bflux)
        # timing reduction: rank r "took" (r + 1) seconds; every rank must see the max
        t = sharding.max_over_ranks(float(rank + 1))
        assert t == float(world)
        # whole-job throughput uses the slowest rank's time
        assert sharding.aggregate_throughput(100, world, t) == 100.0
        counts = torch.tensor([b - a], dtype=torch.int64)
        dist.all_reduce(counts)
        assert int(counts.item()) == g.shape[0]
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_shards_concatenate_to_the_unsharded_result(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    g = wl.random_groups(5, seed=321, N=8, ghost=2)
    full = O.step_groups(g, 8, 2, 2e-3, 1.0 / 8, wl.GAMMA, 1, n_threads=1)
    out = np.concatenate([np.load(tmp_path / ("out%d.npy" % r)) for r in range(world)])
    bf = np.concatenate([np.load(tmp_path / ("bf%d.npy" % r)) for r in range(world)])
    assert np.array_equal(out, full.U_out) and np.array_equal(bf, full.bflux)


@pytest.mark.parametrize("scaling", ["weak", "strong"])
def test_bench_launcher_spawns_its_ranks_and_shards_one_field(scaling):
    """`python bench.py --gpus 2` must itself start two ranks (torch.distributed.run), share ONE generated field and
    partition it with sharding.shard_range; --no-cuda runs that path on gloo up to, not including, the first CUDA call."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_PORT")}
    res = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--no-cuda", "--box", "32",
                          "--scaling", scaling], capture_output=True, text=True, env=env, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    line = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(line) == 1                                       # rank 0 alone prints
    d = json.loads(line[0])
    one = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--no-cuda", "--box", "32"],
                         capture_output=True, text=True, env=env, timeout=300)
    d1 = json.loads([l for l in one.stdout.splitlines() if l.startswith("{")][0])
    assert d["n_gpus"] == 2 and d1["n_gpus"] == 1 and d["max_over_ranks"] == 2.0
    if scaling == "strong":
        assert d["groups_total"] == d1["groups_total"] == 8 and d["groups_rank0"] == 4
    else:
        assert d["groups_total"] == 16 and d["groups_rank0"] == 8
        assert d["checksum_rank0"] == d1["checksum_rank0"]      # every rank holds the same, once-generated field

"""Multi-GPU host logic on CPU: world_size-2 gloo processes (shard by baseline, no data-path collective)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2412_14775_b200 import sharding


@pytest.mark.parametrize("n,world", [(1176, 1), (1176, 2), (1176, 8), (6, 4), (3, 8), (2926, 7)])
def test_shard_baselines_is_a_contiguous_balanced_partition(n, world):
    parts = [sharding.shard_baselines(n, world, r) for r in range(world)]
    assert parts[0][0] == 0 and sum(c for _, c in parts) == n
    for (f0, c0), (f1, _) in zip(parts, parts[1:]):
        assert f1 == f0 + c0
    counts = [c for _, c in parts]
    assert max(counts) - min(counts) <= 1
    with pytest.raises(ValueError):
        sharding.shard_baselines(n, world, world)


def test_rank_work_weak_and_strong():
    """bench.py --gpus N --scaling weak|strong: what each rank processes."""
    for world in (1, 2, 4, 8):
        weak = [sharding.rank_work(1176, world, r, "weak") for r in range(world)]
        assert all(not x["sharded"] and x["b_count"] == 1176 for x in weak)
        assert [x["seed"] for x in weak] == [1234 + r for r in range(world)]           # one subband chunk per rank
        strong = [sharding.rank_work(1176, world, r, "strong") for r in range(world)]
        assert sum(x["b_count"] for x in strong) == 1176                                # ONE chunk, partitioned
        assert all(x["seed"] == 1234 for x in strong)
        assert all(x["sharded"] == (world > 1) for x in strong)
        assert [x["b_first"] for x in strong] == [sharding.shard_baselines(1176, world, r)[0] for r in range(world)]
    with pytest.raises(ValueError):
        sharding.rank_work(3, 8, 7, "strong")                                           # more ranks than baselines
    with pytest.raises(ValueError):
        sharding.rank_work(10, 2, 0, "diagonal")


def test_confusion_counts_by_hand():
    flags = torch.tensor([[[1, 0, 1], [0, 0, 1]], [[0, 0, 0], [1, 1, 1]]]).bool()      # [K=2, W=2, cells=3]
    truth = torch.tensor([[1, 0, 0], [0, 0, 1]]).bool()
    c = sharding.confusion_counts(flags, truth)
    assert c.tolist() == [[1, 4, 0, 2], [2, 4, 1, 2]]
    fa, md = sharding.rates(c)
    assert fa.tolist() == [0.25, 0.5] and md.tolist() == [0.0, 0.5]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_baselines, n_chan, n_win, K, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # the same seeded global masks on every rank; each rank keeps its baseline slice only
        g = torch.Generator().manual_seed(5)
        flags = torch.rand(K, n_win, n_baselines, n_chan, generator=g) < 0.1
        truth = torch.rand(n_win, n_baselines, n_chan, generator=g) < 0.05
        b0, bc = sharding.shard_baselines(n_baselines, world, rank)
        mine = sharding.confusion_counts(flags[:, :, b0:b0 + bc].flatten(2), truth[:, b0:b0 + bc].flatten(1))
        total = sharding.sum_over_ranks(mine.clone())
        full = sharding.confusion_counts(flags.flatten(2), truth.flatten(1))
        assert torch.equal(total, full), (total, full)
        # device-time bookkeeping: MAX over ranks
        t = sharding.max_over_ranks(1.0 + rank)
        assert t == float(world)
        # bench.py --scaling strong: the ranks' shards add up to the one chunk; weak: N chunks
        ws = sharding.rank_work(n_baselines, world, rank, "strong")
        assert (ws["b_first"], ws["b_count"]) == (b0, bc)
        assert sharding.sum_scalar_over_ranks(ws["b_count"] * n_chan) == n_baselines * n_chan
        ww = sharding.rank_work(n_baselines, world, rank, "weak")
        assert sharding.sum_scalar_over_ranks(ww["b_count"] * n_chan) == world * n_baselines * n_chan
        dist.barrier()
        np.save(os.path.join(out_dir, f"ok{rank}.npy"), np.array([b0, bc]))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_partition_and_reductions(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), 15, 4, 6, 3, str(tmp_path)), nprocs=world, join=True)
    parts = [np.load(tmp_path / f"ok{r}.npy") for r in range(world)]
    assert parts[0].tolist() == [0, 8] and parts[1].tolist() == [8, 7]


# ---- bench.py --gpus N starts its own ranks; the plumbing on CPU through --dry-launch -------------------
def _bench(*argv, env_extra=None):
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    env.update(env_extra or {})
    return subprocess.run([sys.executable, os.path.join(root, "bench.py"), *argv], capture_output=True, text=True, env=env,
                          cwd=root, timeout=600)


@pytest.mark.parametrize("scaling", ["weak", "strong"])
def test_bench_gpus_2_launches_two_ranks_by_itself(scaling):
    import json
    res = _bench("--gpus", "2", "--dry-launch", "--scaling", scaling)
    assert res.returncode == 0, res.stderr[-3000:]
    lines = [json.loads(l) for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, res.stdout                                                 # rank 0 alone prints
    rec = lines[0]
    assert rec["dry_launch"] and rec["n_gpus"] == 2 and rec["scaling"] == scaling and rec["max_ms"] == 2.0
    want = [sharding.rank_work(1176, 2, r, scaling) for r in range(2)]
    assert rec["work"] == want
    cells = 1176 * 64 * 7680                                                           # the lofar chunk (BASELINE.json configs[1])
    assert rec["total_samples"] == (2 * cells if scaling == "weak" else cells)


def test_bench_refuses_more_gpus_than_the_node_has():
    n = (torch.cuda.device_count() if torch.cuda.is_available() else 0) + 1
    res = _bench("--gpus", str(max(n, 2)), "--steps", "1")
    assert res.returncode != 0 and "GPUs on this node, found" in res.stderr


def test_bench_refuses_a_world_size_that_contradicts_gpus():
    res = _bench("--gpus", "2", "--dry-launch", env_extra={"WORLD_SIZE": "3", "RANK": "0"})
    assert res.returncode != 0 and "WORLD_SIZE = 3" in res.stderr

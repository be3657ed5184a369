"""N > 1 path on CPU: two processes under the gloo backend (world_size 2).  Cells are independent:
the step shards with no data-path collective, so what has to hold is that the block-cyclic shards partition the cells,
that integrating the shards separately and scattering them back equals integrating everything at once, and that the
only collectives (sum of the work counters, max of the elapsed time) reduce correctly.  The per-shard "step" here is
the CPU oracle -- test infrastructure standing in for the device kernel, which needs a GPU."""
import os
import socket

import numpy as np
import pytest

from paper_2504_04941_b200 import parallel as par
from paper_2504_04941_b200 import workloads as w


def test_shards_partition_the_cells():
    for n, world, block in [(0, 2, 4096), (1, 2, 4096), (10000, 2, 4096), (10000, 3, 128), (4096, 8, 4096), (12345, 4, 1000)]:
        seen = np.concatenate([par.shard_indices(n, r, world, block) for r in range(world)])
        assert seen.size == n and np.array_equal(np.sort(seen), np.arange(n))
        sizes = [par.shard_indices(n, r, world, block).size for r in range(world)]
        assert max(sizes) - min(sizes) <= block
    with pytest.raises(ValueError):
        par.shard_indices(10, 2, 2)


def test_reductions_are_identities_without_a_process_group():
    assert par.max_over_ranks(3.5) == 3.5 and par.sum_over_ranks(2.0) == 2.0
    assert par.allreduce_stats({"a": 1, "b": 2}) == {"a": 1, "b": 2}


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str) -> None:
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import build as obuild
        obuild.build_oracle()
        from oracle import oracle as O
        net, cells, opts = w.make_config(2, 700)
        idx = par.shard_indices(cells.n_cells, rank, world, block=64)
        mine = cells.take(idx)
        T, y, st, stats, _ = O.OracleNetwork(net, opts).step(mine, n_threads=1)
        total = par.allreduce_stats(stats)
        slowest = par.max_over_ranks(10.0 * (rank + 1))
        n_all = par.sum_over_ranks(float(mine.n_cells))
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), idx=idx, y=y, T=T, st=st, slowest=slowest, n_all=n_all,
                 **{f"s_{k}": v for k, v in total.items()}, **{f"l_{k}": v for k, v in stats.items()})
    finally:
        dist.destroy_process_group()


def test_two_ranks_sharded_equals_one_rank(tmp_path, oracle_mod):
    import torch.multiprocessing as mp
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    net, cells, opts = w.make_config(2, 700)
    T1, y1, st1, stats1, _ = oracle_mod.OracleNetwork(net, opts).step(cells, n_threads=1)
    y = np.empty_like(y1); st = np.empty_like(st1)
    outs = [np.load(tmp_path / f"rank{r}.npz") for r in range(world)]
    for o in outs:
        y[o["idx"]] = o["y"]; st[o["idx"]] = o["st"]
    np.testing.assert_array_equal(y, y1)                # cells are independent: sharding changes nothing, bit for bit
    np.testing.assert_array_equal(st, st1)
    for o in outs:
        assert float(o["slowest"]) == 20.0 and float(o["n_all"]) == 700.0
        for k, v in stats1.items():
            assert int(o[f"s_{k}"]) == v                # summed counters of the shards = counters of the whole
    assert sum(int(o["l_n_newton"]) for o in outs) == stats1["n_newton"]


def test_bench_starts_its_own_ranks_when_not_under_torchrun():
    """`python bench.py --gpus 2` (no torchrun environment) must take the launcher path -- one process per GPU -- and not
    silently run one rank: on this CPU-only box that path stops at the device count, with a message that names it."""
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE")}
    env["CUDA_VISIBLE_DEVICES"] = ""
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "1"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode != 0
    assert "--gpus 2 asked for, 0 CUDA device(s) visible" in (r.stderr + r.stdout)


def test_strong_scaling_shards_one_batch():
    """bench.py --scaling strong: every rank draws the SAME full-size batch and keeps its block-cyclic share."""
    net = w.make_network(2)
    whole = w.make_cells(2, net, 10000, seed=w.BASE_SEED + 1002)
    parts = [par.shard_cells(w.make_cells(2, net, 10000, seed=w.BASE_SEED + 1002), r, 4) for r in range(4)]
    assert sum(p.n_cells for p in parts) == whole.n_cells
    back = np.empty_like(whole.y)
    for r, p in enumerate(parts):
        back[par.shard_indices(whole.n_cells, r, 4)] = p.y
    np.testing.assert_array_equal(back, whole.y)

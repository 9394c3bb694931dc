"""N > 1 path on CPU: two gloo ranks each run their env shard (with the oracle standing in for the
device path, same env_id_base contract) and the gathered result must equal the unsharded run bit for bit.
DESIGN.md section 8: environments are independent, so sharding has no collective on the data path."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_22332_b200 import workloads as W
from paper_2606_22332_b200.sharding import shard_inputs, shard_range


def test_shard_range_partitions():
    for E in (1, 7, 16, 20480):
        for world in (1, 2, 3, 8):
            got = [shard_range(E, world, r) for r in range(world)]
            assert got[0][0] == 0 and sum(c for _, c in got) == E
            for (s0, c0), (s1, _) in zip(got, got[1:]):
                assert s1 == s0 + c0
            assert max(c for _, c in got) - min(c for _, c in got) <= 1
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)


def _run_shard(w, first, count, steps):
    from oracle import oracle as O
    ids = np.arange(first, first + count)
    o = O.Oracle(w.patches, w.T, w.L, w.K, ids, physics=w.physics, noise=w.noise, threads=1)
    o.set_geometry(w.types[ids], w.params[ids], w.bank, w.voxel)
    out = None
    for s in range(steps):
        out = o.step(shard_inputs(w.inputs(s), first, count), want=w.outputs, aux=False)
    o.close()
    return out


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.config(4, n_envs=6)
    first, count = shard_range(w.E, world, rank)
    out = _run_shard(w, first, count, steps=3)
    gathered = {}
    for k in ("ft_noisy", "dead", "depth", "marker"):
        t = torch.from_numpy(np.ascontiguousarray(out[k]))
        parts = [torch.empty_like(t) for _ in range(world)]
        dist.all_gather(parts, t)          # equal shard sizes here (6 envs / 2 ranks)
        gathered[k] = torch.cat(parts).numpy()
    dist.barrier()
    if rank == 0:
        q.put(gathered)
    dist.destroy_process_group()


def test_two_rank_shards_equal_unsharded_run():
    world, port = 2, 29000 + os.getpid() % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = q.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = W.config(4, n_envs=6)
    ref = _run_shard(w, 0, w.E, steps=3)
    for k, v in got.items():
        assert np.array_equal(v, ref[k]), k
    assert np.abs(ref["ft_noisy"]).max() > 0          # the noise chain really ran (drift is never 0)

"""The N > 1 path: environments are partitioned across ranks with no data-path collective; one gather of the
per-environment rows at the end.  world_size-2 gloo test on CPU, plus the partition's
invariants.  The per-environment "result" used here is a plain function of each environment's inputs, so the test
needs no GPU and none of the method's arithmetic."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2104_02646_b200 import scenes, sharding


@pytest.mark.parametrize("n_envs,world", [(1024, 8), (5, 2), (3, 4), (1, 2), (7, 7), (1000, 3)])
def test_env_blocks_tile_the_batch(n_envs, world):
    blocks = [sharding.env_block(n_envs, world, r) for r in range(world)]
    assert blocks[0][0] == 0 and blocks[-1][1] == n_envs
    for (a, b), (c, d) in zip(blocks, blocks[1:]):
        assert b == c and a <= b
    sizes = [b - a for a, b in blocks]
    assert max(sizes) - min(sizes) <= 1 and sum(sizes) == n_envs
    with pytest.raises(ValueError):
        sharding.env_block(n_envs, world, world)


def test_shard_scene_slices_every_env_array():
    sc = scenes.make_scene(3, small=True)  # 5 environments
    parts = [sharding.shard_scene(sc, 2, r) for r in range(2)]
    assert [p.n_envs for p in parts] == [3, 2]
    for k in ("x0", "v0", "mass", "tet_mu", "tet_lambda", "mu_c"):
        assert np.array_equal(np.concatenate([getattr(p, k) for p in parts], 0), getattr(sc, k)), k
    for k, v in sc.truth.items():
        assert np.array_equal(np.concatenate([p.truth[k] for p in parts], 0), v), k
    assert parts[0].tets is sc.tets and parts[0].x_rest is sc.x_rest  # the mesh is shared, not copied
    assert sharding.shard_scene(scenes.make_scene(0, small=True), 2, 1) is None  # one environment, second rank idle


def _worker(rank, world, port, n_envs, q):
    import torch
    import torch.distributed as dist

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        sc = scenes.batched_sysid_scene(n_envs=n_envs, n_substeps=4, y0=0.02)
        part = sharding.shard_scene(sc, world, rank)
        # stand-in for the per-environment results of a rollout: (mu_0, lambda_0, mass_0) of each owned environment
        if part is None:
            local = torch.zeros((0, 3), dtype=torch.float64)
        else:
            local = torch.as_tensor(np.stack([part.tet_mu[:, 0], part.tet_lambda[:, 0], part.mass[:, 0]], 1).astype(np.float64))
        rows = sharding.gather_env_rows(local, n_envs, dist)
        # weak-scaling timing contract of bench.py: barrier, then MAX over ranks
        t = torch.tensor([float(rank + 1)])
        dist.barrier()
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        q.put((rank, rows.numpy(), float(t.item())))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_envs", [5, 1])
def test_two_rank_gloo_gather_reassembles_env_order(n_envs):
    import torch.multiprocessing as mp

    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n_envs, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    sc = scenes.batched_sysid_scene(n_envs=n_envs, n_substeps=4, y0=0.02)
    want = np.stack([sc.tet_mu[:, 0], sc.tet_lambda[:, 0], sc.mass[:, 0]], 1).astype(np.float64)
    for rank, rows, tmax in got:
        assert rows.shape == (n_envs, 3) and np.array_equal(rows, want), rank
        assert tmax == 2.0

"""N > 1 path: environments are independent given the shared bitmap, so ranks take
contiguous env shards with no data-path collective.  world_size-2 gloo test on CPU: the sharded
oracle step, gathered, equals the single-process step bit for bit."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _inputs():
    from harness import workloads as W
    import oracle
    wl = W.make_workload(1, n_envs=48)
    n = wl.n_envs
    st = np.zeros((8, n), np.float32)
    dp = np.zeros(n, np.float32)
    ep = np.zeros(n, np.int32)
    oracle.reset(wl.occ, wl.resolution, wl.footprint, None, wl.goal_dist_min, wl.goal_dist_max,
                 np.ones(n, np.uint8), W.seed_tape(wl, 1)[0], st, dp, ep)
    return wl, st, dp, ep, W.action_tape(wl, 1)[0]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from harness import workloads as W
    import oracle
    wl, st, dp, ep, act = _inputs()
    lo, hi = W.shard_envs(wl.n_envs, rank, world)
    s = np.ascontiguousarray(st[:, lo:hi])
    out = oracle.step(wl, s, act[lo:hi], None, dp[lo:hi].copy(), ep[lo:hi].copy())
    mine = torch.from_numpy(np.concatenate([out["ranges"], s.T, out["reward"][:, None]], 1))
    sizes = [W.shard_envs(wl.n_envs, r, world) for r in range(world)]
    bufs = [torch.empty(b - a, mine.shape[1]) for a, b in sizes]
    dist.all_gather(bufs, mine) if len({b - a for a, b in sizes}) == 1 else dist.all_gather_object(bufs, mine)
    if rank == 0:
        q.put(torch.cat([torch.as_tensor(b) for b in bufs], 0).numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_env_sharding_world_size_2():
    sys.path.insert(0, ROOT)
    import oracle
    oracle.build()
    from harness import workloads as W
    assert W.shard_envs(10, 0, 3) == (0, 4) and W.shard_envs(10, 2, 3) == (7, 10)
    covered = [W.shard_envs(65536, r, 8) for r in range(8)]
    assert covered[0][0] == 0 and covered[-1][1] == 65536 and all(a[1] == b[0] for a, b in zip(covered, covered[1:]))
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    wl, st, dp, ep, act = _inputs()
    out = oracle.step(wl, st, act, None, dp, ep)
    want = np.concatenate([out["ranges"], st.T, out["reward"][:, None]], 1)
    assert np.array_equal(got, want)

"""World-size-2 gloo test of the N>1 host logic: disjoint group shards, one-scalar dt reduction; the sharded
oracle run equals the unsharded one bit for bit (groups are independent)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from paper_1712_07070_b200 import inputs, sharding
    f = inputs.turbulence_field(32, 1712, kmax=4, gamma=5 / 3)
    padded = inputs.pack_periodic(f)
    lo, hi = sharding.shard_range(padded.shape[0], rank, world)
    mine = padded[lo:hi].contiguous()
    dt_local, _ = oracle.cfl_dt(inputs.interior(mine).contiguous().numpy(), 1 / 32, 5 / 3, 0.4, 1)
    dt = sharding.global_dt(torch.tensor([dt_local], dtype=torch.float64))
    r = oracle.fluid_advance(mine.numpy(), dt.item(), 1 / 32, 5 / 3, 1, 1, 1)
    q.put((rank, lo, hi, dt_local, dt.item(), r["out"]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_groups_and_reduce_dt():
    sys.path.insert(0, ROOT)
    import oracle
    from paper_1712_07070_b200 import inputs, sharding
    assert [sharding.shard_range(7, r, 3) for r in range(3)] == [(0, 3), (3, 5), (5, 7)]
    assert sharding.shard_range(8, 1, 2) == (4, 8)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=300) for _ in range(2)], key=lambda x: x[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    f = inputs.turbulence_field(32, 1712, kmax=4, gamma=5 / 3)
    padded = inputs.pack_periodic(f)
    dt_all, _ = oracle.cfl_dt(inputs.interior(padded).contiguous().numpy(), 1 / 32, 5 / 3, 0.4, 1)
    assert res[0][4] == res[1][4] == min(res[0][3], res[1][3]) == dt_all
    assert (res[0][1], res[0][2], res[1][1], res[1][2]) == (0, 4, 4, 8)
    full = oracle.fluid_advance(padded.numpy(), dt_all, 1 / 32, 5 / 3, 1, 1, 1)["out"]
    assert np.array_equal(np.concatenate([res[0][5], res[1][5]]), full)

"""World-size-2 gloo test of the N>1 host logic: disjoint group shards, one-scalar dt reduction; the sharded
oracle run equals the unsharded one bit for bit (groups are independent)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q, path):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from paper_1712_07070_b200 import inputs, sharding
    padded = torch.from_numpy(np.load(path))      # the very bytes the parent compares against (not regenerated per process)
    lo, hi = sharding.shard_range(padded.shape[0], rank, world)
    mine = padded[lo:hi].contiguous()
    dt_local, _ = oracle.cfl_dt(inputs.interior(mine).contiguous().numpy(), 1 / 32, 5 / 3, 0.4, 1)
    dt = sharding.global_dt(torch.tensor([dt_local], dtype=torch.float64))
    r = oracle.fluid_advance(mine.numpy(), dt.item(), 1 / 32, 5 / 3, 1, 1, 1)
    q.put((rank, lo, hi, dt_local, dt.item(), r["out"]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_groups_and_reduce_dt(tmp_path):
    sys.path.insert(0, ROOT)
    import oracle
    from paper_1712_07070_b200 import inputs, sharding
    assert [sharding.shard_range(7, r, 3) for r in range(3)] == [(0, 3), (3, 5), (5, 7)]
    assert sharding.shard_range(8, 1, 2) == (4, 8)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    f = inputs.turbulence_field(32, 1712, kmax=4, gamma=5 / 3)
    padded = inputs.pack_periodic(f)
    path = str(tmp_path / "padded.npy")
    np.save(path, padded.numpy())
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q, path)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=900) for _ in range(2)], key=lambda x: x[0])
    for p in procs:
        p.join(timeout=600)
        assert p.exitcode == 0
    dt_all, _ = oracle.cfl_dt(inputs.interior(padded).contiguous().numpy(), 1 / 32, 5 / 3, 0.4, 1)
    assert res[0][4] == res[1][4] == min(res[0][3], res[1][3]) == dt_all
    assert (res[0][1], res[0][2], res[1][1], res[1][2]) == (0, 4, 4, 8)
    full = oracle.fluid_advance(padded.numpy(), dt_all, 1 / 32, 5 / 3, 1, 1, 1)["out"]
    assert np.array_equal(np.concatenate([res[0][5], res[1][5]]), full)


def _retry_worker(rank, world, port, q, path, dt0, dh):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from paper_1712_07070_b200 import inputs, sharding
    oracle.set_threads(2)
    padded = torch.from_numpy(np.load(path))      # the parent's bytes, not a regenerated field
    lo, hi = sharding.shard_range(padded.shape[0], rank, world)
    mine = padded[lo:hi].contiguous().numpy()
    last, counts = {}, []

    def step(dt):
        last["r"] = oracle.fluid_advance(mine, dt, dh, 5 / 3, 1, 1, 1)
        counts.append(last["r"]["stats"]["n_unphysical"])
        return counts[-1]

    dt_used, k = sharding.retry_level(step, dt0)
    aborted = False
    try:
        sharding.retry_level(step, dt0, dt_min=1.01 * dt_used)
    except ArithmeticError:
        aborted = True
    q.put((rank, dt_used, k, counts[:k + 1], last["r"]["out"] if not aborted else None, aborted,
           oracle.fluid_advance(mine, dt_used, dh, 5 / 3, 1, 1, 1)["out"]))
    dist.barrier()
    dist.destroy_process_group()


def _retry_inputs(oracle, inputs):
    # groups are independent given their padded inputs: rank 0's half comes from Mach-3 turbulence, rank 1's from a calm field
    rough = inputs.pack_periodic(inputs.turbulence_field(32, 3, kmax=6, gamma=5 / 3, mach=3.0, sigma=1.0))
    calm = inputs.pack_periodic(inputs.turbulence_field(32, 4, kmax=4, gamma=5 / 3, mach=0.3, sigma=0.2))
    padded = torch.cat([rough[:4], calm[4:]]).contiguous()
    dh = 1 / 32
    dt0 = 5.0 * oracle.cfl_dt(inputs.interior(padded).contiguous().numpy(), dh, 5 / 3, 0.5, 1)[0]
    return padded, dt0, dh


def test_two_ranks_retry_the_level_together(tmp_path):
    """Remedy (iv) is level-wide (L107): both ranks take the same number of reductions and the same dt as the unsharded
    oracle loop, also in attempts where one rank's own shard had no unphysical cell; both abort together."""
    sys.path.insert(0, ROOT)
    import oracle
    from paper_1712_07070_b200 import inputs
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    padded, dt0, dh = _retry_inputs(oracle, inputs)
    path = str(tmp_path / "padded.npy")
    np.save(path, padded.numpy())
    procs = [ctx.Process(target=_retry_worker, args=(r, 2, port, q, path, dt0, dh)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=900) for _ in range(2)], key=lambda x: x[0])
    for p in procs:
        p.join(timeout=600)
        assert p.exitcode == 0
    ref = oracle.fluid_advance_retry(padded.numpy(), dt0, dh, 5 / 3, 1, 1, 1)
    assert ref["n_retries"] >= 2
    for r in res:
        assert (r[1], r[2]) == (ref["dt_used"], ref["n_retries"]) and r[5]
    assert np.array_equal(np.concatenate([res[0][6], res[1][6]]), ref["out"])
    c0, c1 = res[0][3], res[1][3]
    assert all(a + b > 0 for a, b in zip(c0[:-1], c1[:-1])) and c0[-1] == c1[-1] == 0
    assert all(b == 0 for b in c1), (c0, c1)          # rank 1 alone would never have retried: the decision is the level's


def test_count_reduction_picks_the_device_the_backend_needs(monkeypatch):
    """bench.py initialises NCCL only: a CPU tensor cannot be all-reduced there.  The placement is decided by
    the backend, not hard-coded; a tensor argument (the device counter) is accepted as well as an int."""
    sys.path.insert(0, ROOT)
    from paper_1712_07070_b200 import sharding
    monkeypatch.setattr(sharding.dist, "get_backend", lambda: "gloo")
    assert sharding._reduce_device().type == "cpu"
    monkeypatch.setattr(sharding.dist, "get_backend", lambda: "nccl")
    monkeypatch.setattr(sharding.torch.cuda, "current_device", lambda: 3)
    assert sharding._reduce_device() == torch.device("cuda", 3)
    assert sharding.global_count(5) == 5 and sharding.global_count(torch.tensor([7], dtype=torch.int32)) == 7   # no group: identity

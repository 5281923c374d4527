"""World-size-2 gloo test of the host logic of the multi-GPU path."""
import os
import socket

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2503_24286_b200 import inputs, sharding


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # weak scaling: own seed, own batch
        st = inputs.config_states(0, n=257, seed=sharding.rank_state_seed(0, rank))
        # strong sharding of one field
        lo, cnt = sharding.rank_slab(1000, rank, world)
        # the slowest rank sets the step time
        t = sharding.max_over_ranks(10.0 + 5.0 * rank)
        out.put((rank, float(st["T"][0]), lo, cnt, t, sharding.job_throughput(257, world, t)))
    finally:
        dist.destroy_process_group()


def test_two_ranks_own_disjoint_work_and_share_only_the_step_time():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, T0, lo0, c0, t0, v0), (r1, T1, lo1, c1, t1, v1) = res
    assert T0 != T1                                   # different batches
    assert lo0 == 0 and lo0 + c0 == lo1 and lo1 + c1 == 1000 and c0 % 32 == 0   # slabs tile the field
    assert t0 == t1 == 15.0                           # max over ranks, seen by both
    assert v0 == v1 == 2 * 257 / 15e-3


def _slab_worker(rank, world, port, out):
    """What `bench.py --scaling strong` does on every rank, with the oracle in place of the GPU: the same seeded field,
    this rank's slab of it, the rates of the slab's points."""
    from oracle import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        full = inputs.config_states(0, n=1000, seed=sharding.rank_state_seed(0, 0))
        lo, cnt = sharding.rank_slab(1000, rank, world)
        st = {k: np.ascontiguousarray(v[..., lo:lo + cnt]) for k, v in full.items()}
        om = oracle.Oracle(inputs.config_mechanism(0)).get_net_production_rates(st["rho"], st["T"], st["Y"], want_bound=False)
        om = om[0] if isinstance(om, tuple) else om
        out.put((rank, lo, cnt, np.asarray(om)))
    finally:
        dist.destroy_process_group()


def test_strong_sharding_slabs_reproduce_the_single_rank_field():
    """The ranks' slab results, laid side by side, are the single-rank result of the whole field: every point computed
    exactly once, none skipped, bit for bit (points are independent)."""
    from oracle import oracle
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_slab_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=120) for _ in procs), key=lambda r: r[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    full = inputs.config_states(0, n=1000, seed=sharding.rank_state_seed(0, 0))
    whole = oracle.Oracle(inputs.config_mechanism(0)).get_net_production_rates(full["rho"], full["T"], full["Y"], want_bound=False)
    whole = whole[0] if isinstance(whole, tuple) else whole
    assert res[0][1] == 0 and res[0][1] + res[0][2] == res[1][1] and res[1][1] + res[1][2] == 1000
    joined = np.concatenate([r[3] for r in res], axis=1)
    assert joined.shape == whole.shape and np.array_equal(joined, whole)


def test_slabs_partition_any_size():
    for n in (0, 1, 31, 32, 33, 1000, 4096 + 5):
        for world in (1, 2, 3, 8):
            spans = [sharding.rank_slab(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and sum(c for _, c in spans) == n
            for (a, ca), (b, _) in zip(spans, spans[1:]):
                assert a + ca == b
    assert sharding.max_over_ranks(3.5) == 3.5        # no process group: identity
    assert len({sharding.rank_state_seed(2, r) for r in range(8)}) == 8

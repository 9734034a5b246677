"""CPU tests of bench.py's host logic: the N > 1 aggregation (gloo, world size 2: timing = max over
ranks, work = sum over ranks -- the path does not shard, ranks are independent replicas), the oracle
sample plan and the flop accounting."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist

    import bench

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert bench.dist_env() == (rank, world, rank)
    ms = bench.max_over_ranks(100.0 + 50.0 * rank, world)          # rank 1 is the slow replica
    flops = bench.sum_over_ranks(1e12 * (rank + 1), world)
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, ms, flops))


def test_replica_aggregation_world_size_2_gloo():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, flops in res:
        assert ms == 150.0 and flops == 3e12                        # every rank sees max time, summed work
    # whole-job value = all ranks' work / slowest rank's time
    assert res[0][2] / (res[0][1] * 1e-3) / 1e12 == pytest.approx(20.0)


def test_single_rank_is_identity_and_flop_accounting():
    import bench

    assert bench.max_over_ranks(3.5, 1) == 3.5 and bench.sum_over_ranks(2.0, 1) == 2.0
    n = 8192
    assert bench.logical_flops_per_layer(n, False) == 2 * n ** 3      # one N^3 product, 2 flops per FMA
    assert bench.logical_flops_per_layer(n, True) == 6 * n ** 3       # + X.X1 and X1.X [north_star]
    assert bench.issued_flops_per_layer(n, False) == 3 * n ** 3       # 3 plane products on half the tiles
    assert bench.issued_flops_per_layer(n, True) == 9 * n ** 3


def test_oracle_sample_plan_is_bounded():
    import bench

    plan = bench.oracle_sample_plan(8192, True, budget_s=1e9)          # unlimited budget: response, 1 layer
    assert plan["response"] and plan["max_layers"] == 1 and plan["products"] == 4
    plan = bench.oracle_sample_plan(8192, True, budget_s=0.0)          # no budget: smallest sample
    assert not plan["response"] and plan["max_layers"] == 0 and plan["products"] == 1
    # the product count matches what the oracle loop really executes
    import numpy as np

    import oracle

    calls = {"n": 0}

    class Counting(np.ndarray):
        def __matmul__(self, other):
            calls["n"] += 1
            return np.asarray(self) @ np.asarray(other)

    rng = np.random.default_rng(0)
    A = rng.standard_normal((12, 12))
    H = (A + A.T) / 2
    for resp, k in ((True, 1), (False, 1), (False, 0)):
        n_mm = (k + 1) + (2 * k if resp else 0)
        r = oracle.sp2_density(H, 6, H1=H if resp else None, max_layers=k)
        assert r["layers"] == k and r["stop"] == "max_layers"
        assert bench.sample_text(dict(response=resp, max_layers=k, products=n_mm), 12).count(f"{n_mm} float64") == 1

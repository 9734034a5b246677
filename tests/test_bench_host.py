"""CPU tests of bench.py's host logic: the N > 1 aggregation (gloo, world size 2: timing = max over
ranks, work = sum over ranks -- the path does not shard, ranks are independent replicas), the replica launcher of
`bench.py --gpus N` (the real entry point with a stubbed step), the oracle sample plan and the flop accounting."""
import json
import subprocess
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


def _run_bench(argv, env_extra=None):
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    env.update(env_extra or {})
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + argv, capture_output=True, text=True, env=env,
                       timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout                          # rank 0 alone prints, exactly one JSON line
    return json.loads(lines[0])


def test_gpus_n_without_torchrun_starts_n_replicas():
    """`python bench.py --gpus 2` (no torchrun, as a user or the driver may start it) must run TWO ranks, not silently
    time one: main() re-launches itself under torch.distributed.run.  The step is stubbed (a sleep; rank 1 is 10 %
    slower), so this runs on CPU with gloo; everything else is the real entry point."""
    line = _run_bench(["--gpus", "2", "--steps", "4", "--warmup", "1", "--stub-ms", "25"])
    assert line["n_gpus"] == 2 and line["gpus_active"] == 2 and line["steps"] == 4
    assert 27.0 <= line["ms_per_step"] <= 60.0                # the slower rank (27.5 ms per step) sets the time
    assert line["value"] == pytest.approx(2 * 4 * 1e12 / (line["ms_per_step"] * 4e-3) / 1e12, rel=1e-9)   # work of BOTH ranks
    one = _run_bench(["--gpus", "1", "--steps", "4", "--warmup", "1", "--stub-ms", "25"])
    assert one["n_gpus"] == 1 and one["gpus_active"] == 1 and 24.0 <= one["ms_per_step"] <= 50.0


def test_workload_table_names_all_five_configs():
    import bench
    from paper_2107_02737_b200 import inputs

    for k in range(1, 6):
        idx, call = bench.WORKLOADS[f"config{k}"]
        assert idx == k and call == ("sequence" if k == 5 else "response" if inputs.CONFIGS[k].response else "density")
        assert f"N={inputs.CONFIGS[k].n}" in bench.config_text(inputs.CONFIGS[k], call)
    assert bench.WORKLOADS["response"] == bench.WORKLOADS["config4"] and bench.WORKLOADS["density"] == (4, "density")


def test_full_oracle_loop_is_chosen_when_it_fits_and_stale_traffic_is_not_reported(tmp_path):
    import bench

    plan = bench.oracle_sample_plan(128, False, layers=24)             # config 1: 25 tiny products: the full loop
    assert plan["max_layers"] is None and plan["products"] == 25
    plan = bench.oracle_sample_plan(16384, False, budget_s=0.0, layers=38, full_budget_s=1.0)   # config 5: a bounded sample
    assert plan["max_layers"] == 0
    assert "FULL loop" in bench.sample_text(dict(response=False, max_layers=None, products=25), 128, 1)
    # roofline.traffic is the committed ncu constant only while sp2_layer.cu is the file the capture was taken at
    val, src = bench.read_profile_traffic("response")
    blob = bench.git_blob_hash(os.path.join(ROOT, "paper_2107_02737_b200", "csrc", "sp2_layer.cu"))
    if blob in src and "STALE" not in src:
        assert val is not None and val > 1e8
    else:
        assert val is None and "STALE" in src

#!/usr/bin/env python
"""bench.py -- BASELINE.json's headline metric on one B200 (or N independent replicas).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload response|density]

A "step" is one pass of the whole hot path over one synthetic Hamiltonian
of BASELINE.json config 4 (N = 8192, N_occ = 4096, gap 0.05, H and H1 in float64): one
sp2_response call (D and D1; default) or one sp2_density call (--workload density).

value   = effective Tflop/s of the whole job = sum over ranks of F_logical * layers / max-over-ranks time,
          F_logical = 6 N^3 per layer with response, 2 N^3 density only (2 flops per multiply-add;
          the paper counts 1), inputs resident in HBM when the timed region starts.
e2e     = the same metric through sp2_response_host / sp2_density_host: HOST (pinned) buffers in,
          HOST buffers out, copies inside the timed region.
roofline= the layer kernel: issued tensor flops per launch (9 N^3, or 3 N^3 density only: three FP16
          plane products on the upper triangle) / mean launch duration from CUDA events recorded by
          the library on the launching stream around the layer launches, against the measured
          sustained bf16/fp16 dense peak of MEASURED_PEAKS.json.
Multi-GPU: the path does not shard: --gpus N runs N independent
replicas under torchrun, one per GPU, no data-path collective; scaling "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "effective Tflops & ms per density matrix (SP2, N=8192) vs tensor-pipe peak"
UNIT = "Tflop/s (effective, 2 flops per FMA)"
CONFIG_INDEX = 4


def logical_flops_per_layer(n, response):
    return (6.0 if response else 2.0) * float(n) ** 3


def issued_flops_per_layer(n, response):
    return (9.0 if response else 3.0) * float(n) ** 3


def read_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            p = json.load(f)
        return dict(sustained=float(p["bf16_tflops_sustained"]), burst=float(p["bf16_tflops"]),
                    hbm=float(p["hbm_gbs"]), source="measured (MEASURED_PEAKS.json)")
    except Exception:
        return dict(sustained=1400.0, burst=1590.0, hbm=6650.0, source="fallback (B200_PROFILING.md)")


def read_profile_traffic(workload):
    """dram bytes per layer launch from the committed ncu capture (profiles/roofline_traffic.txt), or None."""
    path = os.path.join(ROOT, "profiles", "roofline_traffic.txt")
    try:
        with open(path) as f:
            for line in f:
                line = line.split("#", 1)[0].strip()
                if "=" in line:
                    k, v = (s.strip() for s in line.split("=", 1))
                    if k == f"layer_dram_bytes_per_launch.{workload}":
                        return float(v)
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""

    QUERY = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def mark(self):
        """Start of the timed region: wait (bounded) for the first sample, then drop what was sampled before it."""
        t0 = time.perf_counter()
        while self.proc is not None and not self.rows and time.perf_counter() - t0 < 1.0:
            time.sleep(0.01)
        self.skip = len(self.rows)

    def start(self):
        self.skip = 0
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = self.rows[self.skip:] or self.rows[-1:]      # a very short region may hold no sample of its own
        for row in rows:
            parts = [s.strip() for s in row.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0]))
                smax.append(float(parts[1]))
            except ValueError:
                continue
            for name, val in zip(names, parts[2:6]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return dict(sm_mhz=statistics.median(sm) if sm else None, sm_max_mhz=max(smax) if smax else None,
                    samples=len(sm), reasons=sorted(reasons))


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def max_over_ranks(value, world, device=None):
    """MAX all-reduce of one float over the job (identity for world == 1).  No data-path collective:
    this only aggregates the timing, as the bench contract asks."""
    if world == 1:
        return float(value)
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value, world, device=None):
    if world == 1:
        return float(value)
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


# ------------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py executes oracle/): cpu_baseline and --impl reference
def oracle_sample_plan(n, response, budget_s=12.0):
    """Pick the bounded sample of the workload the unmodified oracle is timed on: the oracle loop
    with max_layers = k.  It evaluates X@X once per loop entry (k + 1 times) and X@Z, Z@X once per
    applied layer, so it runs (k + 1) + 2k (response) N^3-products.  A 1024^3 dgemm calibrates the host."""
    import numpy as np

    m = 1024
    a = np.random.default_rng(0).standard_normal((m, m))
    a @ a
    t0 = time.perf_counter()
    a @ a
    gf = 2.0 * m ** 3 / (time.perf_counter() - t0)
    per_product = 2.0 * float(n) ** 3 / gf
    for resp, k in ((response, 1), (False, 1), (False, 0)):
        products = (k + 1) + (2 * k if resp else 0)
        if products * per_product <= budget_s or (not resp and k == 0):
            return dict(response=resp, max_layers=k, products=products, host_gflops_estimate=gf / 1e9)


def time_oracle_sample(p, plan):
    import oracle

    H = p["H"].astype("float64")
    H1 = p["H1"].astype("float64") if plan["response"] else None
    t0 = time.perf_counter()
    oracle.sp2_density(H, p["n_occ"], H1=H1, max_layers=plan["max_layers"])
    dt = time.perf_counter() - t0
    tflops = plan["products"] * 2.0 * float(p["n"]) ** 3 / dt / 1e12
    return dt, tflops


def host_threads():
    try:
        from threadpoolctl import threadpool_info

        ths = [d.get("num_threads", 0) for d in threadpool_info() if d.get("user_api") == "blas"]
        if ths:
            return max(ths)
    except Exception:
        pass
    return len(os.sched_getaffinity(0))


def sample_text(plan, n):
    what = "response" if plan["response"] else "density-only"
    return (f"oracle.sp2_density on config {CONFIG_INDEX} (N={n}) with max_layers={plan['max_layers']} ({what}): "
            f"{plan['products']} float64 N^3 products of the first layer(s), NumPy/BLAS")


def make_problem(rank, device):
    from paper_2107_02737_b200 import inputs

    cfg = inputs.CONFIGS[CONFIG_INDEX]
    return inputs.make_problem(cfg, seed=cfg.seed + rank, device=device, want_h1=True)


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return 0
    import numpy as np  # noqa: F401

    response = args.workload == "response"
    p = make_problem(0, "cpu" if not _cuda_ok() else "cuda")
    n = p["n"]
    plan = oracle_sample_plan(n, response)
    times = []
    for it in range(args.warmup + args.steps):
        dt, _ = time_oracle_sample(p, plan)
        if it >= args.warmup:
            times.append(dt)
    total = sum(times)
    value = plan["products"] * 2.0 * float(n) ** 3 * len(times) / total / 1e12
    cores = host_threads()
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config {CONFIG_INDEX}: N={n}, N_occ={p['n_occ']}, gap 0.05, "
                               f"{'D and D1' if response else 'D only'}; each step = {sample_text(plan, n)}"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample_text(plan, n)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def _cuda_ok():
    try:
        import torch

        return torch.cuda.is_available()
    except Exception:
        return False


# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2107_02737_b200 import sp2      # raises if the CUDA library is missing: no fallback

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback for the product path)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    response = args.workload == "response"

    p = make_problem(rank, "cuda")
    n, n_occ = p["n"], p["n_occ"]
    H = torch.from_numpy(p["H"]).to(dev)
    H1 = torch.from_numpy(p["H1"]).to(dev) if response else None
    D = torch.empty_like(H)
    D1 = torch.empty_like(H) if response else None
    h = sp2.Sp2Handle(n, response=response, host_staging=True, refinement=args.refine > 0)
    if args.lanczos > 0:
        h.set_options(lanczos_steps=args.lanczos)
    if args.refine > 0:
        if response:
            raise SystemExit("--refine goes with --workload density")
        h.set_options(refine_layers=args.refine, lanczos_steps=args.lanczos)

    def step():
        if response:
            return h.response(H, H1, n_occ, out=D, out1=D1)[2]
        return h.density(H, n_occ, out=D)[1]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    sampler.start()                      # before the warm-up, so that samples are flowing when the timed region starts
    for _ in range(max(args.warmup, 3)):
        step()
    # ---- timed region: exactly K steps, CUDA events on the launching stream, barrier + sync both sides
    stream = torch.cuda.current_stream()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = h.launch_count
    barrier()
    sampler.mark()
    ev0.record(stream)
    results = [step() for _ in range(args.steps)]
    ev1.record(stream)
    barrier()
    clocks = sampler.stop()
    launches = h.launch_count - launches0
    my_ms = ev0.elapsed_time(ev1)
    ms = max_over_ranks(my_ms, world, dev)
    layers = [r["layers"] for r in results]
    my_flops = sum(logical_flops_per_layer(n, response) * L for L in layers)
    total_flops = sum_over_ranks(my_flops, world, dev)
    value = total_flops / (ms * 1e-3) / 1e12

    # ---- roofline of the dominant kernel (rank 0's replica): issued flops / mean layer-launch time
    peaks = read_peaks()
    layer_ms = sum(r["layers_ms"] for r in results) / sum(layers)
    achieved = issued_flops_per_layer(n, response) / (layer_ms * 1e-3) / 1e12
    roofline = {"bound": "tensor", "achieved": achieved, "peak": peaks["sustained"], "unit": "TFLOP/s",
                "frac": achieved / peaks["sustained"], "traffic": read_profile_traffic(args.workload),
                "kernel": "k_layer_tc<2> (tcgen05 kind::f16, FP16 hi/lo x3 products, upper triangle)",
                "flops_per_launch": issued_flops_per_layer(n, response), "ms_per_launch": layer_ms,
                "peak_source": peaks["source"] + ", sustained bf16 (= fp16 kind::f16 rate)",
                "frac_of_burst_peak": achieved / peaks["burst"], "frac_of_nominal_2250": achieved / 2250.0}

    # ---- parity sample at full size on this run's output (sampled entries the oracle computes one by one)
    parity = None
    if rank == 0:
        import oracle

        rng = np.random.default_rng(1)
        rows = rng.integers(0, n, 256)
        cols = rng.integers(0, n, 256)
        Dg = D[torch.from_numpy(rows).to(dev), torch.from_numpy(cols).to(dev)].cpu().numpy()
        De = oracle.density_from_eigenpairs(p["Q"], p["lam"], n_occ, rows, cols)
        r = results[-1]
        from paper_2107_02737_b200 import inputs

        E = inputs.band_energy_closed_form(p["lam"], n_occ)
        parity = {"max_abs_dD_sampled": float(np.abs(Dg - De).max()), "abs_trD_minus_nocc": abs(r["tr_d"] - n_occ),
                  "rel_d_trDH": abs(r["tr_dh"] - E) / abs(E), "layers": r["layers"]}

    # ---- end to end through the host-buffer C-ABI call (pinned host buffers, copies inside the timing)
    e2e_steps = max(1, min(args.steps, 3))
    Hh = torch.from_numpy(p["H"]).pin_memory()
    Dh = torch.empty(n, n, dtype=torch.float64).pin_memory()
    H1h = torch.from_numpy(p["H1"]).pin_memory() if response else None
    D1h = torch.empty(n, n, dtype=torch.float64).pin_memory() if response else None

    def step_host():
        if response:
            return h.response_host(Hh, H1h, n_occ, Dh, D1h)[2]
        return h.density_host(Hh, n_occ, Dh)[1]

    step_host()
    barrier()
    t0 = time.perf_counter()
    res_h = [step_host() for _ in range(e2e_steps)]
    torch.cuda.synchronize()
    my_e2e = time.perf_counter() - t0
    barrier()
    e2e_s = max_over_ranks(my_e2e, world, dev)
    e2e_flops = sum_over_ranks(sum(logical_flops_per_layer(n, response) * r["layers"] for r in res_h), world, dev)
    mats = 2 if response else 1
    e2e = {"value": e2e_flops / e2e_s / 1e12, "unit": UNIT, "h2d_bytes_per_step": mats * n * n * 8,
           "d2h_bytes_per_step": mats * n * n * 8 + 96, "steps": e2e_steps, "ms_per_step": 1e3 * e2e_s / e2e_steps}

    # ---- the oracle on this box's host cores, bounded sample (rank 0, N = 1 only)
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        plan = oracle_sample_plan(n, response, budget_s=20.0)
        dt, tf = time_oracle_sample(p, plan)
        cpu_baseline = {"value": tf, "unit": UNIT, "cores": host_threads(), "kind": "oracle",
                        "sample": sample_text(plan, n), "seconds": dt}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f16", "data": "synthetic",
            "config": {"workload": f"config {CONFIG_INDEX}: N={n}, N_occ={n_occ}, gap 0.05, f64 H"
                                   + (" and H1 -> D and D1 (sp2_response)" if response else " -> D (sp2_density)"),
                       "precision": "FP16 hi + lo operand planes (22 bits), FP32 accumulation in k-segments, f64 scalars, f64 in/out",
                       "replicas": world, "layers_per_step": layers, "refine_layers": args.refine, "lanczos_steps": args.lanczos,
                       "l2_policy": "inputs larger than L2 (H 537 MB, each FP16 plane 134 MB vs 126 MB L2)",
                       "flops_per_layer_logical": logical_flops_per_layer(n, response)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
            "cpu_baseline": cpu_baseline, "parity": parity,
            "paper_context": "paper: >100 'Tflops' (1 FMA = 1 flop) on one A100, N~19000 (PAPER.md:186); not the target",
        }
        print(json.dumps(line), flush=True)
    h.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_sequence(args):
    """--workload sequence: BASELINE.json config 5 (N = 16384, N_occ = 8192, gap 0.2, f32): K consecutive MD-step
    Hamiltonians H_t = H_0 + t 1e-3 P (formed on the device by this harness, outside the library) through
    sp2_sequence_begin / step / end -- no host synchronisation between steps.  Extra workload, not the headline."""
    import torch

    from paper_2107_02737_b200 import inputs, sp2

    rank, world, local = dist_env()
    torch.cuda.set_device(local)
    cfg = inputs.CONFIGS[5]
    p = inputs.make_problem(cfg, seed=cfg.seed + rank, device="cuda", want_p=True)
    n, n_occ = p["n"], p["n_occ"]
    H0 = torch.from_numpy(p["H"]).cuda()
    P = torch.from_numpy(p["P"]).cuda()
    Ht = torch.empty_like(H0)
    D = torch.empty_like(H0)
    h = sp2.Sp2Handle(n)
    if args.lanczos > 0:
        h.set_options(lanczos_steps=args.lanczos)
    for _ in range(max(args.warmup, 3)):
        h.density(H0, n_occ, out=D)
    stream = torch.cuda.current_stream()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    launches0 = h.launch_count
    torch.cuda.synchronize()
    sampler.start()
    ev0.record(stream)
    h.sequence_begin(n, n_occ, n_steps_hint=args.steps)
    for t in range(args.steps):
        torch.add(H0, P, alpha=1e-3 * t, out=Ht)        # harness, not library; stream-ordered before the step
        h.sequence_step(Ht, D)
    res = h.sequence_end()
    ev1.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = ev0.elapsed_time(ev1)
    layers = [r["layers"] for r in res]
    flops = sum(logical_flops_per_layer(n, False) * L for L in layers)
    line = {"metric": METRIC, "value": flops / (ms * 1e-3) / 1e12, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f16", "data": "synthetic",
            "config": {"workload": f"config 5: N={n}, N_occ={n_occ}, gap 0.2, f32, {args.steps} consecutive H_t through "
                                   "sp2_sequence_* (max_layers launches per step, one sync at the end)",
                       "lanczos_steps": args.lanczos, "layers_per_step": layers, "issued_tflops": 1.5 * flops / (ms * 1e-3) / 1e12,
                       "statuses": sorted({r["status"] for r in res}),
                       "max_abs_trD_minus_nocc": max(abs(r["tr_d"] - n_occ) for r in res)},
            "clocks": clocks, "gpu_launches": int(h.launch_count - launches0)}
    print(json.dumps(line), flush=True)
    h.close()
    return 0


def run_congruence(args):
    """--workload congruence: sp2_congruence (H_orth = Z^T H Z) at N = 8192, float64 in and out.
    Extra workload, not the headline; value = issued tensor Tflop/s of the two products
    (2 products x 3 plane products x 2 N^3)."""
    import torch

    from paper_2107_02737_b200 import sp2

    _, _, local = dist_env()
    torch.cuda.set_device(local)
    n = 8192
    g = torch.Generator(device="cuda").manual_seed(20210714)
    Z = torch.randn(n, n, dtype=torch.float64, device="cuda", generator=g) / n ** 0.5 + torch.eye(n, dtype=torch.float64, device="cuda")
    X = torch.randn(n, n, dtype=torch.float64, device="cuda", generator=g)
    X = 0.5 * (X + X.T)
    C = torch.empty_like(X)
    h = sp2.Sp2Handle(n, response=True)
    for _ in range(max(args.warmup, 3)):
        h.congruence(Z, X, out=C)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = h.launch_count
    torch.cuda.synchronize()
    ev0.record()
    for _ in range(args.steps):
        h.congruence(Z, X, out=C)
    ev1.record()
    torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / args.steps
    err = float((C - Z.T @ X @ Z).abs().max())          # cross-check with torch float64 (harness, not library)
    line = {"metric": "issued Tflop/s of sp2_congruence (Z^T X Z, N=8192)", "value": 12.0 * n ** 3 / (ms * 1e-3) / 1e12,
            "unit": "TFLOP/s (issued)", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f16",
            "data": "synthetic", "config": {"workload": "sp2_congruence: C = Z^T X Z, N=8192, f64 in/out, general Z, symmetric X",
                                            "max_abs_err_vs_torch_f64": err, "max_abs_C": float(C.abs().max())},
            "gpu_launches": int(h.launch_count - launches0)}
    print(json.dumps(line), flush=True)
    h.close()
    return 0


def run_batch(args):
    """--workload batch --batch B: sp2_response_batch on config 4's H with B perturbations: one
    stack of layers carries D and D1_0..D1_{B-1}.  Extra workload, not the headline.  value = effective Tflop/s with
    (2 + 4 B) N^3 logical flops per layer; the layer kernel issues (3 + 6 B) N^3."""
    import numpy as np
    import torch

    from paper_2107_02737_b200 import inputs, sp2

    _, _, local = dist_env()
    torch.cuda.set_device(local)
    B = args.batch
    cfg = inputs.CONFIGS[CONFIG_INDEX]
    p = inputs.make_problem(cfg, device="cuda", want_h1=False)
    n, n_occ = p["n"], p["n_occ"]
    H = torch.from_numpy(p["H"]).cuda()
    H1n = inputs.perturbations(n, B, seed=cfg.seed, decades=0.5)
    H1s = [torch.from_numpy(a).cuda() for a in H1n]
    D = torch.empty_like(H)
    D1s = [torch.empty_like(H) for _ in range(B)]
    h = sp2.Sp2Handle(n, batch=B)
    if args.lanczos > 0:
        h.set_options(lanczos_steps=args.lanczos)
    for _ in range(max(args.warmup, 3)):
        h.response_batch(H, H1s, n_occ, out=D, out1s=D1s)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local)
    launches0 = h.launch_count
    torch.cuda.synchronize()
    sampler.start()
    ev0.record()
    res = [h.response_batch(H, H1s, n_occ, out=D, out1s=D1s)[3] for _ in range(args.steps)]
    ev1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = ev0.elapsed_time(ev1)
    layers = [r["layers"] for r in res]
    flops = sum((2.0 + 4.0 * B) * float(n) ** 3 * L for L in layers)
    layer_ms = sum(r["layers_ms"] for r in res) / sum(layers)
    issued = (3.0 + 6.0 * B) * float(n) ** 3 / (layer_ms * 1e-3) / 1e12
    peaks = read_peaks()
    # parity at full size: sampled entries of D and of every D1_b against the closed forms the oracle evaluates one by one
    import oracle

    rng = np.random.default_rng(2)
    rows, cols = rng.integers(0, n, 128), rng.integers(0, n, 128)
    ri, ci = torch.from_numpy(rows).cuda(), torch.from_numpy(cols).cuda()
    dD = float(np.abs(D[ri, ci].cpu().numpy() - oracle.density_from_eigenpairs(p["Q"], p["lam"], n_occ, rows, cols)).max())
    d1 = []
    for b in range(B):
        want = oracle.response_closed_form_sampled(p["Q"], p["lam"], n_occ, H1n[b], rows, cols)
        d1.append(float(np.abs(D1s[b][ri, ci].cpu().numpy() - want).max() / float(D1s[b].abs().max())))
    line = {"metric": METRIC, "value": flops / (ms * 1e-3) / 1e12, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f16", "data": "synthetic",
            "config": {"workload": f"config 4 H (N={n}, N_occ={n_occ}) with {B} perturbations -> D and {B} x D1 "
                                   "(sp2_response_batch)", "batch": B, "lanczos_steps": args.lanczos, "layers_per_step": layers,
                       },
            "clocks": clocks, "gpu_launches": int(h.launch_count - launches0),
            "roofline": {"bound": "tensor", "achieved": issued, "peak": peaks["sustained"], "unit": "TFLOP/s",
                         "frac": issued / peaks["sustained"], "traffic": None, "ms_per_launch": layer_ms,
                         "flops_per_launch": (3.0 + 6.0 * B) * float(n) ** 3, "peak_source": peaks["source"]},
            "parity": {"max_abs_dD_sampled": dD, "max_rel_dD1_sampled": d1, "abs_trD_minus_nocc": abs(res[-1]["tr_d"] - n_occ)}}
    print(json.dumps(line), flush=True)
    h.close()
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", choices=["response", "density", "sequence", "congruence", "batch"], default="response")
    ap.add_argument("--batch", type=int, default=4, help="perturbations per call of --workload batch (1..8)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--lanczos", type=int, default=0,
                    help="Lanczos steps for tighter spectral bounds (SURVEY 8(f) NEXT-3); extra, not the headline")
    ap.add_argument("--refine", type=int, default=0,
                    help="float64 refinement layers after the stack (PAPER.md:170; --workload density only); extra, not the headline")
    args = ap.parse_args(argv)
    if args.impl == "reference":
        return run_reference(args)
    if args.workload == "sequence":
        return run_sequence(args)
    if args.workload == "congruence":
        return run_congruence(args)
    if args.workload == "batch":
        return run_batch(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())

#!/usr/bin/env python
"""bench.py -- BASELINE.json's metric on one B200 (or N independent replicas), for each of its five configs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload config4|config1|config2|config3|config5|density|congruence|batch]

A "step" is one pass of the whole hot path over one synthetic Hamiltonian of the named
config.  Default = config 4, the configuration the metric is quoted on (N = 8192, N_occ = 4096, gap 0.05, H and H1 in
float64 -> D and D1 through ONE sp2_response call).  config1 / config3: one sp2_density call (N = 128 f64 / N = 6000
f32); config2: one sp2_response call (N = 1024); config5: one MD step of the 50-step sweep H_t = H_0 + t 1e-3 P
(N = 16384, f32) through sp2_sequence_begin / step / end (--steps = number of MD steps, one host sync at the end);
`density` = config 4's H through sp2_density (the "ms per density matrix" of the metric).

value    = effective Tflop/s of the whole job = sum over ranks of F_logical * layers / max-over-ranks time,
           F_logical = 6 N^3 per layer with response, 2 N^3 density only (2 flops per multiply-add; the paper counts
           1), inputs resident in HBM when the timed region starts.
e2e      = the same metric through the host-buffer C-ABI calls (sp2_response_host / sp2_density_host): pinned HOST
           buffers in, HOST buffers out, copies inside the timed region.
roofline = the layer kernel: issued tensor flops per launch (9 N^3, or 3 N^3 density only: three FP16 plane products
           on the upper triangle) / mean launch duration from CUDA events recorded by the library on the launching
           stream around the layer launches, against the measured sustained bf16/fp16 dense peak of
           MEASURED_PEAKS.json.  Configs 1-2 are launch/latency-bound: bound "latency", us per layer.
cpu_baseline = the unmodified oracle on this box's host cores: the FULL loop where that takes about a minute or
           less (configs 1-3), else a bounded sample; plus numpy.linalg.eigh + V_occ V_occ^T (the diagonalisation
           route the paper compares against) for N <= 6000 (N = 8192 with --cpu-eigh).
Multi-GPU: the path does not shard: --gpus N runs N independent replicas, one per GPU,
no data-path collective, scaling "weak".  Under torchrun the ranks come from the environment; started plainly with
--gpus N > 1 this script re-launches itself under torch.distributed.run with N ranks.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import socket
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
CONFIG_INDEX = 4                      # the configuration BASELINE.json's metric is quoted on
L2_BYTES = 126 * 2 ** 20

# workload name -> (config index, C-ABI call)
WORKLOADS = {
    "config1": (1, "density"), "config2": (2, "response"), "config3": (3, "density"), "config4": (4, "response"),
    "config5": (5, "sequence"), "response": (4, "response"), "density": (4, "density"), "sequence": (5, "sequence"),
}


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


def git_blob_hash(path):
    """`git hash-object` of a file (sha1 over "blob <len>\\0" + content), without calling git."""
    with open(path, "rb") as f:
        data = f.read()
    return hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()


def read_profile_traffic(key):
    """DRAM bytes per layer launch from the committed ncu capture (profiles/roofline_traffic.txt) -> (bytes or None,
    source string).  The file records the git blob hash of csrc/sp2_layer.cu the capture was taken at; if the kernel
    source has changed since, the constant is stale and None is returned instead of passing it off as a measurement."""
    path = os.path.join(ROOT, "profiles", "roofline_traffic.txt")
    vals = {}
    try:
        with open(path) as f:
            for line in f:
                line = line.split("#", 1)[0].strip()
                if "=" in line:
                    k, v = (s.strip() for s in line.split("=", 1))
                    vals[k] = v
    except Exception:
        return None, "profiles/roofline_traffic.txt missing"
    want = vals.get("sp2_layer_cu_blob")
    have = git_blob_hash(os.path.join(ROOT, "paper_2107_02737_b200", "csrc", "sp2_layer.cu"))
    src = f"profiles/roofline_traffic.txt ({vals.get('capture', 'ncu --set full')}), sp2_layer.cu blob {want}"
    if want != have:
        return None, src + f" -- STALE: current sp2_layer.cu blob is {have}"
    v = vals.get(f"layer_dram_bytes_per_launch.{key}")
    return (float(v) if v is not None else None), src


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


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def spawn_replicas(argv, n):
    """Started without torchrun but with --gpus N > 1: run the same command line under torch.distributed.run with
    N ranks on this node (one replica per GPU), and pass its exit code on."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr",
           "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + list(argv)
    return subprocess.call(cmd)


# ------------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py executes oracle/): cpu_baseline and --impl reference
def host_gflops():
    """float64 matmul rate of this host (a 1024^3 product), to size the oracle sample."""
    import numpy as np

    m = 1024
    a = np.random.default_rng(0).standard_normal((m, m))
    a @ a
    t0 = time.perf_counter()
    a @ a
    return 2.0 * m ** 3 / (time.perf_counter() - t0) / 1e9


def oracle_sample_plan(n, response, budget_s=12.0, layers=None, full_budget_s=60.0):
    """Pick what the unmodified oracle is timed on.  With `layers` (the layer count the GPU solve needed) and a full
    loop that fits `full_budget_s`: the WHOLE oracle loop (max_layers = None).  Otherwise a bounded sample: the oracle
    loop with max_layers = k.  It evaluates X@X once per loop entry (k + 1 times) and X@Z, Z@X once per applied
    layer, so it runs (k + 1) + 2k (response) N^3-products.  A 1024^3 dgemm calibrates the host."""
    gf = host_gflops() * 1e9
    per_product = 2.0 * float(n) ** 3 / gf
    if layers is not None:
        products = (layers + 1) + (2 * layers if response else 0)
        if products * per_product <= full_budget_s:
            return dict(response=response, max_layers=None, products=products, host_gflops_estimate=gf / 1e9)
    for resp, k in ((response, 1), (False, 1), (False, 0)):
        products = (k + 1) + (2 * k if resp else 0)
        if products * per_product <= budget_s or (not resp and k == 0):
            return dict(response=resp, max_layers=k, products=products, host_gflops_estimate=gf / 1e9)


def time_oracle_sample(p, plan):
    """-> (seconds, Tflop/s of the float64 products actually executed, layers run)."""
    import oracle

    H = p["H"].astype("float64")
    H1 = p["H1"].astype("float64") if plan["response"] else None
    kw = {} if plan["max_layers"] is None else dict(max_layers=plan["max_layers"])
    t0 = time.perf_counter()
    r = oracle.sp2_density(H, p["n_occ"], H1=H1, **kw)
    dt = time.perf_counter() - t0
    L = r["layers"]
    products = (L + 1) + (2 * L if plan["response"] else 0)
    return dt, products * 2.0 * float(p["n"]) ** 3 / dt / 1e12, L


def time_eigh(p):
    """numpy.linalg.eigh + V_occ V_occ^T in float64: the diagonalisation route."""
    import numpy as np

    H = p["H"].astype("float64")
    t0 = time.perf_counter()
    w, V = np.linalg.eigh(H)
    Vo = V[:, :p["n_occ"]]
    D = Vo @ Vo.T
    dt = time.perf_counter() - t0
    return dict(seconds=dt, what="numpy.linalg.eigh + V_occ V_occ^T, float64", tr_d=float(np.trace(D)))


def host_threads():
    try:
        from threadpoolctl import threadpool_info

        ths = [d.get("num_threads", 0) for d in threadpool_info() if d.get("user_api") == "blas"]
        if ths:
            return max(ths)
    except Exception:
        pass
    return len(os.sched_getaffinity(0))


def sample_text(plan, n, cfg_index=CONFIG_INDEX):
    what = "response" if plan["response"] else "density-only"
    if plan["max_layers"] is None:
        return (f"oracle.sp2_density on config {cfg_index} (N={n}), the FULL loop ({what}): "
                f"{plan['products']} float64 N^3 products, NumPy/BLAS")
    return (f"oracle.sp2_density on config {cfg_index} (N={n}) with max_layers={plan['max_layers']} ({what}): "
            f"{plan['products']} float64 N^3 products of the first layer(s), NumPy/BLAS")


def cpu_baseline_for(p, cfg_index, response, layers, args):
    """The oracle as it stands on this box's host cores (rank 0, N = 1 only)."""
    n = p["n"]
    plan = oracle_sample_plan(n, response, budget_s=20.0, layers=layers)
    dt, tf, L = time_oracle_sample(p, plan)
    out = {"value": tf, "unit": UNIT.replace("effective", "float64 products executed"), "cores": host_threads(),
           "kind": "oracle", "sample": sample_text(plan, n, cfg_index), "seconds": dt, "layers": L,
           "full_loop": plan["max_layers"] is None}
    if plan["max_layers"] is None:
        out["ms_per_density_matrix"] = 1e3 * dt
    if n <= 6000 or args.cpu_eigh:
        out["eigh"] = time_eigh(p)
    return out


def make_problem(rank, device, cfg_index=CONFIG_INDEX, want_h1=None, want_p=False):
    from paper_2107_02737_b200 import inputs

    cfg = inputs.CONFIGS[cfg_index]
    return inputs.make_problem(cfg, seed=cfg.seed + rank, device=device if cfg.n >= 2048 else "cpu",
                               want_h1=cfg.response if want_h1 is None else want_h1, want_p=want_p)


def config_text(cfg, call):
    gap = cfg.unocc[0] - cfg.occ[1]
    tail = {"response": "H and H1 -> D and D1 (sp2_response)", "density": "H -> D (sp2_density)",
            "sequence": f"{cfg.n_steps} consecutive H_t = H_0 + t 1e-3 P -> D_t (sp2_sequence_*)"}[call]
    return f"config {cfg.index}: N={cfg.n}, N_occ={cfg.n_occ}, gap {gap:g}, {cfg.in_dtype} {tail}"


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return 0
    cfg_index, call = WORKLOADS.get(args.workload, (CONFIG_INDEX, "response"))
    response = call == "response"
    p = make_problem(0, "cuda" if _cuda_ok() else "cpu", cfg_index, want_h1=response)
    n = p["n"]
    plan = oracle_sample_plan(n, response)
    times, tfs = [], []
    for it in range(args.warmup + args.steps):
        dt, tf, _ = time_oracle_sample(p, plan)
        if it >= args.warmup:
            times.append(dt)
            tfs.append(tf)
    total = sum(times)
    value = sum(t * d for t, d in zip(tfs, times)) / total
    cores = host_threads()
    from paper_2107_02737_b200 import inputs

    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": config_text(inputs.CONFIGS[cfg_index], call) + f"; each step = {sample_text(plan, n, cfg_index)}"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample_text(plan, n, cfg_index)},
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
def run_stub(args):
    """Test hook (tests/test_bench_host.py): the launch, barrier, max-over-ranks timing and JSON line of the real
    entry point with the GPU step replaced by a sleep of --stub-ms (rank r sleeps (1 + r/10) times as long), gloo
    instead of NCCL, wall-clock instead of CUDA events.  Never used for a bench number: the line says so."""
    import torch.distributed as dist

    rank, world, _ = dist_env()
    if world > 1:
        dist.init_process_group("gloo", rank=rank, world_size=world)
    for _ in range(args.warmup):
        time.sleep(1e-3 * args.stub_ms)
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        time.sleep(1e-3 * args.stub_ms * (1.0 + 0.1 * rank))
    my_ms = 1e3 * (time.perf_counter() - t0)
    if world > 1:
        dist.barrier()
    ms = max_over_ranks(my_ms, world)
    flops = sum_over_ranks(1e12 * args.steps, world)
    active = sum_over_ranks(1.0, world)
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": flops / (ms * 1e-3) / 1e12, "unit": UNIT, "n_gpus": world,
                          "gpus_active": int(active), "steps": args.steps, "warmup": args.warmup,
                          "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
                          "vs_baseline": None, "dtype": "stub", "data": "none",
                          "config": {"workload": "STUB: sleep, not a measurement"}, "gpu_launches": 0}), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def apply_knobs(h, args):
    """The library options the command line exposes (all default to the library's own defaults), for every workload."""
    if args.lanczos > 0:
        h.set_options(lanczos_steps=args.lanczos)
    if args.max_ctas > 0 or args.persistent or args.seg_kb or args.cta_group or args.power or args.lockstep:
        h.set_options(max_ctas=args.max_ctas, persistent=args.persistent, seg_kb=args.seg_kb, cta_group=args.cta_group,
                      power_squarings=args.power, lockstep=args.lockstep)


def timed_steps(torch, step, k, flush_buf, barrier):
    """Time exactly k steps with CUDA events on the launching stream.  Inputs larger than L2 (flush_buf None): one
    pair of events brackets the k steps.  Inputs that fit in L2: a buffer larger than L2 is overwritten between steps
    and every step gets its own pair of events, so that the flush is NOT counted.  -> (ms of the k steps, results)."""
    stream = torch.cuda.current_stream()
    barrier()
    if flush_buf is None:
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        results = [step() for _ in range(k)]
        ev1.record(stream)
        barrier()
        return ev0.elapsed_time(ev1), results
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(k)]
    results = []
    for a, b in evs:
        flush_buf.add_(1)
        a.record(stream)
        results.append(step())
        b.record(stream)
    barrier()
    return sum(a.elapsed_time(b) for a, b in evs), results


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2107_02737_b200 import inputs, sp2      # raises if the CUDA library is missing: no fallback

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback for the product path)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cfg_index, call = WORKLOADS[args.workload]
    cfg = inputs.CONFIGS[cfg_index]
    response = call == "response"

    p = make_problem(rank, "cuda", cfg_index, want_h1=response)
    n, n_occ = p["n"], p["n_occ"]
    esz = p["H"].dtype.itemsize
    H = torch.from_numpy(p["H"]).to(dev)
    H1 = torch.from_numpy(p["H1"]).to(dev) if response else None
    D = torch.empty_like(H)
    D1 = torch.empty_like(H) if response else None
    h = sp2.Sp2Handle(n, response=response, host_staging=True, refinement=args.refine > 0)
    apply_knobs(h, args)
    if args.refine > 0:
        if response:
            raise SystemExit("--refine goes with a density workload")
        h.set_options(refine_layers=args.refine)

    def step():
        if response:
            return h.response(H, H1, n_occ, out=D, out1=D1)[2]
        return h.density(H, n_occ, out=D)[1]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    in_l2 = (1 + int(response)) * n * n * esz + 4 * (1 + int(response)) * n * n * 2 < L2_BYTES
    flush_buf = torch.zeros(2 * L2_BYTES // 4, dtype=torch.int32, device=dev) if in_l2 else None
    sampler = ClockSampler(local)
    sampler.start()                      # before the warm-up, so that samples are flowing when the timed region starts
    for _ in range(max(args.warmup, 3)):
        step()
    # ---- timed region: exactly K steps, CUDA events on the launching stream, barrier + sync both sides
    launches0 = h.launch_count
    barrier()
    sampler.mark()
    my_ms, results = timed_steps(torch, step, args.steps, flush_buf, barrier)
    clocks = sampler.stop()
    launches = h.launch_count - launches0
    ms = max_over_ranks(my_ms, world, dev)
    layers = [r["layers"] for r in results]
    my_flops = sum(logical_flops_per_layer(n, response) * L for L in layers)
    total_flops = sum_over_ranks(my_flops, world, dev)
    active = int(sum_over_ranks(1.0, world, dev))
    value = total_flops / (ms * 1e-3) / 1e12

    # ---- roofline of the dominant kernel (rank 0's replica): issued flops / mean layer-launch time
    peaks = read_peaks()
    layer_ms = sum(r["layers_ms"] for r in results) / sum(layers)
    achieved = issued_flops_per_layer(n, response) / (layer_ms * 1e-3) / 1e12
    latency_bound = n < 2048                                   # configs 1-2 are launch/latency-bound
    traffic, traffic_src = (read_profile_traffic("response" if response else "density") if cfg_index == 4
                            else (None, "no ncu --set full capture for this config"))
    roofline = {"bound": "latency" if latency_bound else "tensor", "achieved": achieved, "peak": peaks["sustained"],
                "unit": "TFLOP/s", "frac": achieved / peaks["sustained"], "traffic": traffic, "traffic_source": traffic_src,
                "kernel": "layer kernel (tcgen05 kind::f16, FP16 hi/lo x3 products, upper triangle)",
                "flops_per_launch": issued_flops_per_layer(n, response), "ms_per_launch": layer_ms,
                "us_per_layer": 1e3 * layer_ms,
                "peak_source": peaks["source"] + ", sustained bf16 (= fp16 kind::f16 rate)",
                "frac_of_burst_peak": achieved / peaks["burst"], "frac_of_nominal_2250": achieved / 2250.0}
    if latency_bound:
        roofline["note"] = ("launch/latency-bound size: the time per layer is set by the dependency chain of one layer "
                            "(load, MMA, epilogue, grid-wide reduction, controller), not by the tensor pipe")

    # ---- parity sample at full size on this run's output (sampled entries the oracle computes one by one)
    parity = None
    if rank == 0:
        import oracle

        rng = np.random.default_rng(1)
        rows = rng.integers(0, n, 256)
        cols = rng.integers(0, n, 256)
        ri, ci = torch.from_numpy(rows).to(dev), torch.from_numpy(cols).to(dev)
        Dg = D[ri, ci].double().cpu().numpy()
        De = oracle.density_from_eigenpairs(p["Q"], p["lam"], n_occ, rows, cols)
        r = results[-1]
        E = inputs.band_energy_closed_form(p["lam"], n_occ)
        parity = {"max_abs_dD_sampled": float(np.abs(Dg - De).max()), "abs_trD_minus_nocc": abs(r["tr_d"] - n_occ),
                  "rel_d_trDH": abs(r["tr_dh"] - E) / abs(E), "layers": r["layers"],
                  "reference": "exact projector / band energy from the generator's eigenpairs (oracle.density_from_eigenpairs)"}
        if response:
            D1e = oracle.response_closed_form_sampled(p["Q"], p["lam"], n_occ, p["H1"].astype(np.float64), rows, cols)
            parity["max_rel_dD1_sampled"] = float(np.abs(D1[ri, ci].double().cpu().numpy() - D1e).max() / float(D1.abs().max()))

    # ---- end to end through the host-buffer C-ABI call (pinned host buffers, copies inside the timing)
    e2e_steps = max(1, min(args.steps, 3))
    Hh = torch.from_numpy(p["H"]).pin_memory()
    Dh = torch.empty(n, n, dtype=Hh.dtype).pin_memory()
    H1h = torch.from_numpy(p["H1"]).pin_memory() if response else None
    D1h = torch.empty(n, n, dtype=Hh.dtype).pin_memory() if response else None

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
    # what the link alone costs: the same pinned buffers copied in and out with nothing in between (one stream, as
    # in the call: the solve needs all of H and H1 before its first kernel and D, D1 exist only after its last)
    scratch_dev = torch.empty_like(H)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for src in ([Hh, H1h] if response else [Hh]):
        scratch_dev.copy_(src, non_blocking=True)
    for dst in ([Dh, D1h] if response else [Dh]):
        dst.copy_(scratch_dev, non_blocking=True)
    torch.cuda.synchronize()
    link_ms = 1e3 * (time.perf_counter() - t0)
    del scratch_dev
    e2e = {"value": e2e_flops / e2e_s / 1e12, "unit": UNIT, "h2d_bytes_per_step": mats * n * n * esz,
           "d2h_bytes_per_step": mats * n * n * esz + 96, "steps": e2e_steps, "ms_per_step": 1e3 * e2e_s / e2e_steps,
           "link_ms_per_step": link_ms,
           "note": "link_ms_per_step = the same host<->device copies alone; e2e - device time cannot go below it in a blocking call"}

    # ---- the oracle on this box's host cores (rank 0, N = 1 only)
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu_baseline = cpu_baseline_for(p, cfg_index, response, layers[-1], args)

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "gpus_active": active, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f16", "data": "synthetic",
            "config": {"workload": config_text(cfg, call),
                       "precision": "FP16 hi + lo operand planes (22 bits), FP32 accumulation in k-segments, f64 scalars",
                       "replicas": world, "layers_per_step": layers, "refine_layers": args.refine, "lanczos_steps": args.lanczos, "power_squarings": args.power,
                       "l2_policy": ("L2 flushed between steps (a 252 MiB buffer is overwritten; every step has its own pair of "
                                     "CUDA events, the flush is not counted)" if in_l2 else
                                     f"inputs larger than L2 (H {n * n * esz / 2 ** 20:.0f} MiB, each FP16 plane "
                                     f"{n * n * 2 / 2 ** 20:.0f} MiB vs 126 MiB L2)"),
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
    """config5: BASELINE.json config 5 (N = 16384, N_occ = 8192, gap 0.2, f32): K consecutive MD-step Hamiltonians
    H_t = H_0 + t 1e-3 P (formed on the device by this harness, outside the library) through
    sp2_sequence_begin / step / end -- no host synchronisation between steps."""
    import numpy as np
    import torch

    from paper_2107_02737_b200 import inputs, sp2

    rank, world, local = dist_env()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=dev)
    cfg = inputs.CONFIGS[5]
    p = make_problem(rank, "cuda", 5, want_h1=False, want_p=True)
    n, n_occ = p["n"], p["n_occ"]
    H0 = torch.from_numpy(p["H"]).to(dev)
    P = torch.from_numpy(p["P"]).to(dev)
    Ht = torch.empty_like(H0)
    D = torch.empty_like(H0)
    D_first = torch.empty_like(H0)
    h = sp2.Sp2Handle(n, host_staging=True)
    apply_knobs(h, args)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    sampler.start()
    for _ in range(max(args.warmup, 3)):
        h.density(H0, n_occ, out=D)
    stream = torch.cuda.current_stream()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = h.launch_count
    barrier()
    sampler.mark()
    ev0.record(stream)
    h.sequence_begin(n, n_occ, n_steps_hint=args.steps)
    for t in range(args.steps):
        torch.add(H0, P, alpha=1e-3 * t, out=Ht)        # harness, not library; stream-ordered before the step
        h.sequence_step(Ht, D_first if t == 0 else D)
    res = h.sequence_end()
    ev1.record(stream)
    barrier()
    clocks = sampler.stop()
    launches = h.launch_count - launches0
    ms = max_over_ranks(ev0.elapsed_time(ev1), world, dev)
    layers = [r["layers"] for r in res]
    flops = sum_over_ranks(sum(logical_flops_per_layer(n, False) * L for L in layers), world, dev)
    active = int(sum_over_ranks(1.0, world, dev))
    value = flops / (ms * 1e-3) / 1e12
    peaks = read_peaks()
    # roofline: no per-launch events exist inside an un-synchronised sequence, so the issued flops of all layers are
    # divided by the WHOLE timed region (prologue, finalise and the harness' H_t update included: a lower bound on
    # the layer kernel's own rate)
    my_ms = ev0.elapsed_time(ev1)
    achieved = sum(issued_flops_per_layer(n, False) * L for L in layers) / (my_ms * 1e-3) / 1e12
    roofline = {"bound": "tensor", "achieved": achieved, "peak": peaks["sustained"], "unit": "TFLOP/s",
                "frac": achieved / peaks["sustained"], "traffic": None,
                "traffic_source": "no ncu --set full capture for this config",
                "kernel": "layer kernel (tcgen05 kind::f16, FP16 hi/lo x3 products, upper triangle)",
                "flops_per_launch": issued_flops_per_layer(n, False), "ms_per_launch": my_ms / sum(layers),
                "note": "whole timed region / layers (no per-launch events inside an un-synchronised sequence)",
                "peak_source": peaks["source"] + ", sustained bf16 (= fp16 kind::f16 rate)",
                "frac_of_burst_peak": achieved / peaks["burst"], "frac_of_nominal_2250": achieved / 2250.0}
    parity = None
    if rank == 0:
        import oracle

        rng = np.random.default_rng(1)
        rows, cols = rng.integers(0, n, 256), rng.integers(0, n, 256)
        Dg = D_first[torch.from_numpy(rows).to(dev), torch.from_numpy(cols).to(dev)].double().cpu().numpy()
        De = oracle.density_from_eigenpairs(p["Q"], p["lam"], n_occ, rows, cols)
        E = inputs.band_energy_closed_form(p["lam"], n_occ)
        parity = {"max_abs_dD_sampled_t0": float(np.abs(Dg - De).max()),
                  "max_abs_trD_minus_nocc_all_steps": max(abs(r["tr_d"] - n_occ) for r in res),
                  "rel_d_trDH_t0": abs(res[0]["tr_dh"] - E) / abs(E), "statuses": sorted({r["status"] for r in res}),
                  "reference": "t = 0: exact projector / band energy from the generator's eigenpairs"}
    # ---- e2e: per MD step through sp2_density_host (there is no host-buffer twin of the sequence call)
    Hh = torch.from_numpy(p["H"]).pin_memory()
    Dh = torch.empty(n, n, dtype=Hh.dtype).pin_memory()
    h.density_host(Hh, n_occ, Dh)
    barrier()
    e2e_steps = 2
    t0 = time.perf_counter()
    res_h = [h.density_host(Hh, n_occ, Dh)[1] for _ in range(e2e_steps)]
    torch.cuda.synchronize()
    my_e2e = time.perf_counter() - t0
    barrier()
    e2e_s = max_over_ranks(my_e2e, world, dev)
    e2e_flops = sum_over_ranks(sum(logical_flops_per_layer(n, False) * r["layers"] for r in res_h), world, dev)
    e2e = {"value": e2e_flops / e2e_s / 1e12, "unit": UNIT, "h2d_bytes_per_step": n * n * 4, "d2h_bytes_per_step": n * n * 4 + 96,
           "steps": e2e_steps, "ms_per_step": 1e3 * e2e_s / e2e_steps, "call": "sp2_density_host on H_0 (one MD step)"}
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu_baseline = cpu_baseline_for(p, 5, False, layers[0], args)
        cpu_baseline["sample"] += " (1 of the 50 steps' Hamiltonians, t = 0)"
    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "gpus_active": active, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f16", "data": "synthetic",
                "config": {"workload": config_text(cfg, "sequence") + f"; {args.steps} MD steps timed, one host sync at the end",
                           "precision": "FP16 hi + lo operand planes (22 bits), FP32 accumulation in k-segments, f64 scalars",
                           "replicas": world, "lanczos_steps": args.lanczos, "layers_per_step": layers,
                           "l2_policy": "inputs larger than L2 (H 1024 MiB, each FP16 plane 512 MiB vs 126 MiB L2)",
                           "flops_per_layer_logical": logical_flops_per_layer(n, False)},
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
                "cpu_baseline": cpu_baseline, "parity": parity,
                "paper_context": "paper: >100 'Tflops' (1 FMA = 1 flop) on one A100, N~19000 (PAPER.md:186); not the target"}
        print(json.dumps(line), flush=True)
    h.close()
    if world > 1:
        dist.destroy_process_group()
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
    apply_knobs(h, args)
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
    argv = list(sys.argv[1:] if argv is None else argv)
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed steps (default 5; 50 for config5)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", choices=sorted(WORKLOADS) + ["congruence", "batch"], default="config4")
    ap.add_argument("--batch", type=int, default=4, help="perturbations per call of --workload batch (1..8)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-eigh", action="store_true", help="also time numpy eigh + V_occ V_occ^T above N = 6000 (minutes)")
    ap.add_argument("--lanczos", type=int, default=0,
                    help="Lanczos steps for tighter spectral bounds (SURVEY 8(f) NEXT-3); extra, not the headline")
    ap.add_argument("--lockstep", type=int, default=0, help="sp2_options_t.lockstep: 0 auto, 1 on, 2 off")
    ap.add_argument("--power", type=int, default=0,
                    help="sp2_options_t.power_squarings: rigorous power-trace spectral bounds (SURVEY 8(f) NEXT-3); extra, not the headline")
    ap.add_argument("--refine", type=int, default=0,
                    help="float64 refinement layers after the stack (PAPER.md:170; density workloads only); extra, not the headline")
    ap.add_argument("--persistent", type=int, default=0, help="sp2_options_t.persistent (0 auto, 1 persistent kernel, 2 launch per layer)")
    ap.add_argument("--seg-kb", type=int, default=0, help="sp2_options_t.seg_kb (0 = default)")
    ap.add_argument("--cta-group", type=int, default=0, help="sp2_options_t.cta_group (0 = auto, 1 = 128x128 tiles, 2 = 256x256 on CTA pairs)")
    ap.add_argument("--max-ctas", type=int, default=0, help="sp2_options_t.max_ctas: use at most this many CTAs (0 = one per SM)")
    ap.add_argument("--stub-ms", type=float, default=0.0, help=argparse.SUPPRESS)   # test hook, see run_stub
    args = ap.parse_args(argv)
    if args.steps is None:
        args.steps = 50 if WORKLOADS.get(args.workload, (0, ""))[1] == "sequence" and args.impl == "ours" else 5
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_replicas(argv, args.gpus)      # rank 0 of the child job prints the JSON line
    if args.stub_ms > 0:
        return run_stub(args)
    if args.impl == "reference":
        return run_reference(args)
    if args.workload in WORKLOADS and WORKLOADS[args.workload][1] == "sequence":
        return run_sequence(args)
    if args.workload == "congruence":
        return run_congruence(args)
    if args.workload == "batch":
        return run_batch(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())

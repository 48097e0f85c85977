#!/usr/bin/env python
"""bench.py -- headline measurement: pairwise interactions/s (fp32) at N = 262,144 on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl reference]

A "step" is one pass of the whole hot path: one
kick-drift-kick leapfrog step = one all-pairs force evaluation (Eqs. 4-6) + the
fused split-j reduction / kick / drift / radius update, on BASELINE config 4
(two uniform stars of 131,072 elements, q = 0.6, seed 3; synthetic, recipe in
DESIGN.md).  interactions = N^2 ordered pairs per step.

  value      device-resident state, CUDA events on the launching stream around each
             nb_step(1); L2 flushed between steps; max over ranks.
  e2e        the same step through the C ABI with HOST (pinned) buffers: H2D of
             (x, v, a) + nb_step(1) + D2H of (x, v, a) inside the timed region.
  roofline   the all-pairs gravity kernel alone (nb_time_force_kernel: events on its stream)
             against the FP32 CUDA-core peak  SMs x 128 lanes x 2 flop x max clock,
             with the stated 21 flop / interaction convention ("alu" bound).
  per_config the other four BASELINE configs (the paper's kinds of run), each a few
             timed steps the same way (L2 flushed, events per step: mean, median, best) plus the same
             steps issued as one nb_step(K) call ("hot": what a run does), interactions/s, steps/s,
             % of FP32 peak by the 21-flop and the classic 20-flop conventions, gravity-kernel and
             contact-pass times.
  cpu_baseline  the fp64 oracle (oracle/, as it stands) on the box's host cores: a seeded sample of
             i-rows against all N elements on all cores, the same on ONE thread, and one full
             evaluation of config 2.

The path does not shard (north_star: one GPU, no collectives): with --gpus N > 1
every rank runs an independent replica ("replicas only", weak scaling), no
data-path collective; the only torch.distributed calls are the barrier and the
max-over-ranks of the timing.  Under torchrun the ranks are the launcher's; plain
`python bench.py --gpus N` starts the N ranks itself.  `--impl reference` times the
oracle (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "pairwise interactions/sec (fp32) at N=262,144 on 1 B200; % of FP32 peak"
UNIT = "interactions/s"
FLOP_PER_INTERACTION = 21          # 19 FMA-pipe flop + rsqrt + rcp
FLOP_CLASSIC = 20                  # the figure N-body papers usually quote per interaction, for comparability
FP32_LANES_PER_SM = 128
BENCH_CONFIG = 4                   # BASELINE.json configs[3]: the headline throughput config
L2_FLUSH_BYTES = 256 << 20         # > 126 MB L2
CPU_SAMPLE_ROWS = 32768            # cpu_baseline: rows x N fp64 pair evaluations (~10-60 core-seconds)
CPU_SAMPLE_ROWS_1T = 2048          # ... on one thread
# per_config: (timed steps, steps of the one-call "hot" run) for the configs that are not the headline
PER_CONFIG_STEPS = {1: (30, 100), 2: (30, 100), 3: (10, 20), 4: (5, 5), 5: (2, 2)}
REF_ROWS_PER_STEP = 2048           # --impl reference: rows x N per "step"


# ----------------------------------------------------------------------------- distributed glue
def dist_env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), \
        int(os.environ.get("WORLD_SIZE", "1"))


def dist_init(backend: str):
    import torch.distributed as dist
    rank, _, world = dist_env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def reduce_over_ranks(value: float, op: str = "max", device=None) -> float:
    """max / sum of a host scalar over all ranks (identity when not distributed)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return float(t.item())


# ----------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi samples of SM clock and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.proc.terminate()
        sm, smax, reasons, power = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                smax = float(f[1])
                if t0 - 0.05 <= ts <= t1 + 0.05:
                    sm.append(float(f[0]))
                    power.append(float(f[2]))
                    for nme, val in zip(names, f[3:7]):
                        if val.lower().startswith("active"):
                            reasons.add(nme)
            except ValueError:
                continue
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax, "samples": len(sm),
                "power_w_max": max(power) if power else None, "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------- reference arm
def run_reference(args):
    """The oracle as it stands on the host cores: each step = a(rows) for a seeded sample
    of REF_ROWS_PER_STEP elements against all N (rows x N fp64 pair evaluations)."""
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    import numpy as np
    import oracle
    from workloads import make_config, params_f32
    w = make_config(args.config)
    p = params_f32(w.params)
    m = w.posm[:, 3]
    rng = np.random.default_rng(4242)

    def one_step():
        rows = np.sort(rng.choice(w.n, REF_ROWS_PER_STEP, replace=False))
        oracle.accel(w.posm, w.vel, m, w.star, p["R_start"], p, rows=rows)

    for _ in range(max(args.warmup, 1)):
        one_step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        one_step()
    dt = time.perf_counter() - t0
    inter = float(REF_ROWS_PER_STEP) * w.n * args.steps
    value = inter / dt
    sample = f"{REF_ROWS_PER_STEP} seeded i-rows x all N={w.n} j per step (fp64, Eqs. 4-6)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w, p),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }), flush=True)
    return 0


def workload_config(w, p):
    """The `config` object of the JSON line: the same keys and values from both arms (the driver compares them)."""
    return {"workload": w.name, "n": w.n, "n1": w.meta["n1"], "n2": w.meta["n2"], "q": p["q"],
            "eps": p["eps"], "dt": p["dt"], "gamma": p["gamma"], "beta": p["beta"],
            "step": "KDK leapfrog: kick/drift + contact pass (Eqs. 5/6) + all-pairs gravity (Eq. 4) + reduce/kick",
            "l2": "own arm: flushed between timed steps (256 MiB fill); reference arm (CPU oracle): a bounded sample of "
                  "i-rows per step, no GPU",
            "parallelism": "replicas only"}


# ----------------------------------------------------------------------------- own arm
def kernel_source_sha():
    """sha256 over the kernel sources: a committed ncu capture names the sources it was taken from."""
    import hashlib
    h = hashlib.sha256()
    for f in ("nb_kernels.cuh", "nb_cells.cuh", "nb_fused.cuh", "nb_api.cu"):
        with open(os.path.join(ROOT, "paper_2303_12166_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def profile_traffic(kernel):
    """(dram bytes per launch, source) from the committed `ncu --set full` summary of THIS kernel instantiation built
    from THESE sources (profiles/r3_gravity_sym_kernel_full.md carries `kernel = ...`, `kernel_source_sha = ...` and
    `dram_bytes_per_launch = ...` lines), else (None, why): a capture of older sources is not this run's traffic."""
    path = os.path.join(ROOT, "profiles", "r3_gravity_sym_kernel_full.md")
    try:
        text = open(path).read()
    except OSError:
        return None, "no committed capture"
    if kernel.replace(" ", "") not in text.replace(" ", ""):
        return None, f"{os.path.basename(path)} is a capture of another kernel instantiation"
    sha = kernel_source_sha()
    if f"kernel_source_sha = {sha}" not in text:
        return None, f"{os.path.basename(path)} was captured from other kernel sources (now {sha}): re-capture"
    for line in text.splitlines():
        if line.startswith("dram_bytes_per_launch"):
            try:
                return float(line.split("=")[1].split()[0]), (f"profiles/{os.path.basename(path)} (ncu --set full of sources "
                                                               f"{sha}, committed; not measured by this run)")
            except (ValueError, IndexError):
                break
    return None, "no dram_bytes_per_launch line"


def executed_flop_per_interaction(symmetric, i_per_cta, n):
    """FP32 flop the gravity kernel EXECUTES per ordered interaction (FMA-pipe flop + one per MUFU), as opposed to
    the 21 that Eq. 4 needs.  One-sided: 20.5 + 1.5 (the shared reciprocal costs 1.5 multiplies, saves half a MUFU).
    Symmetric: one pair evaluation of 25 + 2 serves two interactions; the diagonal super-tiles (weight S/N) run
    one-sided, 19 + 2 each."""
    if not symmetric:
        return 22.0
    diag = min(1.0, i_per_cta / float(n))
    return (1.0 - diag) * 13.5 + diag * 21.0


def timed_steps(torch, sim, stream, flush, nsteps):
    """nsteps x nb_step(1), each bracketed by events on the launching stream, L2 flushed before each."""
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(nsteps)]
    for e0, e1 in ev:
        flush.fill_(1)                      # L2 flush between timed iterations (outside the events)
        e0.record(stream)
        sim.step(1)                         # a1-a6: kick/drift, all-pairs force, reduce + kick
        e1.record(stream)
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in ev]


def measure_config(torch, nb, idx, dev, stream, flush, peak_tflops, path):
    """One of the BASELINE configs that is not the headline: a few steps timed like the headline's."""
    from workloads import make_config, params_f32
    w = make_config(idx)
    p = params_f32(w.params)
    n = w.n
    sim = nb.Simulation(w.posm, w.vel, w.star, p, device=str(dev), stream=stream, force_path=path)
    nsteps, nhot = PER_CONFIG_STEPS[idx]
    for _ in range(3):
        sim.step(1)
    torch.cuda.synchronize(dev)
    ms = sorted(timed_steps(torch, sim, stream, flush, nsteps))
    mean = sum(ms) / len(ms)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream); sim.step(nhot); e1.record(stream)      # the same steps as ONE call, nothing flushed
    torch.cuda.synchronize(dev)
    hot = e0.elapsed_time(e1) / nhot
    reps = 10 if n <= 70000 else 3
    k_ms = nb.nb_time_force_kernel(sim.ctx, reps)
    c_ms = nb.nb_time_contact_pass(sim.ctx, reps)
    kernel = nb.nb_force_kernel_name(sim.ctx)
    info = nb.nb_get_launch_info(sim.ctx)
    fused = "fused" in kernel               # rows a2-a6 in one cooperative launch: there is no separate gravity kernel
    x = sim.posm.cpu()
    sim.close()
    assert bool(torch.isfinite(x).all())
    inter = float(n) * n
    return {"workload": w.name, "n": n, "kernel": kernel, "steps_timed": nsteps,
            "ms_per_step": mean, "ms_per_step_median": ms[len(ms) // 2], "ms_per_step_best": ms[0],
            "ms_per_step_hot": hot, "steps_per_s": 1e3 / mean, "steps_per_s_hot": 1e3 / hot,
            "interactions_per_s": inter / (mean * 1e-3), "interactions_per_s_hot": inter / (hot * 1e-3),
            "pct_of_fp32_peak": 100.0 * FLOP_PER_INTERACTION * inter / (mean * 1e-3) / (peak_tflops * 1e12),
            "pct_of_fp32_peak_20flop": 100.0 * FLOP_CLASSIC * inter / (mean * 1e-3) / (peak_tflops * 1e12),
            "gravity_kernel_ms": None if fused else k_ms, "contact_pass_ms": None if fused else c_ms,
            "fused_one_launch": fused, "launch": info,
            "note": "ms_per_step: nb_step(1) per event pair, L2 flushed before each; _hot: one nb_step(K) call / K"
                    + ("; one cooperative launch runs rows a2-a6 (launch: elements i per CTA, j segments, CTAs)" if fused else "")}


def cpu_baseline_leg(np, w, p, n):
    """The oracle as it stands on this box's host cores: all cores, one thread, and a full config-2 evaluation."""
    import ctypes
    import oracle
    from workloads import make_config, params_f32
    m = w.posm[:, 3]
    rows = np.sort(np.random.default_rng(99).choice(n, min(CPU_SAMPLE_ROWS, n), replace=False))
    oracle.accel(w.posm, w.vel, m, w.star, p["R_start"], p, rows=rows[:64])     # load + warm
    tt = time.perf_counter()
    oracle.accel(w.posm, w.vel, m, w.star, p["R_start"], p, rows=rows)
    dt = time.perf_counter() - tt
    cores = oracle.num_threads()
    out = {"value": float(len(rows)) * n / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
           "sample": f"{len(rows)} seeded i-rows x all N={n} j, one fp64 evaluation of Eqs. 4-6"}
    try:                                                             # the same on ONE thread
        gomp = ctypes.CDLL("libgomp.so.1")
        gomp.omp_set_num_threads(1)
        r1 = rows[:CPU_SAMPLE_ROWS_1T]
        tt = time.perf_counter()
        oracle.accel(w.posm, w.vel, m, w.star, p["R_start"], p, rows=r1)
        d1 = time.perf_counter() - tt
        gomp.omp_set_num_threads(cores)
        out["one_thread"] = {"value": float(len(r1)) * n / d1, "unit": UNIT, "cores": 1, "seconds": d1,
                             "sample": f"{len(r1)} of the same rows x all N={n} j"}
    except OSError:
        out["one_thread"] = None
    w2 = make_config(2)                                              # one FULL evaluation (BASELINE.md's plan)
    p2 = params_f32(w2.params)
    tt = time.perf_counter()
    oracle.accel(w2.posm, w2.vel, w2.posm[:, 3], w2.star, p2["R_start"], p2)
    d2 = time.perf_counter() - tt
    out["full_config2"] = {"value": float(w2.n) ** 2 / d2, "unit": UNIT, "cores": cores, "seconds": d2,
                           "sample": f"all {w2.n} rows x all {w2.n} j of {w2.name}"}
    return out


def run_own(args):
    import numpy as np
    import torch
    import paper_2303_12166_b200 as nb
    from workloads import params_f32

    rank, local_rank, world = dist_env()
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback "
                         "(use --impl reference for the oracle timing)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist_init("nccl")

    # replicas only: each rank integrates its own binary (same recipe, seed + rank)
    from workloads.configs import CONFIGS, make_binary
    kw = dict(CONFIGS[args.config])
    kw["seed"] = kw["seed"] + rank
    if args.scale != 1.0:                       # the same recipe at another size (crossover measurements; not a BASELINE config)
        kw["n1"] = max(1, int(round(kw["n1"] * args.scale)))
        kw["n2"] = max(1, int(round(kw["n2"] * args.scale)))
        kw["name"] = f"{kw['name']}_x{args.scale:g}"
    w = make_binary(**kw)
    p = params_f32(w.params)
    n = w.n
    stream = torch.cuda.current_stream(dev)
    path = {"auto": nb.NB_PATH_AUTO, "one-sided": nb.NB_PATH_ONE_SIDED, "symmetric": nb.NB_PATH_SYMMETRIC}[args.path]
    sim = nb.Simulation(w.posm, w.vel, w.star, p, device=f"cuda:{local_rank}", stream=stream, force_path=path)
    kernel = nb.nb_force_kernel_name(sim.ctx)
    symmetric = "sym" in kernel
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    info = nb.nb_get_launch_info(sim.ctx)

    for _ in range(args.warmup):
        sim.step(1)
    torch.cuda.synchronize(dev)

    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.12)
    barrier()
    torch.cuda.synchronize(dev)
    launches0 = nb.nb_launch_count(sim.ctx)
    t0 = time.time()
    ms_steps = timed_steps(torch, sim, stream, flush, args.steps)
    torch.cuda.synchronize(dev)
    barrier()
    t1 = time.time()
    launches = nb.nb_launch_count(sim.ctx) - launches0
    clocks = sampler.stop(t0, t1)
    ms_local = sum(ms_steps)
    ms_total = reduce_over_ranks(ms_local, "max", dev)
    value = float(n) * n * args.steps * world / (ms_total * 1e-3)
    ms_sorted = sorted(ms_steps)

    # ---- roofline of the dominant kernel (all-pairs gravity), timed alone on its stream
    k_ms = nb.nb_time_force_kernel(sim.ctx, max(3, min(args.steps, 10)))
    c_ms = nb.nb_time_contact_pass(sim.ctx, max(3, min(args.steps, 10)))
    props = torch.cuda.get_device_properties(dev)
    sms = props.multi_processor_count
    sm_max_mhz = clocks.get("sm_max_mhz") or 1965.0
    peak_tflops = sms * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    step_ms = ms_total / args.steps
    int_per_s = float(n) * n / (k_ms * 1e-3)
    executed = executed_flop_per_interaction(symmetric, info["i_per_cta"], n)
    achieved = executed * int_per_s / 1e12                       # what the ALUs did
    algorithmic = FLOP_PER_INTERACTION * int_per_s / 1e12        # what Eq. 4 needs for the N^2 ordered interactions delivered
    traffic, traffic_src = profile_traffic(kernel)
    # what the launched plan moves per force evaluation besides reading the N positions (ALU-bound: HBM is not the limit)
    T = info["j_splits"]                    # symmetric: super-tiles; one-sided: j splits
    ncontact = 1 if (p["gamma"] > 0 and n >= 8192) else 0
    if "chain" in kernel:                   # no slabs: every CTA adds 2 x S x 3 fp64 sums in place (read + write, L2-resident)
        traffic_model = {"mode": "chain", "slab_bytes_written": 0.0, "slabs": 0,
                         "acc64_read_modify_write_bytes": 48.0 * (T + 1) * n, "contact_slab_bytes": 16.0 * ncontact * n,
                         "note": "T(T+1)/2 CTAs x 2 tiles x S x 24 B read + written in turn order; the update kernel reads "
                                 "48 B/element of sums + the contact slab"}
    elif "fused" in kernel:
        traffic_model = {"mode": "fused", "slab_bytes_written": 0.0, "slabs": 0,
                         "note": "one cooperative launch: no partial sums in global memory; every CTA re-stages the N "
                                 "positions (16 B each) per step"}
    else:
        traffic_model = {"mode": "slabs", "slab_bytes_written": 16.0 * (T + ncontact) * n, "slabs": T + ncontact,
                         "note": "partial sums written once per launch and read once by nb_reduce_update_kernel"}
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": achieved / peak_tflops,
                "achieved_algorithmic": algorithmic, "frac_algorithmic": algorithmic / peak_tflops,
                "traffic": traffic, "traffic_source": traffic_src,
                "traffic_model": traffic_model,
                "kernel": kernel, "kernel_ms": k_ms,
                **({"kernel_ms_note": "n < 8192: the step runs in ONE cooperative launch (nb_fused_step_kernel); kernel_ms and "
                                      "contact_pass_ms time the stand-alone one-sided gravity kernel and index-order contact "
                                      "pass of the unfused path, for orientation only"} if "fused" in kernel else {}),
                "executed_flop_per_interaction": executed, "flop_per_interaction": FLOP_PER_INTERACTION,
                "pair_evaluations": "each unordered pair once (Newton's third law)" if symmetric
                                    else "every ordered pair",
                "note": "achieved/frac: FP32 flop the kernel EXECUTES (13.5 per ordered interaction when every unordered "
                        "pair is evaluated once) against the FP32 peak; *_algorithmic: the 21 flop per ordered interaction "
                        "of SURVEY 8(d) x N^2 delivered -- can reach 1 because half of them are never evaluated; "
                        "pipe occupancies (FMA, XU) are ncu counters, not derived here: profiles/r3_gravity_sym_kernel_full.md",
                "kernel_share_of_step": k_ms / step_ms,
                "contact_pass_ms": c_ms, "contact_pass_share_of_step": c_ms / step_ms,
                "interactions_per_s": int_per_s,
                "peak_source": f"derived: {sms} SMs x 128 FP32 lanes x 2 flop x "
                               f"{sm_max_mhz:.0f} MHz (clocks.max.sm); DESIGN.md 'Roofline'"}

    # ---- e2e: host (pinned) buffers through the C ABI, copies inside the timed region
    hp = torch.empty((n, 4), dtype=torch.float32).pin_memory()
    hv = torch.empty((n, 4), dtype=torch.float32).pin_memory()
    ha = torch.empty((n, 4), dtype=torch.float32).pin_memory()
    nb.nb_download_state(sim.ctx, hp, hv, ha)
    e2e_steps = max(3, min(args.steps, 10))
    for _ in range(2):
        nb.nb_upload_state(sim.ctx, hp, hv, ha); sim.step(1); nb.nb_download_state(sim.ctx, hp, hv, ha)
    barrier()
    torch.cuda.synchronize(dev)
    e2e_ms = 0.0
    for _ in range(e2e_steps):
        flush.fill_(1)
        torch.cuda.synchronize(dev)
        tt = time.perf_counter()
        nb.nb_upload_state(sim.ctx, hp, hv, ha)      # H2D x, v, a
        sim.step(1)
        nb.nb_download_state(sim.ctx, hp, hv, ha)    # D2H x, v, a (synchronises)
        e2e_ms += (time.perf_counter() - tt) * 1e3
    e2e_ms = reduce_over_ranks(e2e_ms, "max", dev)
    e2e_value = float(n) * n * e2e_steps * world / (e2e_ms * 1e-3)
    state_bytes = 3 * n * 16
    assert bool(torch.isfinite(hp).all()) and bool(torch.isfinite(hv).all())
    sim.close()

    # ---- the other BASELINE configs, and the oracle on this box's host cores (rank 0, N=1 only)
    per_config, cpu_baseline = None, None
    if rank == 0 and world == 1:
        if not args.no_per_config:
            per_config = [measure_config(torch, nb, idx, dev, stream, flush, peak_tflops, path)
                          for idx in sorted(PER_CONFIG_STEPS) if idx != args.config]
        if not args.no_cpu_baseline:
            cpu_baseline = cpu_baseline_leg(np, w, p, n)

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": workload_config(w, p),
            "launch": info,
            "ms_per_step_median": ms_sorted[len(ms_sorted) // 2], "ms_per_step_best": ms_sorted[0],
            "steps_per_s": 1e3 / step_ms,
            "pct_of_fp32_peak": 100.0 * FLOP_PER_INTERACTION * value / world / (peak_tflops * 1e12),
            "pct_of_fp32_peak_20flop": 100.0 * FLOP_CLASSIC * value / world / (peak_tflops * 1e12),
            "roofline": roofline,
            "per_config": per_config,
            "cpu_baseline": cpu_baseline,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": state_bytes,
                    "d2h_bytes_per_step": state_bytes, "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps},
            "gpu_launches": int(launches),
            "clocks": clocks,
        }), flush=True)
    try:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()
    except Exception:
        pass
    return 0


# ----------------------------------------------------------------------------- N replicas from one command
def spawn_ranks(args, argv, script=None):
    """`python bench.py --gpus N` without a launcher: start the N ranks (one process per GPU, RANK / LOCAL_RANK /
    WORLD_SIZE / MASTER_* set as torchrun would), relay rank 0's line, fail if any rank fails.  `script`: the file
    the ranks run (this one)."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    procs = []
    for r in range(args.gpus):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(args.gpus), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, script or os.path.abspath(__file__)] + list(argv), env=env,
                                      stdout=subprocess.PIPE if r == 0 else subprocess.DEVNULL, text=True))
    out, _ = procs[0].communicate()
    rcs = [procs[0].returncode] + [pr.wait() for pr in procs[1:]]
    sys.stdout.write(out)
    sys.stdout.flush()
    return max(abs(rc) for rc in rcs)


def main(argv=None):
    argv = sys.argv[1:] if argv is None else list(argv)
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, choices=[1, 2, 3, 4, 5], default=BENCH_CONFIG,
                    help="BASELINE config timed as the headline (default 4, the one the metric is quoted on)")
    ap.add_argument("--scale", type=float, default=1.0,
                    help="scale the element counts of --config (same recipe and seed): for crossover measurements only")
    ap.add_argument("--path", choices=["auto", "one-sided", "symmetric"], default="auto",
                    help="row-a2 kernel (nb_set_force_path); auto = the library's choice")
    ap.add_argument("--impl", choices=["own", "reference"], default="own")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg")
    ap.add_argument("--no-per-config", action="store_true", help="skip the other four configs")
    args = ap.parse_args(argv)
    if args.steps < 1 or args.warmup < 0 or args.gpus < 1:
        ap.error("--steps >= 1, --warmup >= 0, --gpus >= 1")
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args, argv)
    return run_own(args)


if __name__ == "__main__":
    sys.exit(main())

#!/usr/bin/env python
"""bench.py -- headline measurement: pairwise interactions/s (fp32) at N = 262,144 on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

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
  cpu_baseline  the fp64 oracle (oracle/, as it stands) on the box's host cores, on a
             seeded sample of i-rows against all N elements.

The path does not shard (north_star: one GPU, no collectives): with --gpus N > 1
every rank runs an independent replica ("replicas only", weak scaling), no
data-path collective; the only torch.distributed calls are the barrier and the
max-over-ranks of the timing.  `--impl reference` times the oracle (rank 0 only).
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
FP32_LANES_PER_SM = 128
BENCH_CONFIG = 4                   # BASELINE.json configs[3]: the headline throughput config
L2_FLUSH_BYTES = 256 << 20         # > 126 MB L2
CPU_SAMPLE_ROWS = 32768            # cpu_baseline: rows x N fp64 pair evaluations (~10-60 core-seconds)
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
    w = make_config(BENCH_CONFIG)
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
        "config": {"workload": w.name, "n": w.n, "note": "CPU oracle, bounded sample of the same workload"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }), flush=True)
    return 0


# ----------------------------------------------------------------------------- own arm
def ncu_traffic_bytes(kernel):
    """dram bytes per force-kernel launch from the committed ncu --set full summary of `kernel`, or None."""
    name = "r1_gravity_sym_kernel_full.md" if "sym" in kernel else "r1_gravity_kernel_full.md"
    path = os.path.join(ROOT, "profiles", name)
    try:
        for line in open(path):
            if line.startswith("dram_bytes_per_launch"):
                return float(line.split("=")[1].split()[0])
    except (OSError, ValueError, IndexError):
        pass
    return None


def run_own(args):
    import numpy as np
    import torch
    import paper_2303_12166_b200 as nb
    from workloads import make_config, params_f32

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback "
                         "(use --impl reference for the oracle timing)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist_init("nccl")

    # replicas only: each rank integrates its own binary (same recipe, seed + rank)
    from workloads.configs import CONFIGS, make_binary
    kw = dict(CONFIGS[BENCH_CONFIG])
    kw["seed"] = kw["seed"] + rank
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

    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.12)
    barrier()
    torch.cuda.synchronize(dev)
    launches0 = nb.nb_launch_count(sim.ctx)
    t0 = time.time()
    for e0, e1 in ev:
        flush.fill_(1)                      # L2 flush between timed iterations (outside the events)
        e0.record(stream)
        sim.step(1)                         # a1-a6: kick/drift, all-pairs force, reduce + kick
        e1.record(stream)
    torch.cuda.synchronize(dev)
    barrier()
    t1 = time.time()
    launches = nb.nb_launch_count(sim.ctx) - launches0
    clocks = sampler.stop(t0, t1)
    ms_local = sum(a.elapsed_time(b) for a, b in ev)
    ms_total = reduce_over_ranks(ms_local, "max", dev)
    value = float(n) * n * args.steps * world / (ms_total * 1e-3)

    # ---- roofline of the dominant kernel (all-pairs gravity), timed alone on its stream
    k_ms = nb.nb_time_force_kernel(sim.ctx, max(3, min(args.steps, 10)))
    c_ms = nb.nb_time_contact_pass(sim.ctx, max(3, min(args.steps, 10)))
    props = torch.cuda.get_device_properties(dev)
    sm_max_mhz = clocks.get("sm_max_mhz") or 1965.0
    peak_tflops = props.multi_processor_count * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    achieved = FLOP_PER_INTERACTION * float(n) * n / (k_ms * 1e-3) / 1e12
    step_ms = ms_total / args.steps
    # What the kernel executes per ordered interaction (FMA-pipe flop + one per MUFU), as opposed to the
    # 21 flop Eq. 4 itself needs (the convention `achieved` uses).  One-sided kernel: 20.5 + 1.5 (Montgomery
    # costs 1.5 more multiplies and saves half a MUFU).  Symmetric kernel: one pair evaluation of 25 + 2
    # serves two interactions (the super-tiles on the diagonal run one-sided, 19 + 2 each: weight S/N).
    if symmetric:
        diag = info["i_per_cta"] / float(n)
        executed = (1.0 - diag) * 13.5 + diag * 21.0
    else:
        executed = 22.0
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": achieved / peak_tflops, "traffic": ncu_traffic_bytes(kernel),
                "kernel": kernel, "kernel_ms": k_ms,
                "executed_flop_per_interaction": executed,
                "frac_executed": achieved / peak_tflops * executed / FLOP_PER_INTERACTION,
                "pair_evaluations": "each unordered pair once (Newton's third law)" if symmetric
                                    else "every ordered pair",
                "note": "achieved/frac use the ALGORITHMIC 21 flop per ordered interaction (SURVEY 8d); the symmetric "
                        "kernel evaluates half of them, so frac can reach 1 -- frac_executed is what the ALUs did",
                "kernel_share_of_step": k_ms / step_ms,
                "contact_pass_ms": c_ms, "contact_pass_share_of_step": c_ms / step_ms,
                "interactions_per_s": float(n) * n / (k_ms * 1e-3),
                "flop_per_interaction": FLOP_PER_INTERACTION,
                "peak_source": f"derived: {props.multi_processor_count} SMs x 128 FP32 lanes x 2 flop x "
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

    # ---- the oracle, as it stands, on this box's host cores (rank 0, N=1 only)
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        rows = np.sort(np.random.default_rng(99).choice(n, CPU_SAMPLE_ROWS, replace=False))
        oracle.accel(w.posm, w.vel, w.posm[:, 3], w.star, p["R_start"], p, rows=rows[:64])     # load + warm
        tt = time.perf_counter()
        oracle.accel(w.posm, w.vel, w.posm[:, 3], w.star, p["R_start"], p, rows=rows)
        dt = time.perf_counter() - tt
        cpu_baseline = {"value": float(len(rows)) * n / dt, "unit": UNIT, "cores": oracle.num_threads(),
                        "kind": "oracle", "seconds": dt,
                        "sample": f"{len(rows)} seeded i-rows x all N={n} j, one fp64 evaluation of Eqs. 4-6"}

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "n": n, "n1": w.meta["n1"], "n2": w.meta["n2"], "q": p["q"],
                       "eps": p["eps"], "dt": p["dt"], "gamma": p["gamma"], "beta": p["beta"],
                       "step": "KDK leapfrog: kick/drift + contact pass (Eqs. 5/6) + all-pairs gravity (Eq. 4) + reduce/kick",
                       "l2": "flushed between timed steps (256 MiB fill)", "parallelism": "replicas only",
                       "launch": info},
            "steps_per_s": 1e3 / step_ms,
            "pct_of_fp32_peak": 100.0 * FLOP_PER_INTERACTION * value / world / (peak_tflops * 1e12),
            "roofline": roofline,
            "cpu_baseline": cpu_baseline,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": state_bytes,
                    "d2h_bytes_per_step": state_bytes, "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps},
            "gpu_launches": int(launches),
            "clocks": clocks,
        }), flush=True)
    sim.close()
    try:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()
    except Exception:
        pass
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--path", choices=["auto", "one-sided", "symmetric"], default="auto",
                    help="row-a2 kernel (nb_set_force_path); auto = the library's choice")
    ap.add_argument("--impl", choices=["own", "reference"], default="own")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg")
    args = ap.parse_args(argv)
    if args.steps < 1 or args.warmup < 0:
        ap.error("--steps >= 1, --warmup >= 0")
    return run_reference(args) if args.impl == "reference" else run_own(args)


if __name__ == "__main__":
    sys.exit(main())

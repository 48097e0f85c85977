"""One rank of bench.py's timing path with the GPU taken out (gloo, a sleep for a step): lets the CPU-only test
tests/test_bench_host.py drive bench.spawn_ranks() through the rank spawning, the barriers and the max-over-ranks.
Test scaffolding: it uses bench.py's own dist_env / dist_init / barrier / reduce_over_ranks and prints a line of the
same shape."""
import argparse
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=4)
    ap.add_argument("--warmup", type=int, default=0)
    args = ap.parse_args()
    rank, _, world = bench.dist_env()
    if world != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}")
    bench.dist_init("gloo")
    bench.barrier()
    ms_local = 0.0
    for _ in range(args.steps):
        tt = time.perf_counter()
        time.sleep(0.002 * (1 + rank))                 # rank 1 is the slower one: the max must pick it
        ms_local += (time.perf_counter() - tt) * 1e3
    bench.barrier()
    ms_total = bench.reduce_over_ranks(ms_local, "max")
    units = bench.reduce_over_ranks(1000.0 * args.steps, "sum")
    if rank == 0:
        print(json.dumps({"impl": "stub", "metric": bench.METRIC, "value": units / (ms_total * 1e-3), "unit": bench.UNIT,
                          "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_total / args.steps,
                          "scaling": "weak", "config": {"workload": "stub", "parallelism": "replicas only"}}), flush=True)
    import torch.distributed as dist
    if dist.is_initialized():
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

"""Phase times of nb_fused_step_kernel (n < 8,192: whole leapfrog steps in one cooperative launch), a development aid.

    python -m paper_2303_12166_b200.build --prof          # libnb_prof.so: the library with -DNB_FUSED_PROF
    python -m paper_2303_12166_b200.fused_phases [scale]  # on a B200; config 1 at `scale` (default 1: N = 2,048)

The profiling build stamps %globaltimer (thread 0 of every CTA) at the phase boundaries of the kernel; this script
runs nb_step(4) as one launch and prints, per stamp, the earliest / median / latest CTA (microseconds from the first
stamp; the timer's resolution is ~0.26 us).  S = positions staged, G = gravity loop done, F = contact terms done,
U = reduction + kick + drift done (before the grid barrier), sync = after the grid barrier.
"""
from __future__ import annotations

import ctypes as C
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
PROF_LIB = os.path.join(HERE, "libnb_prof.so")
sys.path.insert(0, os.path.dirname(HERE))


def main(scale: float = 1.0, K: int = 4) -> int:
    import numpy as np
    import torch
    import paper_2303_12166_b200 as nb
    from workloads import make_config, params_f32

    if not os.path.exists(PROF_LIB):
        raise SystemExit("build it first: python -m paper_2303_12166_b200.build --prof")
    nb.LIB_PATH = PROF_LIB                 # (`python -m` imports the package before this module: the library is not loaded yet)
    w = make_config(1, scale=scale)
    sim = nb.Simulation(w.posm, w.vel, w.star, params_f32(w.params), device="cuda:0")
    if nb.nb_force_kernel_name(sim.ctx) != "nb_fused_step_kernel":
        raise SystemExit(f"n = {w.n}: not on the fused path")
    sim.step(3); sim.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); sim.step(K); e1.record(); torch.cuda.synchronize()
    info = nb.nb_get_launch_info(sim.ctx)
    print(f"n = {w.n}: nb_step({K}) = one launch, {e0.elapsed_time(e1) * 1e3:.2f} us by CUDA events; {info}")
    buf = np.zeros((512, 64), dtype=np.int64)
    fn = nb.lib().nb_debug_fused_prof
    fn.argtypes = [C.c_void_p]
    if fn(buf.ctypes.data) != 0:
        raise SystemExit("nb_debug_fused_prof failed")
    names = ["start", "open", "open-sync"]
    for e in range(K):
        names += [f"S{e}", f"G{e}", f"F{e}"]
        if e + 1 < K:
            names += [f"U{e}", f"U{e}-sync"]
    t = buf[:info["force_ctas"], :len(names)].astype(np.float64)
    t -= t[:, 0].min()
    prev = 0.0
    for k, nm in enumerate(names):
        col = t[:, k] / 1e3
        print(f"{nm:10s} min {col.min():7.2f}  median {np.median(col):7.2f}  max {col.max():7.2f} us   (+{col.max() - prev:5.2f})")
        prev = col.max()
    sim.close()
    return 0


if __name__ == "__main__":
    sys.exit(main(float(sys.argv[1]) if len(sys.argv) > 1 else 1.0))

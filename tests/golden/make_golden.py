"""Write the stored expected values under tests/golden/ -- calls ONLY oracle/ and workloads/.

  python tests/golden/make_golden.py 3 4      # configs to (re)generate

For BASELINE configs whose 10-step fp64 trajectory is too slow to recompute inside
the GPU test run (config 3: 10 x 4.3e9 pairs, config 4: 10 x 6.9e10 pairs), the oracle's
positions and velocities after 10 leapfrog steps are stored for a seeded sample of
elements, together with a hash of the float32 inputs they belong to.  Nothing here
comes from the CUDA path.
"""
import hashlib
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from workloads import make_config, params_f32  # noqa: E402

NSTEPS = 10
NSAMPLE = 1024
HERE = os.path.dirname(os.path.abspath(__file__))


def input_hash(w) -> str:
    h = hashlib.sha256()
    h.update(np.ascontiguousarray(w.posm).tobytes())
    h.update(np.ascontiguousarray(w.vel).tobytes())
    return h.hexdigest()


def sample_rows(n: int, idx: int) -> np.ndarray:
    return np.sort(np.random.default_rng(1000 + idx).choice(n, NSAMPLE, replace=False))


def main(idxs):
    for idx in idxs:
        w = make_config(idx)
        p = params_f32(w.params)
        t = time.time()
        s = oracle.Sim(w.posm, w.vel, w.star, p)
        s.step(NSTEPS)
        rows = sample_rows(w.n, idx)
        out = np.concatenate([rows[:, None].astype(np.float64), s.x[rows], s.v[rows]], axis=1)
        path = os.path.join(HERE, f"config{idx}_step{NSTEPS}_sample.txt")
        hdr = (f"oracle state after {NSTEPS} KDK steps (PAPER.md:89, reading A7), BASELINE config {idx}, N={w.n}\n"
               f"written by tests/golden/make_golden.py from oracle/ only; inputs sha256={input_hash(w)}\n"
               f"R after {NSTEPS} steps = {s.radii().tolist()}\n"
               f"columns: element index, x, y, z, vx, vy, vz")
        np.savetxt(path, out, fmt=["%d"] + ["%.17g"] * 6, header=hdr)
        print(f"config {idx}: {path}  ({time.time() - t:.0f} s, {oracle.num_threads()} threads)", flush=True)


if __name__ == "__main__":
    main([int(a) for a in sys.argv[1:]] or [3, 4])

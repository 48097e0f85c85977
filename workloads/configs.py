"""Synthetic binary-star element sets shaped like the paper's runs.

The paper builds each star out of N elements of
equal mass and a per-star common element radius, and puts two such stars in
orbit.  It prints no N, dt, gamma, beta, eps or radii, so
the five workloads below are the ones BASELINE.json names, completed by the
recipe of SURVEY.md section 8(d) / DESIGN.md "Input recipe".

Nothing here evaluates the method: positions, velocities and masses are drawn
from numpy's PCG64 in float64 and rounded ONCE to float32; those float32 arrays
are the single source for both the GPU library and the fp64 oracle.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, Optional

import numpy as np

PHI_PACK = 0.64          # element packing fraction -> ~5 contacts per element
GAMMA = 400.0            # repulsion strength  (400 G M1^2 / R1^5 with G=M1=R1=1)
BETA = 0.5               # diverging reduction fraction
V_DEAD_FRAC = 1.0e-4     # reading A5: dead band, in units of sqrt(G (M1+M2)/a)
TAU_S_FRAC = 1.0e-5      # reading A6: width of the either-branch-accepted band
NOISE_FRAC = 0.05        # velocity noise sigma, in units of omega*a (configs 2-5)

# Config 3 ramps the donor's element radius so that the star "fills the Roche
# lobe": factor = r_L(1/q; k=0.6) * a / R_1 for q=0.4, a=2.5, R_1=1.  The value is
# a literal here (this module may not implement Eq. 3); tests check it against
# both the oracle's and the library's Eq. 3.
CONFIG3_RAMP_FACTOR = 1.149683


@dataclasses.dataclass
class Workload:
    name: str
    posm: np.ndarray      # float32 [N,4]  x, y, z, m
    vel: np.ndarray       # float32 [N,4]  vx, vy, vz, 0
    star: np.ndarray      # int32   [N]    0 for star 1, 1 for star 2 (star 1 first)
    params: Dict[str, object]   # G, eps, dt, q, gamma, beta, R_start, R_end, n_ramp, v_dead, tau_s, lens_mode
    meta: Dict[str, object]     # a (separation), omega, n1, n2, nsteps, seed, M1, M2

    @property
    def n(self) -> int:
        return int(self.posm.shape[0])


def _uniform_sphere(rng: np.random.Generator, n: int, radius: float) -> np.ndarray:
    g = rng.standard_normal((n, 3))
    g /= np.linalg.norm(g, axis=1, keepdims=True)
    u = rng.random(n)
    return g * (radius * np.cbrt(u))[:, None]


def _plummer(rng: np.random.Generator, n: int, b: float) -> np.ndarray:
    g = rng.standard_normal((n, 3))
    g /= np.linalg.norm(g, axis=1, keepdims=True)
    u = rng.random(n)
    r = b / np.sqrt(u ** (-2.0 / 3.0) - 1.0)
    bad = r > 10.0 * b
    while bad.any():                      # redraw the tail beyond 10 b
        u2 = rng.random(int(bad.sum()))
        r[bad] = b / np.sqrt(u2 ** (-2.0 / 3.0) - 1.0)
        bad = r > 10.0 * b
    return g * r[:, None]


def make_binary(*, name: str, seed: int, n1: int, n2: int, shape: str,
                radius1: float, radius2: float, q: float, a: float, eps: float,
                dt: float, nsteps: int, mass_sigma: float = 0.0,
                noise_frac: float = NOISE_FRAC, ramp_factor1: float = 1.0,
                ramp_factor2: float = 1.0, n_ramp: int = 0, gamma: float = GAMMA, beta: float = BETA,
                G: float = 1.0) -> Workload:
    """Two stars of elements on a circular orbit with synchronous rotation.

    Draw order (fixed): star-1 positions, star-2 positions, masses, velocity noise.
    """
    rng = np.random.default_rng(seed)
    M1, M2 = 1.0, float(q)
    draw = _uniform_sphere if shape == "uniform" else _plummer
    p1 = draw(rng, n1, radius1)
    p2 = draw(rng, n2, radius2)
    c1 = np.array([-a * q / (1.0 + q), 0.0, 0.0])
    c2 = np.array([a / (1.0 + q), 0.0, 0.0])
    x = np.concatenate([p1 + c1, p2 + c2], axis=0)

    if mass_sigma > 0.0:
        w1 = rng.lognormal(0.0, mass_sigma, n1)
        w2 = rng.lognormal(0.0, mass_sigma, n2)
        m = np.concatenate([M1 * w1 / w1.sum(), M2 * w2 / w2.sum()])
    else:
        m = np.concatenate([np.full(n1, M1 / n1), np.full(n2, M2 / max(n2, 1))])

    omega = math.sqrt(G * (M1 + M2) / a ** 3)          # Keplerian, softening ignored
    v = np.stack([-omega * x[:, 1], omega * x[:, 0], np.zeros(len(x))], axis=1)
    if noise_frac > 0.0:
        v = v + rng.standard_normal(v.shape) * (noise_frac * omega * a)

    posm = np.zeros((n1 + n2, 4), dtype=np.float32)
    posm[:, :3] = x.astype(np.float32)
    posm[:, 3] = m.astype(np.float32)
    vel = np.zeros((n1 + n2, 4), dtype=np.float32)
    vel[:, :3] = v.astype(np.float32)
    star = np.concatenate([np.zeros(n1, np.int32), np.ones(n2, np.int32)])

    # reading A3: no two elements may coincide after rounding to float32
    if n1 + n2 > 1:
        uniq = np.unique(posm[:, :3].view([("", np.float32)] * 3)).shape[0]
        assert uniq == n1 + n2, "duplicate element positions after float32 rounding"

    re1 = radius1 * (PHI_PACK / n1) ** (1.0 / 3.0)
    re2 = radius2 * (PHI_PACK / max(n2, 1)) ** (1.0 / 3.0)
    vscale = math.sqrt(G * (M1 + M2) / a)
    params = dict(G=G, eps=eps, dt=dt, q=q, gamma=gamma, beta=beta,
                  R_start=(re1, re2), R_end=(re1 * ramp_factor1, re2 * ramp_factor2),
                  n_ramp=int(n_ramp), v_dead=V_DEAD_FRAC * vscale,
                  tau_s=TAU_S_FRAC * vscale, lens_mode=0)
    meta = dict(a=a, omega=omega, n1=n1, n2=n2, nsteps=nsteps, seed=seed,
                M1=M1, M2=M2, shape=shape, radius=(radius1, radius2))
    return Workload(name, posm, vel, star, params, meta)


# BASELINE.json "configs", in order; values not fixed there follow SURVEY.md 8(d).
CONFIGS = {
    1: dict(name="config1_N2048", seed=0, n1=1024, n2=1024, shape="uniform",
            radius1=1.0, radius2=0.6, q=0.5, a=3.0, eps=0.01, dt=1e-3, nsteps=10,
            noise_frac=0.0),
    2: dict(name="config2_N16384", seed=1, n1=8192, n2=8192, shape="plummer",
            radius1=1.0, radius2=0.8, q=0.8, a=4.0, eps=0.005, dt=1e-3, nsteps=0,
            mass_sigma=0.1),
    3: dict(name="config3_N65536", seed=2, n1=49152, n2=16384, shape="uniform",
            radius1=1.0, radius2=0.5, q=0.4, a=2.5, eps=0.003, dt=5e-4, nsteps=1000,
            ramp_factor1=CONFIG3_RAMP_FACTOR, n_ramp=1000),
    4: dict(name="config4_N262144", seed=3, n1=131072, n2=131072, shape="uniform",
            radius1=1.0, radius2=0.6 ** (1.0 / 3.0), q=0.6, a=3.0, eps=0.002,
            dt=2e-4, nsteps=100),
    5: dict(name="config5_N1048576", seed=4, n1=786432, n2=262144, shape="uniform",
            radius1=1.0, radius2=0.4, q=0.3, a=3.0, eps=0.001, dt=2e-4, nsteps=0),
}


def make_config(idx: int, scale: Optional[float] = None) -> Workload:
    """Build BASELINE config `idx` (1..5).  `scale` (<1) shrinks both stars'
    element counts by that factor (same recipe, same seed) for quick tests."""
    kw = dict(CONFIGS[idx])
    if scale is not None:
        kw["n1"] = max(1, int(round(kw["n1"] * scale)))
        kw["n2"] = max(1, int(round(kw["n2"] * scale)))
        kw["name"] = f"{kw['name']}_x{scale:g}"
    return make_binary(**kw)


def params_f32(params: Dict[str, object]) -> Dict[str, object]:
    """The model parameters as the library holds them: every real rounded once to
    float32 (returned as Python floats).  Feed THIS dict to both sides so that
    a comparison never sees parameter rounding."""
    f = lambda v: float(np.float32(v))
    out = dict(params)
    for k in ("G", "eps", "dt", "q", "gamma", "beta", "v_dead"):
        if k in out:
            out[k] = f(out[k])
    for k in ("R_start", "R_end"):
        if k in out:
            out[k] = tuple(f(v) for v in out[k])
    return out


# the paper's three kinds of run (Fig. 5), as parameter sets of the
# same recipe.  The paper prints no numbers for them; sizes are kept small enough for a full oracle run.
SCENARIOS = {
    # I-III: main-sequence donor filling its lobe + compact accretor (white dwarf): few, small elements
    "ms_white_dwarf": dict(name="scenario_ms_white_dwarf", seed=11, n1=16384, n2=1024, shape="uniform",
                           radius1=1.0, radius2=0.08, q=0.6, a=2.6, eps=0.004, dt=5e-4, nsteps=200,
                           ramp_factor1=1.12, n_ramp=200),
    # IV-VI: non-conservative case B, two main-sequence stars, BOTH expanding
    "case_b_both_expand": dict(name="scenario_case_b", seed=12, n1=8192, n2=8192, shape="uniform",
                               radius1=1.0, radius2=0.9, q=0.8, a=2.4, eps=0.005, dt=5e-4, nsteps=200,
                               ramp_factor1=1.2, ramp_factor2=1.2, n_ramp=200),
    # VII-IX: red giant (large, tenuous) + main-sequence star, Algol-like
    "algol_red_giant": dict(name="scenario_algol", seed=13, n1=12288, n2=8192, shape="uniform",
                            radius1=1.5, radius2=0.5, q=0.5, a=3.4, eps=0.005, dt=1e-3, nsteps=200,
                            ramp_factor1=1.1, n_ramp=100),
}


def make_scenario(key: str, scale: Optional[float] = None) -> Workload:
    kw = dict(SCENARIOS[key])
    if scale is not None:
        kw["n1"] = max(1, int(round(kw["n1"] * scale)))
        kw["n2"] = max(1, int(round(kw["n2"] * scale)))
    return make_binary(**kw)

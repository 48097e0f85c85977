"""fp64 CPU oracle for the all-pairs binary-star element model -- TEST INFRASTRUCTURE.

Thin ctypes marshalling around oracle/nb_oracle.c (see its header for the
passages of the paper each routine restates and the readings taken).  Inputs
are the float32 workload arrays promoted to double.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this package; it imports nothing from paper_2303_12166_b200.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional, Sequence, Tuple

import numpy as np

from .build import build as _build

_LIB = None


class _Params(C.Structure):
    _fields_ = [("G", C.c_double), ("eps", C.c_double), ("gamma", C.c_double),
                ("beta", C.c_double), ("v_dead", C.c_double), ("tau_s", C.c_double),
                ("lens_mode", C.c_int32), ("pad_", C.c_int32)]


def load():
    global _LIB
    if _LIB is None:
        lib = C.CDLL(_build())
        dp, ip, lp = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int64)
        lib.orc_lens_volume.restype = C.c_double
        lib.orc_lens_volume.argtypes = [C.c_double, C.c_double, C.c_int32]
        lib.orc_rep_potential.restype = C.c_double
        lib.orc_rep_potential.argtypes = [C.c_double, C.c_double, C.c_double]
        lib.orc_roche_lobe_radius.restype = C.c_double
        lib.orc_roche_lobe_radius.argtypes = [C.c_double, C.c_double]
        lib.orc_l1_distance.restype = C.c_double
        lib.orc_l1_distance.argtypes = [C.c_double]
        lib.orc_accel.restype = None
        lib.orc_accel.argtypes = [C.c_int64, dp, dp, dp, ip, dp, C.POINTER(_Params),
                                  C.c_int64, lp, dp, dp, dp]
        lib.orc_radii.restype = None
        lib.orc_radii.argtypes = [C.c_int64, dp, dp, C.c_int64, dp]
        lib.orc_step.restype = None
        lib.orc_step.argtypes = [C.c_int64, dp, dp, dp, ip, C.POINTER(_Params), dp, dp,
                                 C.c_int64, C.c_double, C.c_int64, C.c_int64, dp, ip]
        lib.orc_energy.restype = None
        lib.orc_energy.argtypes = [C.c_int64, dp, dp, dp, ip, dp, C.POINTER(_Params), dp, dp]
        _LIB = lib
    return _LIB


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _params(p: Dict[str, object]) -> _Params:
    return _Params(float(p["G"]), float(p["eps"]), float(p.get("gamma", 0.0)),
                   float(p.get("beta", 1.0)), float(p.get("v_dead", 0.0)),
                   float(p.get("tau_s", 0.0)), int(p.get("lens_mode", 0)), 0)


def _f64(a, cols: Optional[int] = None) -> np.ndarray:
    a = np.asarray(a)
    if cols is not None:
        a = a[:, :cols]
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    """OpenMP threads the oracle will use (OMP_NUM_THREADS, else all cores)."""
    env = os.environ.get("OMP_NUM_THREADS")
    return int(env) if env else (os.cpu_count() or 1)


def lens_volume(r: float, R: float, lens_mode: int = 0) -> float:
    return load().orc_lens_volume(float(r), float(R), int(lens_mode))


def rep_potential(r: float, R: float, gamma: float) -> float:
    return load().orc_rep_potential(float(r), float(R), float(gamma))


def roche_lobe_radius(mass_ratio: float, k: float = 0.6) -> float:
    return load().orc_roche_lobe_radius(float(mass_ratio), float(k))


def l1_distance(q: float) -> float:
    return load().orc_l1_distance(float(q))


def radii(nstep: int, R_start: Sequence[float], R_end: Sequence[float], n_ramp: int) -> np.ndarray:
    rs, re, out = _f64(R_start), _f64(R_end), np.zeros(2)
    load().orc_radii(int(nstep), _dp(rs), _dp(re), int(n_ramp), _dp(out))
    return out


def accel(pos, vel, mass, star, R, params, rows=None, want_diag: bool = False):
    """a_i for i in rows (all if None).  pos/vel: [n,>=3], mass [n], star [n], R [2].
    Returns a [nrows,3] float64, and (kappa, delta) too if want_diag."""
    x, v, m = _f64(pos, 3), _f64(vel, 3), _f64(mass)
    st = np.ascontiguousarray(star, dtype=np.int32)
    Rr = _f64(R)
    n = x.shape[0]
    if rows is None:
        nr, rp = n, None
    else:
        rows = np.ascontiguousarray(rows, dtype=np.int64)
        nr, rp = rows.shape[0], rows.ctypes.data_as(C.POINTER(C.c_int64))
    a = np.zeros((nr, 3))
    kap = np.zeros(nr) if want_diag else None
    dl = np.zeros(nr) if want_diag else None
    prm = _params(params)
    load().orc_accel(n, _dp(x), _dp(v), _dp(m), st.ctypes.data_as(C.POINTER(C.c_int32)),
                     _dp(Rr), C.byref(prm), nr, rp, _dp(a),
                     _dp(kap) if want_diag else None, _dp(dl) if want_diag else None)
    return (a, kap, dl) if want_diag else a


class Sim:
    """Oracle-side state for multi-step runs: x, v (float64, promoted from the
    float32 inputs), the step count n and the cached a(x_n) (reading A7)."""

    def __init__(self, posm, vel, star, params):
        self.x = _f64(posm, 3).copy()
        self.v = _f64(vel, 3).copy()
        self.m = _f64(np.asarray(posm)[:, 3]).copy()
        self.star = np.ascontiguousarray(star, dtype=np.int32)
        self.params = dict(params)
        self.n = 0
        self.acc = np.zeros_like(self.x)
        self.have_acc = C.c_int32(0)

    def radii(self) -> np.ndarray:
        p = self.params
        return radii(self.n, p["R_start"], p["R_end"], int(p.get("n_ramp", 0)))

    def accel(self, rows=None, want_diag=False):
        return accel(self.x, self.v, self.m, self.star, self.radii(), self.params,
                     rows=rows, want_diag=want_diag)

    def step(self, k: int = 1) -> None:
        p = self.params
        prm = _params(p)
        rs, re = _f64(p["R_start"]), _f64(p["R_end"])
        load().orc_step(self.x.shape[0], _dp(self.x), _dp(self.v), _dp(self.m),
                        self.star.ctypes.data_as(C.POINTER(C.c_int32)), C.byref(prm),
                        _dp(rs), _dp(re), int(p.get("n_ramp", 0)), float(p["dt"]),
                        int(self.n), int(k), _dp(self.acc), C.byref(self.have_acc))
        self.n += int(k)

    def energy(self) -> Dict[str, object]:
        if not self.have_acc.value:
            self.acc[:] = self.accel()
            self.have_acc = C.c_int32(1)
        out = np.zeros(12)
        prm = _params(self.params)
        R = self.radii()
        load().orc_energy(self.x.shape[0], _dp(self.x), _dp(self.v), _dp(self.m),
                          self.star.ctypes.data_as(C.POINTER(C.c_int32)), _dp(R),
                          C.byref(prm), _dp(self.acc), _dp(out))
        return dict(KE=out[0], Ug=out[1], Urep=out[2], E=out[3], P=out[4:7].copy(),
                    L=out[7:10].copy(), Fnet=out[10], step=self.n)

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
        lib.orc_contact_list.restype = None
        lib.orc_contact_list.argtypes = [C.c_int64, dp, dp, ip, dp, C.c_int64, lp, C.c_int64, lp, lp, dp, dp]
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


def contact_list(pos, vel, star, R, rows=None, cap: int = 64):
    """Contact pairs (r < R_i + R_j, A2/A3) of the elements in rows (all if None).
    Returns count [nrows] (all pairs of the row), and j [nrows,cap] (-1 beyond count), r, rdot
    [nrows,cap] (NaN beyond count) holding the first `cap` pairs of every row in j order."""
    x, v = _f64(pos, 3), _f64(vel, 3)
    st = np.ascontiguousarray(star, dtype=np.int32)
    Rr = _f64(R)
    n = x.shape[0]
    lp = C.POINTER(C.c_int64)
    if rows is None:
        nr, rp = n, None
    else:
        rows = np.ascontiguousarray(rows, dtype=np.int64)
        nr, rp = rows.shape[0], rows.ctypes.data_as(lp)
    count = np.zeros(nr, np.int64)
    jj = np.full((nr, cap), -1, np.int64)
    rr = np.full((nr, cap), np.nan)
    rd = np.full((nr, cap), np.nan)
    load().orc_contact_list(n, _dp(x), _dp(v), st.ctypes.data_as(C.POINTER(C.c_int32)), _dp(Rr), nr, rp,
                            int(cap), count.ctypes.data_as(lp), jj.ctypes.data_as(lp), _dp(rr), _dp(rd))
    return count, jj, rr, rd


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


# ---------------------------------------------------------------------------------------------
# NEXT rows of SURVEY.md 8(f) -- plain numpy, fp64 (same rules: test infrastructure only).

def _sim_relax(self, k: int, kappa: float) -> None:
    """f2, star construction / relaxation (the elements are put together and the star
    is left to settle; the paper gives no procedure -- DESIGN.md reading A17): k leapfrog steps, each
    followed by v <- (1 - kappa dt) v, the factor clamped at 0."""
    f = max(0.0, 1.0 - float(kappa) * float(self.params["dt"]))
    for _ in range(int(k)):
        self.step(1)
        self.v *= f


Sim.relax = _sim_relax

TRANSFER_FIELDS = ("M0", "M1", "a", "d0", "rL0", "rL1", "Mcross0", "Mcross1", "Min0", "Min1", "Mout0", "Mout1")


def transfer_diagnostics(pos, vel, mass, star, k: float = 0.6, band: float = 0.0) -> Dict[str, object]:
    """f3, mass transfer through L1 (reading A18).

    Centres X_s, V_s and masses M_s of the two stars by membership; separation a = |X_1 - X_0| and
    unit vector e; the L1 plane at distance d0 from X_0 along e (force balance, l1_distance); the
    lobe radii rL_s = a * Eq. 3 with the star's own mass in the numerator.  Per star s (o = other):
      Mcross_s  mass of its elements on the far side of the L1 plane,
      Min_s     mass of its elements inside the other star's lobe sphere |x - X_o| < rL_o,
      Ldisk_s   their angular momentum about the other star, sum m (x - X_o) x (v - V_o),
      Mout_s    mass of its elements outside both lobe spheres.
    `band` > 0 also returns 'ambiguous': the mass of elements within `band` of any of the decision
    surfaces (either answer is acceptable for them in a comparison)."""
    x, v, m = _f64(pos, 3), _f64(vel, 3), _f64(mass)
    st = np.asarray(star).astype(np.int64)
    M = np.array([m[st == s].sum() for s in (0, 1)])
    X = np.array([(m[st == s, None] * x[st == s]).sum(0) / M[s] if M[s] > 0 else np.zeros(3) for s in (0, 1)])
    V = np.array([(m[st == s, None] * v[st == s]).sum(0) / M[s] if M[s] > 0 else np.zeros(3) for s in (0, 1)])
    out: Dict[str, object] = dict(M0=M[0], M1=M[1], X=X, V=V)
    if not (M[0] > 0 and M[1] > 0):
        out.update(a=0.0, d0=0.0, rL0=0.0, rL1=0.0, Mcross0=0.0, Mcross1=0.0, Min0=0.0, Min1=0.0,
                   Mout0=0.0, Mout1=0.0, Ldisk=np.zeros((2, 3)), ambiguous=0.0)
        return out
    d = X[1] - X[0]
    a = float(np.sqrt(d @ d))
    e = d / a
    if M[1] <= M[0]:
        d0 = a * l1_distance(M[1] / M[0])                 # star 0 is the primary m1 of PAPER.md:28
    else:
        d0 = a * (1.0 - l1_distance(M[0] / M[1]))
    rL = np.array([a * roche_lobe_radius(M[0] / M[1], k), a * roche_lobe_radius(M[1] / M[0], k)])
    u = (x - X[0]) @ e
    r0 = np.linalg.norm(x - X[0], axis=1)
    r1 = np.linalg.norm(x - X[1], axis=1)
    rs = [r0, r1]
    Mcross, Min, Mout, Ld = np.zeros(2), np.zeros(2), np.zeros(2), np.zeros((2, 3))
    for s in (0, 1):
        o = 1 - s
        mine = st == s
        crossed = (u > d0) if s == 0 else (u < d0)
        Mcross[s] = m[mine & crossed].sum()
        inside = mine & (rs[o] < rL[o])
        Min[s] = m[inside].sum()
        Ld[s] = (m[inside, None] * np.cross(x[inside] - X[o], v[inside] - V[o])).sum(0)
        Mout[s] = m[mine & (r0 > rL[0]) & (r1 > rL[1])].sum()
    amb = 0.0
    if band > 0:
        near = (np.abs(u - d0) < band) | (np.abs(r0 - rL[0]) < band) | (np.abs(r1 - rL[1]) < band)
        amb = float(m[near].sum())
    out.update(a=a, d0=d0, rL0=rL[0], rL1=rL[1], Mcross0=Mcross[0], Mcross1=Mcross[1], Min0=Min[0],
               Min1=Min[1], Mout0=Mout[0], Mout1=Mout[1], Ldisk=Ld, ambiguous=amb)
    return out


def splat(pos, star, centre, half_width: float, axis_u: int, axis_v: int, W: int, H: int) -> np.ndarray:
    """f4, headless point splat replacing the paper's OpenGL viewer (the paper states no
    shader math -- DESIGN.md reading A19): orthographic projection on coordinate axes (axis_u, axis_v),
    pixel (floor((x_u - c_u) s + W/2), floor((x_v - c_v) s + H/2)) with s = W / (2 half_width), all in
    float32 with one rounding per operation (the pixel index is an integer decided by floating point:
    both sides take it in the kernel's precision); image[star][py][px] counts the elements, uint32."""
    p = np.asarray(pos)[:, :3].astype(np.float32)
    st = np.asarray(star).astype(np.int64)
    c = np.asarray(centre, dtype=np.float32)
    s = np.float32(np.float32(W) / np.float32(np.float32(2.0) * np.float32(half_width)))
    fu = (p[:, axis_u] - c[axis_u]).astype(np.float32) * s
    fu = (fu.astype(np.float32) + np.float32(0.5 * W)).astype(np.float32)
    fv = (p[:, axis_v] - c[axis_v]).astype(np.float32) * s
    fv = (fv.astype(np.float32) + np.float32(0.5 * H)).astype(np.float32)
    pu, pv = np.floor(fu), np.floor(fv)
    ok = (pu >= 0) & (pu < W) & (pv >= 0) & (pv < H)
    img = np.zeros((2, H, W), dtype=np.uint32)
    np.add.at(img, (st[ok], pv[ok].astype(np.int64), pu[ok].astype(np.int64)), 1)
    return img


def splat_exact(pos, star, centre, half_width: float, axis_u: int, axis_v: int, W: int, H: int):
    """f4 by its DEFINITION (reading A19), in float64 on the float32 inputs: element i lands in pixel
    (floor(t_u), floor(t_v)), t_u = (x_u - c_u) W/(2 half_width) + W/2, t_v = (x_v - c_v) W/(2 half_width) + H/2
    (square pixels), counted in image[star][py][px] if inside the window.

    A float32 evaluation of t (four roundings: the difference, the scale W/(2 hw), the product, the sum) is off
    by at most 2^-24 (3 |t - W/2| + |t|) <= 3 W 2^-24 pixels inside the window, so an element whose t lies
    within that band of an integer may legitimately land in the neighbouring pixel (or across the window's
    edge).  Returns (image uint32 [2,H,W], ambiguous uint32 [2,H+2,W+2]): ambiguous counts those elements in
    their exact pixel, on a grid padded by one pixel on every side (index +1) so that elements just outside
    the window are kept too."""
    p = np.asarray(pos)[:, :3].astype(np.float32).astype(np.float64)
    st = np.asarray(star).astype(np.int64)
    c = np.asarray(centre, dtype=np.float32).astype(np.float64)
    s = float(W) / (2.0 * float(np.float32(half_width)))
    tu = (p[:, axis_u] - c[axis_u]) * s + 0.5 * W
    tv = (p[:, axis_v] - c[axis_v]) * s + 0.5 * H
    pu, pv = np.floor(tu), np.floor(tv)
    ok = (pu >= 0) & (pu < W) & (pv >= 0) & (pv < H)
    img = np.zeros((2, H, W), dtype=np.uint32)
    np.add.at(img, (st[ok], pv[ok].astype(np.int64), pu[ok].astype(np.int64)), 1)
    band_u, band_v = 3.0 * W * 2.0 ** -24, 3.0 * max(W, H) * 2.0 ** -24
    near = (np.abs(tu - np.rint(tu)) <= band_u) | (np.abs(tv - np.rint(tv)) <= band_v)
    keep = near & (pu >= -1) & (pu <= W) & (pv >= -1) & (pv <= H)
    amb = np.zeros((2, H + 2, W + 2), dtype=np.uint32)
    np.add.at(amb, (st[keep], pv[keep].astype(np.int64) + 1, pu[keep].astype(np.int64) + 1), 1)
    return img, amb

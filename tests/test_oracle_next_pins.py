"""Pins of the oracle routines of the NEXT rows: relaxation (f2), mass-transfer
diagnostics (f3), point splat (f4).  Same rule as test_oracle_pins.py: closed forms with literal
numbers, symmetries, brute force -- never the oracle's own formula re-typed."""
import math

import numpy as np
import pytest

import oracle
from workloads import make_config, params_f32

P0 = dict(G=1.0, eps=0.0, gamma=0.0, beta=1.0, v_dead=0.0, tau_s=0.0, lens_mode=0, dt=0.1,
          R_start=(0.0, 0.0), R_end=(0.0, 0.0), n_ramp=0)


# ------------------------------------------------------------------ f2: relaxation
def test_relax_force_free_closed_form():
    # G = 0: no forces.  f = 1 - kappa dt = 0.8.  The velocity during step k is v0 f^k, so
    # v_n = v0 f^n and x_n = x0 + dt v0 (1 - f^n)/(1 - f):  n = 5 -> v = 0.32768 v0,
    # x = x0 + 0.1 * (1 - 0.32768)/0.2 v0 = x0 + 0.33616 v0
    s = oracle.Sim(np.array([[1.0, 2.0, 3.0, 1.0]]), np.array([[2.0, -1.0, 0.5, 0.0]]), [0], dict(P0, G=0.0))
    s.relax(5, 2.0)
    assert s.v[0] == pytest.approx(np.array([2.0, -1.0, 0.5]) * 0.32768, rel=1e-14)
    assert s.x[0] == pytest.approx(np.array([1.0, 2.0, 3.0]) + 0.33616 * np.array([2.0, -1.0, 0.5]), rel=1e-14)
    assert s.n == 5


def test_relax_without_damping_is_the_plain_step_and_clamp():
    w = make_config(1, scale=0.125)
    p = params_f32(w.params)
    a, b = oracle.Sim(w.posm, w.vel, w.star, p), oracle.Sim(w.posm, w.vel, w.star, p)
    a.relax(4, 0.0); b.step(4)
    assert np.array_equal(a.x, b.x) and np.array_equal(a.v, b.v)
    c = oracle.Sim(w.posm, w.vel, w.star, p)
    c.relax(2, 10.0 / p["dt"])                      # kappa dt >= 1: the factor is clamped at 0
    assert (c.v == 0).all()


def test_relax_drains_energy_and_keeps_momentum_direction():
    # a bound two-body orbit, point masses: with damping E decreases at every step, P -> f^n P, and the
    # separation shrinks; with beta = 1 and no contact nothing else dissipates
    x = np.array([[-0.5, 0, 0, 1.0], [0.5, 0, 0, 1.0]])
    v = np.array([[0.1, -0.7, 0, 0], [0.1, 0.7, 0, 0]])     # net momentum (0.2, 0, 0)
    s = oracle.Sim(x, v, [0, 1], dict(P0, dt=1e-3, eps=1e-3))
    E = [s.energy()["E"]]
    for _ in range(20):
        s.relax(50, 0.5)
        E.append(s.energy()["E"])
    assert all(b < a for a, b in zip(E, E[1:]))
    f = (1 - 0.5e-3) ** 1000
    assert s.energy()["P"] == pytest.approx([0.2 * f, 0, 0], abs=1e-12)
    assert np.linalg.norm(s.x[1] - s.x[0]) < 1.0


# ------------------------------------------------------------------ f3: transfer diagnostics
def _tracer_system(q=0.5, a=2.0, tm=1e-12):
    """Two heavy elements (masses 1 and q, separation a on the x axis) + hand-placed tracers."""
    x0, x1 = -a * q / (1 + q), a / (1 + q)
    d0 = 0.570752 * a                                # P9: L1 distance from the primary, q = 0.5
    rL1 = 0.320788 * a                               # P8: Eq. 3 (k = 0.6) at q = 0.5
    pos = [[x0, 0, 0], [x1, 0, 0],
           [x0 + d0 + 0.01, 0.3, 0],                 # donor tracer just beyond the L1 plane, outside lobe 1
           [x0 + d0 - 0.01, -0.2, 0.1],              # donor tracer just short of it
           [x1, 0.5 * rL1, 0],                       # donor tracer on a circular orbit inside lobe 1
           [x0, 0, 5.0]]                             # donor tracer far away: outside both lobes
    vel = [[0, 0, 0], [0, 0.25, 0], [0, 0, 0], [0, 0, 0], [-0.4, 0.25, 0], [0, 0, 0]]
    m = [1.0, q, tm, tm, tm, tm]
    star = [0, 1, 0, 0, 0, 0]
    return np.array(pos), np.array(vel), np.array(m), np.array(star), (x0, x1, d0, rL1)


def test_transfer_diagnostics_hand_placed_tracers():
    pos, vel, m, star, (x0, x1, d0, rL1) = _tracer_system()
    d = oracle.transfer_diagnostics(pos, vel, m, star)
    assert d["M0"] == pytest.approx(1.0, abs=1e-11) and d["M1"] == 0.5
    assert d["a"] == pytest.approx(2.0, abs=1e-10)
    assert d["d0"] == pytest.approx(d0, abs=2e-6) and d["rL1"] == pytest.approx(rL1, abs=2e-6)
    assert d["rL0"] == pytest.approx(0.44004 * 2.0, abs=1e-4)      # Eq. 3 at mass ratio 2, worked by hand
    assert d["Mcross0"] == pytest.approx(2e-12, rel=1e-9)          # the tracer beyond the plane + the orbiting one
    assert d["Mcross1"] == 0.0
    assert d["Min0"] == pytest.approx(1e-12, rel=1e-9) and d["Min1"] == 0.0
    # outside both lobe SPHERES (rL0 = 0.880, rL1 = 0.642; they do not reach the L1 plane at 1.1415): the far
    # tracer and both tracers next to the plane (1.15 and 0.90 / 0.91 from the two centres)
    assert d["Mout0"] == pytest.approx(3e-12, rel=1e-9)
    # orbiting tracer: r = (0, rL1/2, 0), v - V1 = (-0.4, 0, 0): L = m r x v = m (0, 0, 0.4 rL1/2)
    assert d["Ldisk"][0] == pytest.approx([0, 0, 1e-12 * 0.4 * 0.5 * rL1], abs=1e-18)
    assert (d["Ldisk"][1] == 0).all()


def test_transfer_diagnostics_heavier_second_star_uses_the_mirrored_l1():
    # masses (0.5, 1): star 1 is the primary; L1 sits 0.570752 a from IT, i.e. d0 = (1 - 0.570752) a
    pos = np.array([[0.0, 0, 0], [3.0, 0, 0]])
    d = oracle.transfer_diagnostics(pos, np.zeros((2, 3)), [0.5, 1.0], [0, 1])
    assert d["d0"] == pytest.approx((1 - 0.570752) * 3.0, abs=3e-6)
    assert d["rL0"] == pytest.approx(0.320788 * 3.0, abs=3e-6) and d["rL1"] == pytest.approx(0.44004 * 3.0, abs=2e-4)


def test_transfer_diagnostics_invariances_and_label_swap():
    w = make_config(3, scale=1 / 32)
    rng = np.random.default_rng(7)
    x = w.posm[:, :3].astype(np.float64)
    x[: w.n // 20] += [1.2, 0.1, 0.0]                  # push some donor elements over to the accretor
    v, m, st = w.vel[:, :3].astype(np.float64), w.posm[:, 3].astype(np.float64), w.star
    d = oracle.transfer_diagnostics(x, v, m, st)
    assert d["Mcross0"] > 0 and d["Min0"] > 0 and d["Mout0"] >= 0
    Q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] = -Q[:, 0]
    shift, boost = np.array([3.0, -2.0, 0.7]), np.array([0.3, 0.1, -0.2])
    d2 = oracle.transfer_diagnostics(x @ Q.T + shift, v @ Q.T + boost, m, st)
    for k in oracle.TRANSFER_FIELDS:
        assert d2[k] == pytest.approx(d[k], rel=1e-10, abs=1e-13), k
    assert d2["Ldisk"] == pytest.approx(d["Ldisk"] @ Q.T, rel=1e-9, abs=1e-13)
    # swap the labels (and the storage order): every per-star output swaps
    order = np.concatenate([np.where(st == 1)[0], np.where(st == 0)[0]])
    d3 = oracle.transfer_diagnostics(x[order], v[order], m[order], 1 - st[order])
    for k0, k1 in (("M0", "M1"), ("rL0", "rL1"), ("Mcross0", "Mcross1"), ("Min0", "Min1"), ("Mout0", "Mout1")):
        assert d3[k0] == pytest.approx(d[k1], rel=1e-12, abs=1e-15) and d3[k1] == pytest.approx(d[k0], rel=1e-12, abs=1e-15)
    assert d3["d0"] == pytest.approx(d["a"] - d["d0"], rel=1e-12)
    assert d3["Ldisk"][::-1] == pytest.approx(d["Ldisk"], rel=1e-10, abs=1e-15)


def test_transfer_diagnostics_brute_force_tiny():
    rng = np.random.default_rng(1)
    n = 12
    x, v = rng.standard_normal((n, 3)), rng.standard_normal((n, 3))
    x[6:, 0] += 3.0
    m = rng.uniform(0.5, 1.5, n)
    st = np.array([0] * 6 + [1] * 6)
    d = oracle.transfer_diagnostics(x, v, m, st)
    M = [sum(m[i] for i in range(n) if st[i] == s) for s in (0, 1)]
    X = [sum(m[i] * x[i] for i in range(n) if st[i] == s) / M[s] for s in (0, 1)]
    V = [sum(m[i] * v[i] for i in range(n) if st[i] == s) / M[s] for s in (0, 1)]
    a = math.dist(X[0], X[1])
    e = (X[1] - X[0]) / a
    mc, mi, mo = [0.0, 0.0], [0.0, 0.0], [0.0, 0.0]
    L = np.zeros((2, 3))
    for i in range(n):
        s = st[i]; o = 1 - s
        u = float((x[i] - X[0]) @ e)
        if (s == 0 and u > d["d0"]) or (s == 1 and u < d["d0"]):
            mc[s] += m[i]
        if math.dist(x[i], X[o]) < d["rL" + str(o)]:
            mi[s] += m[i]
            L[s] += m[i] * np.cross(x[i] - X[o], v[i] - V[o])
        if math.dist(x[i], X[0]) > d["rL0"] and math.dist(x[i], X[1]) > d["rL1"]:
            mo[s] += m[i]
    assert [d["Mcross0"], d["Mcross1"]] == pytest.approx(mc) and [d["Min0"], d["Min1"]] == pytest.approx(mi)
    assert [d["Mout0"], d["Mout1"]] == pytest.approx(mo) and d["Ldisk"] == pytest.approx(L)
    assert d["a"] == pytest.approx(a)


def test_transfer_diagnostics_detached_config_has_no_transfer():
    w = make_config(1)
    d = oracle.transfer_diagnostics(w.posm, w.vel, w.posm[:, 3], w.star)
    assert d["Mcross0"] == d["Mcross1"] == d["Min0"] == d["Min1"] == d["Mout0"] == d["Mout1"] == 0.0


# ------------------------------------------------------------------ f4: point splat
def test_splat_hand_example():
    # window centred at (1, 2), half width 2, 8 x 8 pixels of 0.5: x in [-1, 3), y in [0, 4)
    pos = np.array([[-1.0, 0.0, 9.0], [2.9, 3.9, 0.0], [1.0, 2.0, 0.0], [1.2, 2.4, 5.0], [3.0, 2.0, 0.0], [0.0, -0.1, 0.0]])
    star = np.array([0, 0, 1, 1, 1, 0])
    img = oracle.splat(pos, star, [1.0, 2.0, 0.0], 2.0, 0, 1, 8, 8)
    assert img.dtype == np.uint32 and img.shape == (2, 8, 8)
    assert img[0, 0, 0] == 1 and img[0, 7, 7] == 1 and img[1, 4, 4] == 2
    assert img.sum() == 4                             # x = 3.0 and y = -0.1 fall outside


def test_splat_matches_histogram_away_from_pixel_edges_and_shifts_exactly():
    rng = np.random.default_rng(3)
    W = H = 64
    pos = rng.uniform(-1.9, 1.9, (5000, 3))
    frac = (pos[:, [0, 2]] + 2.0) * 16.0
    keep = (np.abs(frac - np.round(frac)) > 1e-3).all(1)   # not within 1e-3 pixel of an edge
    pos = pos[keep].astype(np.float32)
    star = (rng.uniform(size=len(pos)) < 0.3).astype(np.int32)
    img = oracle.splat(pos, star, [0.0, 0.0, 0.0], 2.0, 0, 2, W, H)
    for s in (0, 1):
        h, _, _ = np.histogram2d(pos[star == s, 2].astype(np.float64), pos[star == s, 0].astype(np.float64),
                                 bins=[H, W], range=[[-2, 2], [-2, 2]])
        assert np.array_equal(img[s], h.astype(np.uint32))
    assert img.sum() == len(pos)
    # moving the window by exactly one pixel (0.0625, a power of two) moves the image by one pixel
    img2 = oracle.splat(pos, star, [0.0625, 0.0, 0.0], 2.0, 0, 2, W, H)
    assert np.array_equal(img2[:, :, :-1], img[:, :, 1:])


def test_splat_exact_hand_example_and_ambiguous_band():
    # the same window as test_splat_hand_example: 8 x 8 pixels of 0.5, x in [-1, 3), y in [0, 4)
    pos = np.array([[-1.0, 0.0, 9.0], [2.9, 3.9, 0.0], [1.0, 2.0, 0.0], [1.2, 2.4, 5.0], [3.0, 2.0, 0.0], [0.0, -0.1, 0.0]])
    star = np.array([0, 0, 1, 1, 1, 0])
    img, amb = oracle.splat_exact(pos, star, [1.0, 2.0, 0.0], 2.0, 0, 1, 8, 8)
    assert img.dtype == np.uint32 and img.shape == (2, 8, 8) and amb.shape == (2, 10, 10)
    assert img[0, 0, 0] == 1 and img[0, 7, 7] == 1 and img[1, 4, 4] == 2 and img.sum() == 4
    # elements exactly on a pixel edge are ambiguous: (-1, 0) -> corner of pixel (0,0); (1, 2) -> corner of (4,4);
    # (3, 2) -> one pixel right of the window (padded index 8+1); (0, -0.1) -> x on the edge of column 2, one row
    # below the window (padded row 0); the other two are well inside their pixels
    assert amb[0, 0 + 1, 0 + 1] == 1 and amb[1, 4 + 1, 4 + 1] == 1 and amb[1, 4 + 1, 8 + 1] == 1
    assert amb[0, -1 + 1, 2 + 1] == 1 and amb.sum() == 4
    # the band is 3 W 2^-24 pixels: 8 pixels -> 1.43e-6 pixel = 7.2e-7 length units here
    eps_in, eps_out = 0.5 * 1.0e-6, 0.5 * 2.0e-6
    pos = np.array([[0.5 + eps_in, 1.25, 0.0], [0.5 - eps_in, 1.25, 0.0], [0.5 + eps_out, 1.25, 0.0]])
    img, amb = oracle.splat_exact(pos, np.zeros(3, int), [1.0, 2.0, 0.0], 2.0, 0, 1, 8, 8)
    assert img[0, 2, 3] == 2 and img[0, 2, 2] == 1             # decided exactly, whichever side
    assert amb[0, 2 + 1, 3 + 1] == 1 and amb[0, 2 + 1, 2 + 1] == 1 and amb.sum() == 2


def test_splat_exact_is_the_histogram_and_the_float32_recipe_agrees_off_the_band():
    rng = np.random.default_rng(8)
    W, H = 96, 64
    pos = rng.uniform(-2.2, 2.2, (20000, 3)).astype(np.float32)
    star = (rng.uniform(size=len(pos)) < 0.4).astype(np.int32)
    c, hw = [0.125, 0.0, -0.25], 2.0
    img, amb = oracle.splat_exact(pos, star, c, hw, 0, 2, W, H)
    half_v = hw * H / W
    for s in (0, 1):
        q = pos[star == s].astype(np.float64)
        # numpy's own binning of the same window (its last bin is closed on the right: no point sits there)
        h, _, _ = np.histogram2d(q[:, 2], q[:, 0], bins=[H, W],
                                 range=[[c[2] - half_v, c[2] + half_v], [c[0] - hw, c[0] + hw]])
        assert np.array_equal(img[s], h.astype(np.uint32))
    assert 0 < img.sum() < len(pos)
    # the float32 recipe (what the kernel computes) differs from the definition only through ambiguous elements:
    # per pixel, by no more than the ambiguous elements of its 3 x 3 neighbourhood
    f32 = oracle.splat(pos, star, c, hw, 0, 2, W, H).astype(np.int64)
    nb_amb = sum(amb[:, 1 + dy:1 + dy + H, 1 + dx:1 + dx + W].astype(np.int64) for dy in (-1, 0, 1) for dx in (-1, 0, 1))
    assert (np.abs(f32 - img.astype(np.int64)) <= nb_amb).all()
    # with points placed on purpose a hair around pixel edges the two may differ, but only inside that allowance
    edge = np.zeros((4000, 3), np.float32)
    k = rng.integers(0, W, 4000)
    edge[:, 0] = (c[0] - hw + k * (2 * hw / W) + rng.uniform(-3e-7, 3e-7, 4000)).astype(np.float32)
    edge[:, 2] = rng.uniform(-1.0, 1.0, 4000).astype(np.float32)
    img, amb = oracle.splat_exact(edge, np.zeros(4000, int), c, hw, 0, 2, W, H)
    f32 = oracle.splat(edge, np.zeros(4000, int), c, hw, 0, 2, W, H).astype(np.int64)
    nb_amb = sum(amb[:, 1 + dy:1 + dy + H, 1 + dx:1 + dx + W].astype(np.int64) for dy in (-1, 0, 1) for dx in (-1, 0, 1))
    assert amb.sum() > 1000 and (np.abs(f32 - img.astype(np.int64)) <= nb_amb).all()
    assert abs(int(f32.sum()) - int(img.sum())) <= int(amb[:, :, [0, 1, W, W + 1]].sum() + amb[:, [0, 1, H, H + 1], :].sum())

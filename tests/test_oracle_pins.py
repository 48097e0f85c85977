"""Pins of the fp64 oracle against what the paper and the mathematics fix.

None of these re-types the oracle's formula: each is a closed form with literal
hand-computed numbers, a symmetry, a conservation law, an independent numerical
integration, or a textbook special case.
"""
import math

import numpy as np
import pytest

import oracle
from workloads import make_binary, make_config

P0 = dict(G=1.0, eps=0.0, gamma=0.0, beta=1.0, v_dead=0.0, tau_s=0.0, lens_mode=0)


def _acc(x, m, *, v=None, star=None, R=(0.0, 0.0), **kw):
    x = np.asarray(x, float)
    v = np.zeros_like(x) if v is None else np.asarray(v, float)
    star = np.zeros(len(x), np.int32) if star is None else star
    return oracle.accel(x, v, np.asarray(m, float), star, R, dict(P0, **kw))


# ---------------------------------------------------------------- P1: Eq. 4
def test_p1_two_body_hand_sum():
    # m1=1 at 0, m2=2 at x=3, eps=1: a1 = 2/(3+1)^2 = 0.125 toward +x,
    # a2 = 1/16 = 0.0625 toward -x  (Eq. 4 divided by m_i)
    a = _acc([[0, 0, 0], [3, 0, 0]], [1, 2], eps=1.0)
    assert a[0] == pytest.approx([0.125, 0, 0], abs=1e-15)
    assert a[1] == pytest.approx([-0.0625, 0, 0], abs=1e-15)


def test_p1_collinear_unequal_masses_literal():
    # x = 0,1,3  m = 1,2,4  G=2 eps=0.5 ; numbers worked by hand:
    # a0 = 2*2/1.5^2 + 2*4/3.5^2 = 1.777777778 + 0.653061224 = 2.430839002
    # a1 = -2*1/1.5^2 + 2*4/2.5^2 = -0.888888889 + 1.28 = 0.391111111
    # a2 = -(2*1/3.5^2 + 2*2/2.5^2) = -(0.163265306 + 0.64) = -0.803265306
    a = _acc([[0, 0, 0], [1, 0, 0], [3, 0, 0]], [1, 2, 4], G=2.0, eps=0.5)
    assert a[:, 0] == pytest.approx([2.430839002, 0.391111111, -0.803265306], abs=2e-9)
    assert np.abs(a[:, 1:]).max() == 0.0


def test_p1_equilateral_and_tetrahedron_closed_forms():
    L, eps, m, G = 2.0, 0.3, 0.7, 1.3
    tri = np.array([[0, 0, 0], [L, 0, 0], [L / 2, L * math.sqrt(3) / 2, 0]])
    a = _acc(tri, [m] * 3, G=G, eps=eps)
    c = tri.mean(0)
    mag = math.sqrt(3) * G * m / (L + eps) ** 2       # 2 cos30 = sqrt 3
    for i in range(3):
        u = (c - tri[i]) / np.linalg.norm(c - tri[i])
        assert a[i] == pytest.approx(mag * u, abs=1e-14)
    s = L / math.sqrt(8.0)                            # tetrahedron of edge L
    tet = s * np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], float)
    a = _acc(tet, [m] * 4, G=G, eps=eps)
    mag = math.sqrt(6) * G * m / (L + eps) ** 2       # 3 * sqrt(2/3)
    for i in range(4):
        u = -tet[i] / np.linalg.norm(tet[i])
        assert a[i] == pytest.approx(mag * u, abs=1e-14)


def test_softening_is_r_plus_eps_squared_not_plummer():
    # r=1, eps=0.5: (r+eps)^2 = 2.25 -> 0.4444...; Plummer (r^2+eps^2)^{3/2}*... would give 0.7155
    a = _acc([[0, 0, 0], [0, 1, 0]], [1, 1], eps=0.5)
    assert a[0, 1] == pytest.approx(1.0 / 2.25, abs=1e-15)


def test_always_attractive_without_repulsion():
    rng = np.random.default_rng(5)
    x = rng.standard_normal((2, 3))
    a = _acc(x, [1.0, 3.0], eps=0.01)
    d = x[1] - x[0]
    assert np.dot(a[0], d) > 0 and np.dot(a[1], -d) > 0


# ------------------------------------------------- P2: displaced (lens) volume
def test_p2_lens_volume_closed_form_limits():
    R = 0.7
    assert oracle.lens_volume(0.0, R) == pytest.approx(4.0 / 3.0 * math.pi * R ** 3, rel=1e-15)
    assert abs(oracle.lens_volume(2 * R, R)) < 1e-15
    h = 1e-6
    slope = (oracle.lens_volume(2 * R, R) - oracle.lens_volume(2 * R - h, R)) / h
    assert abs(slope) < 1e-5                                  # touches zero with zero slope
    for r in (0.0, 0.35, 0.7, 1.05, 1.4):                    # factored form of the same cubic
        fact = math.pi * (2 * R - r) ** 2 * (4 * R + r) / 12.0
        assert oracle.lens_volume(r, R) == pytest.approx(fact, abs=1e-15)
    # the literal printed r^2/12 form does NOT vanish at first contact (reading A1)
    assert oracle.lens_volume(2.0, 1.0, 1) == pytest.approx(-math.pi / 3.0, rel=1e-12)


def test_p2_lens_volume_is_sphere_sphere_overlap_monte_carlo():
    # "proportional to the displaced volume": overlap of two radius-R balls
    rng = np.random.default_rng(11)
    R, n = 1.0, 2_000_000
    g = rng.standard_normal((n, 3))
    g /= np.linalg.norm(g, axis=1, keepdims=True)
    p = g * np.cbrt(rng.random(n))[:, None] * R              # uniform in ball 1 at origin
    for r in (0.4, 1.0, 1.6):
        inside = np.linalg.norm(p - np.array([r, 0, 0]), axis=1) < R
        vol = inside.mean() * 4.0 / 3.0 * math.pi * R ** 3
        assert oracle.lens_volume(r, R) == pytest.approx(vol, rel=0, abs=6e-3)


def test_rep_potential_is_integral_of_force():
    R, g = 0.5, 7.0
    assert abs(oracle.rep_potential(2 * R, R, g)) < 1e-15
    for r in (0.1, 0.4, 0.8):
        h = 1e-5
        dU = (oracle.rep_potential(r + h, R, g) - oracle.rep_potential(r - h, R, g)) / (2 * h)
        assert -dU == pytest.approx(g * oracle.lens_volume(r, R), rel=1e-8)


# ------------------------------------------------------ P3 / A5: Eqs. 5 and 6
def test_contact_hand_numbers_and_branch():
    # G=0 isolates the repulsion. R=1, r=1: V = pi(4/3 - 1 + 1/12) = 5 pi/12 = 1.308996939
    # gamma=3, m_i=2, m_j=5: converging a_i = 3*1.308996939/2 = 1.963495408 away from j,
    # a_j = 3*1.308996939/5 = 0.785398163 away from i; diverging (beta=0.25) a quarter of that.
    x = [[0, 0, 0], [1, 0, 0]]
    kw = dict(G=0.0, gamma=3.0, beta=0.25, R=(1.0, 1.0))
    a = _acc(x, [2, 5], v=[[0.1, 0, 0], [-0.1, 0, 0]], **kw)      # converging
    assert a[:, 0] == pytest.approx([-1.963495408, 0.785398163], abs=1e-9)
    a = _acc(x, [2, 5], v=[[-0.1, 0, 0], [0.1, 0, 0]], **kw)      # diverging
    assert a[:, 0] == pytest.approx([-0.490873852, 0.196349541], abs=1e-9)
    a = _acc(x, [2, 5], v=[[0, 1, 0], [0, 1, 0]], **kw)           # rdot == 0 -> gamma*beta (A5)
    assert a[:, 0] == pytest.approx([-0.490873852, 0.196349541], abs=1e-9)
    # dead band: rdot = -0.2 is converging only if v_dead < 0.2
    v = [[0.1, 0, 0], [-0.1, 0, 0]]
    assert _acc(x, [2, 5], v=v, v_dead=0.3, **kw)[0, 0] == pytest.approx(-0.490873852, abs=1e-9)
    assert _acc(x, [2, 5], v=v, v_dead=0.1, **kw)[0, 0] == pytest.approx(-1.963495408, abs=1e-9)
    # not in contact (r >= R_i + R_j): nothing
    assert np.abs(_acc([[0, 0, 0], [2.0, 0, 0]], [2, 5], v=v, **kw)).max() == 0.0


def test_cross_star_pair_uses_mean_radius():
    # A2: R_i=0.6 (star 0), R_j=1.0 (star 1): contact iff r < 1.6, R_ij = 0.8
    star = np.array([0, 1], np.int32)
    kw = dict(G=0.0, gamma=1.0, beta=1.0, R=(0.6, 1.0), star=star)
    assert np.abs(_acc([[0, 0, 0], [1.61, 0, 0]], [1, 1], **kw)).max() == 0.0
    a = _acc([[0, 0, 0], [1.2, 0, 0]], [1, 1], **kw)
    V = math.pi * (2 * 0.8 - 1.2) ** 2 * (4 * 0.8 + 1.2) / 12.0   # 0.184306...
    assert a[0, 0] == pytest.approx(-V, rel=1e-12) and a[1, 0] == pytest.approx(V, rel=1e-12)


def _head_on(beta, dt=2e-4, steps=6000):
    R = 0.1
    posm = np.array([[-0.15, 0, 0, 1.0], [0.15, 0, 0, 1.0]], np.float32)
    vel = np.array([[0.5, 0, 0, 0], [-0.5, 0, 0, 0]], np.float32)
    p = dict(P0, G=0.0, gamma=2.0e4, beta=beta, dt=dt, R_start=(R, R), R_end=(R, R), n_ramp=0)
    s = oracle.Sim(posm, vel, np.zeros(2, np.int32), p)
    s.step(steps)
    return s


def test_p3_restitution_elastic_iff_beta_one():
    s = _head_on(1.0)
    assert s.v[0, 0] == pytest.approx(-0.5, abs=2e-5) and s.v[1, 0] == pytest.approx(0.5, abs=2e-5)
    s = _head_on(0.5)
    e = abs(s.v[0, 0]) / 0.5                  # coefficient of restitution
    # energy returned on the way out is beta times the energy stored on the way in
    assert e == pytest.approx(math.sqrt(0.5), abs=2e-3)
    assert s.x[0, 0] < -0.1 and s.x[1, 0] > 0.1   # they separated again


# ----------------------------------------------- P4/P5/P6: invariants of a run
@pytest.fixture(scope="module")
def small_binary():
    return make_binary(name="t", seed=7, n1=300, n2=212, shape="uniform", radius1=1.0,
                       radius2=0.6, q=0.5, a=3.0, eps=0.01, dt=1e-3, nsteps=0,
                       noise_frac=0.05, ramp_factor1=1.3, n_ramp=40)


def test_p4_newtons_third_law(small_binary):
    w = small_binary
    m = w.posm[:, 3].astype(float)
    a, kap, dl = oracle.accel(w.posm, w.vel, m, w.star, w.params["R_start"], w.params, want_diag=True)
    net = np.linalg.norm((m[:, None] * a).sum(0))
    assert net / (m * np.linalg.norm(a, axis=1)).sum() < 1e-13
    assert (kap >= 1.0 - 1e-12).all()
    # contacts do occur in this workload (otherwise the test above pins only gravity)
    a0 = oracle.accel(w.posm, w.vel, m, w.star, w.params["R_start"], dict(w.params, gamma=0.0))
    assert (np.linalg.norm(a - a0, axis=1) > 0).sum() > 50


def test_p5_momentum_and_angular_momentum_conserved_with_contacts_and_ramp(small_binary):
    w = small_binary
    s = oracle.Sim(w.posm, w.vel, w.star, w.params)
    e0 = s.energy()
    s.step(80)                                 # crosses the end of the 40-step ramp
    e1 = s.energy()
    pscale = (s.m * np.linalg.norm(s.v, axis=1)).sum()
    assert np.abs(e1["P"] - e0["P"]).max() / pscale < 1e-13
    assert np.abs(e1["L"] - e0["L"]).max() / np.abs(e0["L"]).max() < 1e-13
    assert s.n == 80
    R = s.radii()
    assert R[0] == pytest.approx(np.float32(w.params["R_end"][0]), rel=1e-7)


def test_p6_energy_conserved_when_conservative_and_decreasing_when_inelastic(small_binary):
    w = small_binary
    base = dict(w.params, n_ramp=0, R_end=w.params["R_start"])

    def drift(beta, dt, steps, gamma=None):
        p = dict(base, beta=beta, dt=dt)
        if gamma is not None:
            p["gamma"] = gamma
        s = oracle.Sim(w.posm, w.vel, w.star, p)
        e0 = s.energy()["E"]
        s.step(steps)
        return (s.energy()["E"] - e0) / abs(e0)

    d1 = drift(1.0, 1e-3, 40)
    d2 = drift(1.0, 5e-4, 80)
    assert abs(d1) < 1e-3                         # stiff contacts: (omega_c dt)^2 ~ 1e-2 of U_rep ripple
    assert d1 / d2 == pytest.approx(4.0, rel=0.05)  # error ~ dt^2 over the same physical time
    assert abs(drift(1.0, 1e-3, 40, gamma=0.0)) < 1e-6
    assert drift(0.5, 1e-3, 40) < -10 * abs(d1)  # beta < 1 is an energy sink


def test_force_is_minus_gradient_of_energy(small_binary):
    # ties accel (Eqs. 4,5) to the potentials of orc_energy, whose gravity part is
    # pinned by the two-body closed form below and repulsion part by A12's integral
    w = small_binary
    p = dict(w.params, beta=1.0, n_ramp=0, R_end=w.params["R_start"])
    s = oracle.Sim(w.posm, w.vel, w.star, p)
    a = s.accel()
    U = lambda: s.energy()["Ug"] + s.energy()["Urep"]
    h = 1e-6
    for i, c in ((0, 0), (17, 1), (400, 2)):
        x0 = s.x[i, c]
        s.x[i, c] = x0 + h; up = U()
        s.x[i, c] = x0 - h; um = U()
        s.x[i, c] = x0
        assert -(up - um) / (2 * h) / s.m[i] == pytest.approx(a[i, c], rel=2e-6, abs=1e-9)


def test_two_body_potential_closed_form():
    posm = np.array([[0, 0, 0, 2.0], [0, 4, 0, 3.0]], np.float32)
    s = oracle.Sim(posm, np.zeros((2, 4), np.float32), np.zeros(2, np.int32),
                   dict(P0, G=0.5, eps=1.0, dt=1.0, R_start=(0, 0), R_end=(0, 0), n_ramp=0))
    assert s.energy()["Ug"] == pytest.approx(-0.5 * 2 * 3 / 5.0, rel=1e-15)   # -G m1 m2/(r+eps)


# --------------------------------------- P7: circular two-body orbit, leapfrog
def _two_body(a, eps, m1, m2, dt, steps):
    M = m1 + m2
    om = math.sqrt(M / (a * (a + eps) ** 2))      # G=1; softened circular frequency
    posm = np.array([[-a * m2 / M, 0, 0, m1], [a * m1 / M, 0, 0, m2]])
    vel = np.array([[0, -om * a * m2 / M, 0, 0], [0, om * a * m1 / M, 0, 0]])
    s = oracle.Sim(posm, vel, np.zeros(2, np.int32),
                   dict(P0, eps=eps, dt=dt, R_start=(0, 0), R_end=(0, 0), n_ramp=0))
    s.x[:], s.v[:], s.m[:] = posm[:, :3], vel[:, :3], posm[:, 3]   # keep full double inputs
    s.step(steps)
    return s, posm, om


@pytest.mark.parametrize("a,eps,M,T", [(3.0, 0.01, 1.5, 26.74616), (1.0, 0.1, 2.0, 4.887171),
                                        (1.0, 0.0, 1.0, 2 * math.pi)])
def test_p7_softened_circular_orbit_period_and_radius(a, eps, M, T):
    assert 2 * math.pi * math.sqrt(a * (a + eps) ** 2 / M) == pytest.approx(T, rel=2e-7)
    n = 10000
    s, posm, om = _two_body(a, eps, M / 3, 2 * M / 3, T / n, n)
    sep = np.linalg.norm(s.x[1] - s.x[0])
    assert sep == pytest.approx(a, rel=1e-6)                       # radius constant
    assert np.abs(s.x - posm[:, :3]).max() / a < 1e-4             # back at the start after T


def test_leapfrog_is_second_order():
    a, eps, M = 1.0, 0.1, 2.0
    T = 2 * math.pi * math.sqrt(a * (a + eps) ** 2 / M)
    errs = []
    for n in (200, 400, 800):
        s, posm, _ = _two_body(a, eps, 1.0, 1.0, T / n, n)
        errs.append(np.abs(s.x - posm[:, :3]).max())
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.1)
    assert errs[1] / errs[2] == pytest.approx(4.0, rel=0.1)


# ------------------------------------------------- P8 / P9: Eq. 3 and L1
EQ3_K06 = {0.3: 0.281031, 0.4: 0.303053, 0.5: 0.320788, 0.6: 0.335667, 0.8: 0.359772,
           1.0: 0.378921, 2.5: 0.459873, 1 / 0.6: 0.423791, 1 / 0.3: 0.485382}
EQ3_K069 = {0.3: 0.267237, 0.4: 0.287073, 1.0: 0.354265, 2.5: 0.424055}
L1_DIST = {0.3: 0.620867, 0.4: 0.592948, 0.5: 0.570752, 0.6: 0.552343, 0.8: 0.522950, 1.0: 0.5}


def test_p8_eq3_values():
    for q, val in EQ3_K06.items():
        assert oracle.roche_lobe_radius(q, 0.6) == pytest.approx(val, abs=1e-6)
    for q, val in EQ3_K069.items():          # constant as printed
        assert oracle.roche_lobe_radius(q, 0.69) == pytest.approx(val, abs=1e-6)
    # hand evaluation at q=1: 0.49/(0.6 + ln 2) = 0.378921
    assert oracle.roche_lobe_radius(1.0, 0.6) == pytest.approx(0.49 / (0.6 + math.log(2.0)), rel=1e-14)


def _lobe_volume_radius(q_self_over_other: float) -> float:
    """Volume-equivalent radius of the Roche lobe of the star whose mass is the
    numerator, by direct numerical integration of the Roche potential (a=1,
    G(M1+M2)=1): along each ray from the star, the lobe ends where the potential
    first climbs back to its L1 value."""
    qq = q_self_over_other
    mu_s, mu_o = qq / (1 + qq), 1 / (1 + qq)       # this star at origin side
    xs, xo = -mu_o, mu_s                           # barycentre at 0, separation 1
    xl1 = xs + oracle.l1_distance(1.0 / qq)        # l1_distance(q) is measured from the primary of q=m2/m1

    def phi(x, y, z):
        r1 = np.sqrt((x - xs) ** 2 + y ** 2 + z ** 2)
        r2 = np.sqrt((x - xo) ** 2 + y ** 2 + z ** 2)
        return -mu_s / r1 - mu_o / r2 - 0.5 * (x ** 2 + y ** 2)

    phi1 = phi(xl1, 0.0, 0.0)
    nth, nph, nr = 96, 192, 1500
    ct = (np.arange(nth) + 0.5) / nth * 2 - 1
    ph = (np.arange(nph) + 0.5) / nph * 2 * math.pi
    CT, PH = np.meshgrid(ct, ph, indexing="ij")
    ST = np.sqrt(1 - CT ** 2)
    ux, uy, uz = ST * np.cos(PH), ST * np.sin(PH), CT
    rr = (np.arange(nr) + 0.5) / nr * (xl1 - xs) * 1.0001
    inside = np.ones_like(ux, bool)
    rmax = np.zeros_like(ux)
    for r in rr:                                   # march outwards
        inside &= phi(xs + r * ux, r * uy, r * uz) < phi1
        rmax = np.where(inside, r, rmax)
    vol = (rmax ** 3 / 3.0).mean() * 4 * math.pi
    return (3 * vol / (4 * math.pi)) ** (1.0 / 3.0)


@pytest.mark.parametrize("q", [0.4, 1.0, 2.5])
def test_p8_eq3_against_integrated_lobe_volume(q):
    rl = _lobe_volume_radius(q)
    assert oracle.roche_lobe_radius(q, 0.6) == pytest.approx(rl, rel=0.01)          # standard constant
    assert abs(oracle.roche_lobe_radius(q, 0.69) / rl - 1) > 0.04                    # printed 0.69 is off (A9)


def test_p9_l1_location():
    for q, d in L1_DIST.items():
        assert oracle.l1_distance(q) == pytest.approx(d, abs=1e-6)
    assert oracle.l1_distance(1.0) == pytest.approx(0.5, abs=1e-12)
    # a massless element at L1 co-rotates: a + omega^2 x = 0 (omega^2 = G M / a^3, eps=gamma=0)
    q, a = 0.4, 2.5
    M1, M2 = 1.0, q
    x1, x2 = -a * q / (1 + q), a / (1 + q)
    xt = x1 + a * oracle.l1_distance(q)
    acc = _acc([[x1, 0, 0], [x2, 0, 0], [xt, 0, 0]], [M1, M2, 1e-12])
    om2 = (M1 + M2) / a ** 3
    assert acc[2, 0] + om2 * xt == pytest.approx(0.0, abs=1e-9)


def test_config3_ramp_factor_literal_matches_eq3():
    from workloads.configs import CONFIG3_RAMP_FACTOR
    q, a, R1 = 0.4, 2.5, 1.0
    assert oracle.roche_lobe_radius(1 / q, 0.6) * a / R1 == pytest.approx(CONFIG3_RAMP_FACTOR, abs=1e-6)


# ---------------------------------------------------------- P10: shell theorem
def test_p10_shell_theorem_uniform_sphere():
    w = make_binary(name="s", seed=3, n1=20000, n2=1, shape="uniform", radius1=1.0, radius2=0.1,
                    q=1e-9, a=50.0, eps=1e-6, dt=1.0, nsteps=0, noise_frac=0.0, gamma=0.0)
    x = w.posm[:-1, :3].astype(float)
    c = x.mean(0)                       # centre of mass (equal masses): kills the dipole term
    probes = np.array([[1.5, 0, 0], [0, -3.0, 0], [0, 0, 6.0]]) + c      # outside: GM/r^2
    xx = np.concatenate([x, probes])
    mm = np.concatenate([w.posm[:-1, 3].astype(float), np.full(len(probes), 1e-30)])
    a = oracle.accel(xx, np.zeros_like(xx), mm, np.zeros(len(xx), np.int32), (0, 0),
                     dict(P0, eps=1e-6))
    for k, pr in enumerate(probes - c):
        r = np.linalg.norm(pr)
        assert a[len(x) + k] == pytest.approx(-pr / r ** 3, rel=0, abs=1e-2 / r ** 2)   # sampling quadrupole ~ N^-1/2 / r^4
    # inside: the mean radial acceleration over a shell of elements is -G M r / R^3
    d = x - c
    r = np.linalg.norm(d, axis=1)
    arad = (a[:len(x)] * d).sum(1) / r
    for lo, hi in ((0.3, 0.4), (0.5, 0.6), (0.7, 0.8), (0.9, 1.0)):
        sel = (r >= lo) & (r < hi)
        assert sel.sum() > 500
        assert arad[sel].mean() == pytest.approx(-r[sel].mean(), abs=0.02)


# -------------------------------------------------------- expanding-star rule
def test_radius_ramp_linear_in_step_count():
    Rs, Re = (0.02, 0.03), (0.05, 0.03)
    f32 = lambda v: float(np.float32(v))
    assert oracle.radii(0, Rs, Re, 100)[0] == f32(0.02)
    assert oracle.radii(50, Rs, Re, 100)[0] == f32(0.035)
    assert oracle.radii(100, Rs, Re, 100)[0] == f32(0.05)
    assert oracle.radii(1000, Rs, Re, 100)[0] == f32(0.05)       # stays at R_end
    assert oracle.radii(7, Rs, Re, 100)[1] == f32(0.03)          # other star static
    assert oracle.radii(7, Rs, Re, 0)[0] == f32(0.02)            # n_ramp=0: R = R_start
    inc = np.diff([oracle.radii(n, Rs, Re, 100)[0] for n in range(101)])
    assert np.allclose(inc, 0.0003, atol=1e-8)


def test_kdk_uses_cached_acceleration_and_half_step_velocity():
    # one step by hand for a two-body problem (A7): v_half = v0 + dt/2 a(x0); x1 = x0 + dt v_half;
    # v1 = v_half + dt/2 a(x1)
    posm = np.array([[0, 0, 0, 1.0], [2, 0, 0, 1.0]], np.float32)
    vel = np.array([[0, 0.125, 0, 0], [0, -0.125, 0, 0]], np.float32)   # exact in float32
    p = dict(P0, eps=0.5, dt=0.25, R_start=(0, 0), R_end=(0, 0), n_ramp=0)
    s = oracle.Sim(posm, vel, np.zeros(2, np.int32), p)
    s.step(1)
    a0 = 1 / 2.5 ** 2                                  # 0.16 toward each other
    vhx = 0.125 * a0                                   # 0.02
    x0 = 0.25 * vhx                                    # 0.005
    assert s.x[0] == pytest.approx([x0, 0.03125, 0], abs=1e-15)
    d = np.array([2 - 2 * x0, -0.0625, 0])
    r = np.linalg.norm(d)
    a1 = d / r / (r + 0.5) ** 2
    assert s.v[0] == pytest.approx(np.array([vhx, 0.125, 0]) + 0.125 * a1, abs=1e-15)
    # splitting a run into several calls changes nothing (cached acceleration)
    s1 = oracle.Sim(posm, vel, np.zeros(2, np.int32), p); s1.step(6)
    s2 = oracle.Sim(posm, vel, np.zeros(2, np.int32), p); s2.step(2); s2.step(4)
    assert np.array_equal(s1.x, s2.x) and np.array_equal(s1.v, s2.v)


def test_rows_subset_and_thread_count_independence():
    w = make_config(1, scale=0.25)
    m = w.posm[:, 3]
    a = oracle.accel(w.posm, w.vel, m, w.star, w.params["R_start"], w.params)
    rows = np.array([5, 0, 300, 511])
    ar = oracle.accel(w.posm, w.vel, m, w.star, w.params["R_start"], w.params, rows=rows)
    assert np.array_equal(a[rows], ar)


# ------------------------- A6: the allowance every parity assertion subtracts (orc_accel's delta)
def test_a6_delta_hand_numbers_band_and_branch_independence():
    # geometry of test_contact_hand_numbers_and_branch: R = 1, r = 1 -> pi V = 5 pi/12 = 1.308996939,
    # gamma = 3, beta = 0.25, m = (2, 5), rdot = -0.2.  A pair within tau_s of the switch contributes
    # (1 - beta) gamma pi V / m_i:  0.75 * 3 * 1.308996939 / 2 = 1.472621556,  / 5 = 0.589048623.
    x = [[0, 0, 0], [1, 0, 0]]
    v = [[0.1, 0, 0], [-0.1, 0, 0]]
    kw = dict(P0, G=0.0, gamma=3.0, beta=0.25)

    def delta(**over):
        a, kap, dl = oracle.accel(np.array(x, float), np.array(over.pop("v", v), float), np.array([2.0, 5.0]),
                                  np.zeros(2, np.int32), over.pop("R", (1.0, 1.0)), dict(kw, **over), want_diag=True)
        return a, dl

    a_lo, dl = delta(v_dead=0.2 - 5e-6, tau_s=1e-5)          # |rdot + v_dead| = 5e-6 <= tau_s
    assert dl == pytest.approx([1.472621556, 0.589048623], abs=1e-9)
    a_hi, dl2 = delta(v_dead=0.2 + 5e-6, tau_s=1e-5)         # the other side of the switch: same allowance
    assert np.array_equal(dl, dl2)
    # ... and the two sides differ by exactly that allowance (gamma vs gamma*beta on the one pair)
    assert np.abs(a_lo - a_hi)[:, 0] == pytest.approx(dl, rel=1e-12)
    assert delta(v_dead=0.2 - 5e-6, tau_s=1e-6)[1] == pytest.approx([0.0, 0.0], abs=0)    # outside the band
    assert delta(v_dead=0.2 + 5e-6, tau_s=4.9e-6)[1] == pytest.approx([0.0, 0.0], abs=0)
    assert delta(v_dead=0.2 + 5e-6, tau_s=5.1e-6)[1][0] > 0                                # band edge is 5e-6
    assert delta(v_dead=0.0, tau_s=1e-5)[1] == pytest.approx([0.0, 0.0], abs=0)            # rdot = -0.2 is far from 0
    # the band is |rdot + v_dead|, in velocity units, symmetric: rdot = +0.2 (diverging) with v_dead = 0 is far, too
    assert delta(v=[[-0.1, 0, 0], [0.1, 0, 0]], v_dead=0.0, tau_s=0.19)[1] == pytest.approx([0.0, 0.0], abs=0)
    assert delta(v=[[-0.1, 0, 0], [0.1, 0, 0]], v_dead=0.0, tau_s=0.21)[1][0] == pytest.approx(1.472621556, abs=1e-9)
    # a pair that is not in contact has no allowance, whatever its rdot
    x[1][0] = 2.0
    assert delta(v_dead=0.2, tau_s=1.0)[1] == pytest.approx([0.0, 0.0], abs=0)
    x[1][0] = 1.0
    # gamma = 0 (no contact terms at all) and beta = 1 (both branches equal): nothing to allow for
    assert delta(v_dead=0.2, tau_s=1.0, gamma=0.0)[1] == pytest.approx([0.0, 0.0], abs=0)
    assert delta(v_dead=0.2, tau_s=1.0, beta=1.0)[1] == pytest.approx([0.0, 0.0], abs=0)


def test_a6_delta_sums_over_the_ambiguous_pairs_of_a_row_only():
    # element 0 touches 1 (on the switch) and 2 (clearly converging): only pair (0,1) is allowed for.
    # R = 1: pair (0,1) r = 1 -> pi V = 5 pi/12; pair (0,2) r = 1.5 -> pi (0.5)^2 (5.5)/12 = 0.359974158
    x = np.array([[0, 0, 0], [1, 0, 0], [-1.5, 0, 0]], float)           # 1 and 2 are 2.5 apart: no contact
    v = np.array([[0, 0, 0], [-0.2, 0, 0], [3.0, 0, 0]], float)
    p = dict(P0, G=0.0, gamma=2.0, beta=0.5, v_dead=0.2, tau_s=1e-9)
    a, kap, dl = oracle.accel(x, v, np.array([1.0, 1.0, 4.0]), np.zeros(3, np.int32), (1.0, 1.0), p, want_diag=True)
    assert dl == pytest.approx([0.5 * 2.0 * 1.308996939, 0.5 * 2.0 * 1.308996939, 0.0], abs=1e-9)
    # rdot == -v_dead exactly is NOT converging (A5: strict <): pair (0,1) takes gamma*beta, pair (0,2) gamma
    assert a[0] == pytest.approx([-1.0 * 1.308996939 + 2.0 * 0.359974158, 0.0, 0.0], abs=1e-9)
    assert a[2] == pytest.approx([-2.0 * 0.359974158 / 4.0, 0.0, 0.0], abs=1e-9)


def test_kappa_hand_values():
    # kappa_i = sum_j |a_ij| / |a_i|.  Two bodies: one term, kappa = 1 exactly.
    a, kap, dl = oracle.accel(np.array([[0, 0, 0], [3.0, 0, 0]]), np.zeros((2, 3)), np.array([1.0, 2.0]),
                              np.zeros(2, np.int32), (0, 0), dict(P0, eps=1.0), want_diag=True)
    assert kap == pytest.approx([1.0, 1.0], abs=1e-15) and (dl == 0).all()
    # the collinear case of test_p1_collinear_unequal_masses_literal: the middle element is pulled both ways,
    # kappa_1 = (0.888888889 + 1.28) / 0.391111111 = 5.545454545; the outer ones one way only
    a, kap, _ = oracle.accel(np.array([[0, 0, 0], [1.0, 0, 0], [3.0, 0, 0]]), np.zeros((3, 3)),
                             np.array([1.0, 2.0, 4.0]), np.zeros(3, np.int32), (0, 0), dict(P0, G=2.0, eps=0.5),
                             want_diag=True)
    assert kap == pytest.approx([1.0, 5.545454545, 1.0], abs=2e-9)
    # a contact term counts with its own magnitude: gravity 1/(1+0)^2 = 1 toward j, repulsion 3 * 5pi/12 / 2 away
    a, kap, _ = oracle.accel(np.array([[0, 0, 0], [1.0, 0, 0]]), np.array([[0.1, 0, 0], [-0.1, 0, 0]]),
                             np.array([2.0, 1.0]), np.zeros(2, np.int32), (1.0, 1.0),
                             dict(P0, G=1.0, gamma=3.0, beta=0.25), want_diag=True)
    assert a[0, 0] == pytest.approx(1.0 - 1.963495408, abs=1e-9) and kap[0] == pytest.approx(1.0, abs=1e-12)


def test_energy_net_force_output_hand_pair():
    # out[10] = |sum_i m_i a_i| of the acceleration array handed in: m = (2, 3), a = ((1,0,0), (0,2,0))
    # -> |(2, 6, 0)| = sqrt(40) = 6.32455532
    posm = np.array([[0, 0, 0, 2.0], [0, 4, 0, 3.0]], np.float32)
    s = oracle.Sim(posm, np.zeros((2, 4), np.float32), np.zeros(2, np.int32),
                   dict(P0, eps=1.0, dt=1.0, R_start=(0, 0), R_end=(0, 0), n_ramp=0))
    s.acc[:] = [[1.0, 0, 0], [0, 2.0, 0]]
    s.have_acc.value = 1
    assert s.energy()["Fnet"] == pytest.approx(6.32455532, abs=1e-8)
    s.have_acc.value = 0                      # computed from the state: Newton's third law, exactly opposite forces
    assert s.energy()["Fnet"] == pytest.approx(0.0, abs=1e-15)


def test_contact_list_hand_and_brute_force():
    # hand pair of the tests above: r = 1, rdot = -0.2, seen from both sides; a third element out of reach
    x = np.array([[0, 0, 0], [1, 0, 0], [0, 2.5, 0]], float)
    v = np.array([[0.1, 0, 0], [-0.1, 0, 0], [0, 0, 0]], float)
    cnt, jj, rr, rd = oracle.contact_list(x, v, np.array([0, 0, 1], np.int32), (1.0, 1.0))
    assert cnt.tolist() == [1, 1, 0] and jj[:, 0].tolist() == [1, 0, -1]
    assert rr[:2, 0] == pytest.approx([1.0, 1.0]) and rd[:2, 0] == pytest.approx([-0.2, -0.2], abs=1e-15)
    # A2: cross-star reach is R_0 + R_1 = 1.6 < 2.5; with R_1 = 2 element 2 touches 0 (r = 2.5 < 3) but sideways: rdot = 0...
    cnt, jj, rr, rd = oracle.contact_list(x, v, np.array([0, 0, 1], np.int32), (1.0, 2.0), rows=[2, 0])
    assert cnt.tolist() == [2, 2] and jj[0, :2].tolist() == [0, 1] and jj[1, :2].tolist() == [1, 2]
    assert rr[0, 0] == pytest.approx(2.5) and rd[0, 0] == pytest.approx(0.0, abs=1e-15)
    # ... and moving toward it along the line of centres: rdot = -speed, the same seen from either element
    v[2] = [0, -0.7, 0]
    assert oracle.contact_list(x, v, np.array([0, 0, 1], np.int32), (1.0, 2.0), rows=[2])[3][0, 0] == pytest.approx(-0.7)
    assert oracle.contact_list(x, v, np.array([0, 0, 1], np.int32), (1.0, 2.0), rows=[0])[3][0, 1] == pytest.approx(-0.7)
    # brute force on a seeded workload, with numpy: same counts, same partners, same rdot; cap truncates the lists only
    w = make_binary(name="t", seed=9, n1=200, n2=150, shape="uniform", radius1=1.0, radius2=0.6, q=0.5, a=1.4,
                    eps=0.01, dt=1e-3, nsteps=0)
    R = np.array(w.params["R_start"])
    X, V = w.posm[:, :3].astype(float), w.vel[:, :3].astype(float)
    cnt, jj, rr, rd = oracle.contact_list(X, V, w.star, R, cap=6)
    d = X[None, :, :] - X[:, None, :]
    r = np.sqrt((d ** 2).sum(-1))
    reach = R[w.star][:, None] + R[w.star][None, :]
    touch = (r < reach) & (r > 0)
    assert np.array_equal(cnt, touch.sum(1)) and cnt.max() > 6 and (cnt == 0).any()
    rdot = (d * (V[None, :, :] - V[:, None, :])).sum(-1) / np.where(r > 0, r, 1.0)
    for i in range(w.n):
        js = np.flatnonzero(touch[i])[:6]
        assert jj[i, :len(js)].tolist() == js.tolist() and (jj[i, len(js):] == -1).all()
        assert np.allclose(rd[i, :len(js)], rdot[i, js], rtol=1e-13, atol=1e-15)
    # the contact terms of orc_accel act on exactly these rows
    p = dict(w.params, R_start=tuple(R))
    a1 = oracle.accel(w.posm, w.vel, w.posm[:, 3], w.star, R, p)
    a0 = oracle.accel(w.posm, w.vel, w.posm[:, 3], w.star, R, dict(p, gamma=0.0))
    assert np.array_equal(np.linalg.norm(a1 - a0, axis=1) > 0, cnt > 0)


def test_a6_population_follows_from_the_rdot_density(small_binary):
    """The number of rows with delta > 0 is what the rdot distribution of the contact pairs predicts:
    pairs within tau_s of -v_dead.  (The GPU tests bound their A6 population the same way.)"""
    w = small_binary
    R = np.array(w.params["R_start"]) * 1.5
    p = dict(w.params, tau_s=0.02 * w.meta["omega"] * w.meta["a"])      # a wide band so that it is populated
    _, _, dl = oracle.accel(w.posm, w.vel, w.posm[:, 3], w.star, R, p, want_diag=True)
    cnt, jj, rr, rd = oracle.contact_list(w.posm, w.vel, w.star, R, cap=int(64))
    assert cnt.max() <= 64
    inband = np.abs(rd + p["v_dead"]) <= p["tau_s"]                      # NaN (no pair) compares False
    assert np.array_equal(dl > 0, inband.any(1)) and 3 < (dl > 0).sum() < w.n


# ------------------------------------------------------------------ round 3: the last unpinned output, A3 in energies, P5 as written
def test_angular_and_linear_momentum_by_hand():
    """orc_energy's P and L against numbers worked out by hand (not by conservation, which a flipped sign or a
    permuted component would survive): m = 2 at x = (1, 2, 3), v = (0.5, -1, 0.25) has x cross v = (3.5, 1.25, -2),
    m = 3 at x = (-1, 0, 2), v = (0, 1, -1) has x cross v = (-2, -1, -1)."""
    posm = np.array([[1.0, 2.0, 3.0, 2.0], [-1.0, 0.0, 2.0, 3.0]])
    vel = np.array([[0.5, -1.0, 0.25, 0.0], [0.0, 1.0, -1.0, 0.0]])
    p = dict(G=1.0, eps=0.1, dt=1e-3, q=1.0, gamma=0.0, beta=1.0, R_start=(0.0, 0.0), R_end=(0.0, 0.0), n_ramp=0)
    one = oracle.Sim(posm[:1], vel[:1], np.zeros(1, np.int32), p).energy()
    assert np.allclose(one["L"], [7.0, 2.5, -4.0], rtol=0, atol=1e-15)
    assert np.allclose(one["P"], [1.0, -2.0, 0.5], rtol=0, atol=1e-15)
    both = oracle.Sim(posm, vel, np.array([0, 1], np.int32), p).energy()
    assert np.allclose(both["L"], [1.0, -0.5, -7.0], rtol=0, atol=1e-15)
    assert np.allclose(both["P"], [1.0, 1.0, -2.5], rtol=0, atol=1e-15)
    assert both["KE"] == pytest.approx(0.5 * 2 * (0.25 + 1 + 0.0625) + 0.5 * 3 * 2.0, abs=1e-15)


def test_a3_coincident_pair_no_force_but_its_potentials_by_formula():
    """Reading A3: two distinct elements at one point exert no force on each other (d/r has no
    direction there), while both potentials are evaluated by their formulas, which are finite at r = 0 when
    eps > 0: the pair adds -G m_i m_j / eps to U_grav and gamma pi R^4 to U_rep (A12 at r = 0).  With a third
    element present the coincident two feel only it -- and equally."""
    posm = np.array([[0.5, -1.0, 2.0, 2.0], [0.5, -1.0, 2.0, 3.0]])
    vel = np.zeros((2, 4))
    star = np.zeros(2, np.int32)
    p = dict(G=1.5, eps=0.25, dt=1e-3, q=1.0, gamma=400.0, beta=0.5, R_start=(0.1, 0.1), R_end=(0.1, 0.1), n_ramp=0)
    a = oracle.accel(posm, vel, posm[:, 3], star, p["R_start"], p)
    assert (a == 0).all()
    e = oracle.Sim(posm, vel, star, p).energy()
    assert e["Ug"] == pytest.approx(-1.5 * 6.0 / 0.25, rel=1e-15)               # -36
    assert e["Urep"] == pytest.approx(400.0 * np.pi * float(np.float32(0.1)) ** 4, rel=1e-12)   # the radius is an fp32 model parameter (A8)
    third = np.array([[0.5, -1.0, 4.0, 1.0]])                                  # 2 above them, out of contact
    posm3 = np.concatenate([posm, third]); vel3 = np.zeros((3, 4)); star3 = np.zeros(3, np.int32)
    a3 = oracle.accel(posm3, vel3, posm3[:, 3], star3, p["R_start"], p)
    g = 1.5 * 1.0 / (2.0 + 0.25) ** 2
    assert np.allclose(a3[0], [0, 0, g], atol=1e-15) and np.array_equal(a3[0], a3[1])
    assert np.allclose(a3[2], [0, 0, -1.5 * 5.0 / 2.25 ** 2], atol=1e-15)
    # eps = 0: the singularity eps exists to remove -- U_grav of the coincident pair diverges
    with np.errstate(divide="ignore"):
        e0 = oracle.Sim(posm, vel, star, dict(p, eps=0.0)).energy()
    assert e0["Ug"] == -np.inf and (oracle.accel(posm, vel, posm[:, 3], star, p["R_start"], dict(p, eps=0.0)) == 0).all()


def test_p5_as_written_config1_thousand_steps():
    """total momentum and angular momentum of config 1 (N = 2,048, contacts on) over 1,000 leapfrog
    steps (the integrator is 'conservative'), relative to sum m |v| and |L|, at the 1e-12 the survey states."""
    w = make_config(1)
    s = oracle.Sim(w.posm, w.vel, w.star, w.params)
    e0 = s.energy()
    pscale = (s.m * np.linalg.norm(s.v, axis=1)).sum()
    for _ in range(4):
        s.step(250)
        e = s.energy()
        assert np.abs(e["P"] - e0["P"]).max() / pscale < 1e-12
        assert np.abs(e["L"] - e0["L"]).max() / np.linalg.norm(e0["L"]) < 1e-12
    assert s.n == 1000
    assert np.isfinite(e["E"]) and e["E"] < e0["E"]                             # beta < 1: the contacts of the unrelaxed stars dissipate

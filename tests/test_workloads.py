"""The seeded input recipes: shapes, determinism, derived numbers."""
import numpy as np
import pytest

from workloads import CONFIGS, make_binary, make_config, params_f32


@pytest.mark.parametrize("idx,n1,n2,omega,re1,re2", [
    (1, 1024, 1024, 0.235702, 0.085499, 0.051299),
    (2, 8192, 8192, 0.167705, 0.042749, 0.034200),
    (3, 49152, 16384, 0.299333, 0.023526, 0.016965),
])
def test_config_tables(idx, n1, n2, omega, re1, re2):
    w = make_config(idx)
    assert (w.meta["n1"], w.meta["n2"], w.n) == (n1, n2, n1 + n2)
    assert w.meta["omega"] == pytest.approx(omega, abs=1e-6)
    assert w.params["R_start"] == pytest.approx((re1, re2), abs=1e-6)
    assert w.posm.dtype == np.float32 and w.posm.shape == (w.n, 4) and w.vel.shape == (w.n, 4)
    assert (w.star[:n1] == 0).all() and (w.star[n1:] == 1).all()
    m = w.posm[:, 3].astype(np.float64)
    q = CONFIGS[idx]["q"]
    assert m[:n1].sum() == pytest.approx(1.0, rel=1e-6) and m[n1:].sum() == pytest.approx(q, rel=1e-6)
    # barycentre at the origin, stars where the recipe puts them
    a = w.meta["a"]
    assert w.posm[:n1, 0].mean() == pytest.approx(-a * q / (1 + q), abs=0.05)
    assert w.posm[n1:, 0].mean() == pytest.approx(a / (1 + q), abs=0.05)


def test_config1_is_rigid_rotation_and_config3_ramps():
    w = make_config(1)
    om = w.meta["omega"]
    assert np.allclose(w.vel[:, 0], -om * w.posm[:, 1], atol=1e-6)
    assert np.allclose(w.vel[:, 1], om * w.posm[:, 0], atol=1e-6)
    assert (w.vel[:, 2] == 0).all() and w.params["n_ramp"] == 0
    w3 = make_config(3, scale=1 / 64)
    assert w3.params["n_ramp"] == 1000
    assert w3.params["R_end"][0] / w3.params["R_start"][0] == pytest.approx(1.149683, rel=1e-9)
    assert w3.params["R_end"][1] == w3.params["R_start"][1]


def test_generation_is_deterministic_and_seeded():
    a, b = make_config(2, scale=1 / 16), make_config(2, scale=1 / 16)
    assert np.array_equal(a.posm, b.posm) and np.array_equal(a.vel, b.vel)
    c = make_binary(**dict(CONFIGS[2], n1=512, n2=512, seed=99))
    assert not np.array_equal(a.posm, c.posm)
    assert np.std(np.log(a.posm[:512, 3])) == pytest.approx(0.1, rel=0.15)      # lognormal masses


def test_params_f32_rounds_once():
    p = params_f32(make_config(1).params)
    for k in ("G", "eps", "dt", "gamma", "beta", "v_dead"):
        assert p[k] == float(np.float32(p[k]))
    assert all(v == float(np.float32(v)) for v in p["R_start"] + p["R_end"])
    assert p["n_ramp"] == 0 and p["lens_mode"] == 0

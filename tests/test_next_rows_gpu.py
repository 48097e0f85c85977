"""GPU parity of the SURVEY.md 8(f) "next" rows, through the C ABI, against the oracle:
f1 scenario variants (parameter sets of the same kernels), f2 relaxation steps, f3 mass-transfer
diagnostics, f4 point splat."""
import numpy as np
import pytest

import oracle
from workloads import make_config, make_scenario, params_f32, SCENARIOS

pytestmark = pytest.mark.gpu

POS_TOL = 1.0e-4
ACC_TOL = 2.0e-5


def _sim(nb, w, p=None, **kw):
    return nb.Simulation(w.posm, w.vel, w.star, p or params_f32(w.params), **kw)


# ------------------------------------------------------------------ f1: scenarios
@pytest.mark.parametrize("key", sorted(SCENARIOS))
def test_scenario_accel_and_ten_steps(nb, key):
    """Each of the paper's three kinds of run: accelerations and a 10-step
    trajectory, with the per-star radius ramps (both stars expanding in case B)."""
    w = make_scenario(key)
    p = params_f32(w.params)
    s = _sim(nb, w, p)
    a = s.compute_accel().cpu().numpy().astype(np.float64)[:, :3]
    a_or, kap, dl = oracle.accel(w.posm, w.vel, w.posm[:, 3], w.star, p["R_start"], p, want_diag=True)
    err = np.linalg.norm(a - a_or, axis=1)
    an = np.linalg.norm(a_or, axis=1)
    assert (np.maximum(err - dl, 0) / an).max() <= ACC_TOL
    from test_parity_gpu import _a6_population
    _a6_population(w, p, np.arange(w.n), dl, cap=64)              # the allowance covers a predictable sliver of rows
    s.step(10); s.synchronize()
    o = oracle.Sim(w.posm, w.vel, w.star, p); o.step(10)
    x = s.posm.cpu().numpy().astype(np.float64)[:, :3]
    step, R = nb.nb_get_step(s.ctx)
    assert step == 10 and np.array_equal(np.asarray(R, np.float64), o.radii().astype(np.float32).astype(np.float64))
    if key == "case_b_both_expand":
        assert R[0] > p["R_start"][0] and R[1] > p["R_start"][1]
    assert np.linalg.norm(x - o.x, axis=1).max() / w.meta["a"] <= POS_TOL
    from test_parity_gpu import _check_velocities
    _check_velocities(s.vel.cpu().numpy().astype(np.float64)[:, :3], o.v, w)
    s.close()


def test_scenario_long_run_invariants_and_transfer_begins(nb):
    """Case B at a quarter of its size, the full 200-step ramp: momentum and angular momentum conserved,
    no NaN, and the expanding stars start to push elements across the L1 plane."""
    w = make_scenario("case_b_both_expand", scale=0.25)
    s = _sim(nb, w)
    e0, t0 = s.energy(), s.transfer_diagnostics()
    s.step(200)
    e1, t1 = s.energy(), s.transfer_diagnostics()
    assert t1["step"] == 200 and np.isfinite([e1["E"], e1["KE"]]).all()
    Lz = abs(e0["L"][2])
    assert np.abs(np.array(e1["P"]) - np.array(e0["P"])).max() < 1e-5 * 0.3
    assert np.abs(np.array(e1["L"]) - np.array(e0["L"])).max() < 1e-4 * Lz
    assert t1["M0"] == pytest.approx(t0["M0"], rel=1e-12) and t1["M1"] == pytest.approx(t0["M1"], rel=1e-12)
    assert t1["Mcross0"] + t1["Mcross1"] >= t0["Mcross0"] + t0["Mcross1"]
    s.close()


# ------------------------------------------------------------------ f2: relaxation
@pytest.mark.parametrize("kappa", [0.0, 5.0, 40.0, 5000.0])
def test_relax_parity(nb, kappa):
    w = make_config(1)
    p = params_f32(w.params)
    s = _sim(nb, w, p)
    s.relax(10, kappa); s.synchronize()
    o = oracle.Sim(w.posm, w.vel, w.star, p); o.relax(10, kappa)
    x = s.posm.cpu().numpy().astype(np.float64)[:, :3]
    v = s.vel.cpu().numpy().astype(np.float64)[:, :3]
    assert np.linalg.norm(x - o.x, axis=1).max() / w.meta["a"] <= POS_TOL
    from test_parity_gpu import _check_velocities
    _check_velocities(v, o.v, w)
    if kappa * p["dt"] >= 1.0:
        assert (v == 0).all()
    assert nb.nb_get_step(s.ctx)[0] == 10
    s.close()


def test_relax_zero_damping_is_nb_step_bitwise_and_mixes_with_it(nb):
    import torch
    w = make_config(3, scale=0.75)                  # symmetric kernel + radius ramp
    p = params_f32(w.params)
    a, b = _sim(nb, w, p), _sim(nb, w, p)
    a.relax(3, 0.0); a.step(2); b.step(5)
    a.synchronize(); b.synchronize()
    # relax() splits the two half kicks that step() merges (v + h a + h a vs v + 2h a): same to rounding
    assert torch.allclose(a.posm, b.posm, rtol=0, atol=2e-6) and torch.allclose(a.vel, b.vel, rtol=0, atol=2e-6)
    assert nb.nb_get_step(a.ctx) == nb.nb_get_step(b.ctx)
    a.close(); b.close()


def test_relax_settles_a_single_star(nb):
    """One star alone (a star is put together from elements first): damping drains the
    kinetic energy the Poisson-random placement releases; momentum stays ~0; the star stays bound."""
    w = make_config(1)
    n1 = w.meta["n1"]
    posm, vel, star = w.posm[:n1].copy(), np.zeros_like(w.vel[:n1]), w.star[:n1].copy()
    p = params_f32(dict(w.params, dt=2e-3))
    s = nb.Simulation(posm, vel, star, p)
    s.relax(150, 0.0)
    hot = s.energy()
    s.relax(300, 25.0)
    cold = s.energy()
    assert cold["KE"] < 0.2 * hot["KE"] and cold["E"] < hot["E"]
    assert np.abs(cold["P"]).max() < 1e-5
    x = s.posm.cpu().numpy()[:, :3].astype(np.float64)
    r = np.linalg.norm(x - x.mean(0), axis=1)
    assert np.isfinite(r).all() and np.median(r) < 1.5
    s.close()


def test_relax_argument_errors(nb):
    s = _sim(nb, make_config(1, scale=0.125))
    L = nb.lib()
    assert L.nb_relax(s.ctx, -1, 0.0) == nb.NB_EINVAL
    assert L.nb_relax(s.ctx, 1, -0.5) == nb.NB_EINVAL
    assert L.nb_relax(s.ctx, 1, float("nan")) == nb.NB_EINVAL
    assert L.nb_relax(None, 1, 0.0) == nb.NB_EINVAL
    assert L.nb_relax(s.ctx, 0, 1.0) == nb.NB_OK
    s.close()


# ------------------------------------------------------------------ f3: transfer diagnostics
def _check_transfer(nb, posm, vel, star, p, k=0.6):
    s = nb.Simulation(posm, vel, star, p)
    g = s.transfer_diagnostics(k)
    s.close()
    o = oracle.transfer_diagnostics(posm, vel, posm[:, 3], star, k, band=1e-9)
    for f in ("M0", "M1", "a", "d0", "rL0", "rL1"):
        assert g[f] == pytest.approx(o[f], rel=1e-12), f
    assert np.allclose(g["X"], o["X"], rtol=0, atol=1e-12) and np.allclose(g["V"], o["V"], rtol=0, atol=1e-12)
    slack = o["ambiguous"] + 1e-12 * (o["M0"] + o["M1"])       # elements sitting on a decision surface
    for f in ("Mcross0", "Mcross1", "Min0", "Min1", "Mout0", "Mout1"):
        assert abs(g[f] - o[f]) <= slack, (f, g[f], o[f])
    Lscale = max(np.abs(o["Ldisk"]).max(), 1e-300)
    assert np.abs(np.array(g["Ldisk"]) - o["Ldisk"]).max() <= 1e-11 * Lscale + slack * 10
    return g, o


@pytest.mark.parametrize("idx", [1, 3])
def test_transfer_diagnostics_parity_detached(nb, idx):
    w = make_config(idx)
    g, _ = _check_transfer(nb, w.posm, w.vel, w.star, params_f32(w.params))
    assert g["Mcross0"] == g["Min0"] == 0.0 and g["step"] == 0


@pytest.mark.parametrize("k", [0.6, 0.69])
def test_transfer_diagnostics_parity_with_transferred_mass(nb, k):
    """Config 3 with a twentieth of the donor displaced toward and past the accretor: every output
    is non-trivial (elements beyond L1, inside the accretor's lobe with angular momentum, and outside)."""
    w = make_config(3)
    rng = np.random.default_rng(5)
    m = w.n // 20
    w.posm[:m, :3] += np.float32([1.3, 0.05, 0.0]) + rng.normal(0, 0.4, (m, 3)).astype(np.float32)
    w.posm[m:2 * m, 2] += np.float32(3.0)            # a puff far above the plane: outside both lobes
    g, o = _check_transfer(nb, w.posm, w.vel, w.star, params_f32(w.params), k)
    assert g["Mcross0"] > 0.01 and g["Min0"] > 0.001 and g["Mout0"] > 0.01 and abs(g["Ldisk"][0][2]) > 0


def test_transfer_diagnostics_heavier_second_star_and_single_star(nb):
    w = make_config(1)
    w.posm[w.star == 1, 3] *= np.float32(4.0)        # star 1 becomes the primary: mirrored L1
    g, o = _check_transfer(nb, w.posm, w.vel, w.star, params_f32(w.params))
    assert g["M1"] > g["M0"] and g["d0"] < 0.5 * g["a"]
    n1 = w.meta["n1"]
    s = nb.Simulation(w.posm[:n1].copy(), w.vel[:n1].copy(), w.star[:n1].copy(), params_f32(w.params))
    g1 = s.transfer_diagnostics()
    s.close()
    assert g1["M1"] == 0.0 and g1["a"] == 0.0 and g1["Mcross0"] == 0.0
    assert g1["M0"] == pytest.approx(float(w.posm[:n1, 3].astype(np.float64).sum()), rel=1e-12)


def test_transfer_diagnostics_argument_errors(nb):
    import ctypes as C
    s = _sim(nb, make_config(1, scale=0.125))
    out = (C.c_double * 32)()
    L = nb.lib()
    assert L.nb_transfer_diagnostics(s.ctx, 0.0, out) == nb.NB_EINVAL
    assert L.nb_transfer_diagnostics(s.ctx, 0.6, None) == nb.NB_EINVAL
    assert L.nb_transfer_diagnostics(None, 0.6, out) == nb.NB_EINVAL
    s.close()


# ------------------------------------------------------------------ f4: point splat
def _splat_vs_definition(got, pos, star, centre, hw, axes, W, H):
    """The kernel's image against the fp64 definition (oracle.splat_exact): per pixel they may differ by no more
    than the number of elements of the pixel's 3 x 3 neighbourhood that sit within the float32 rounding band of a
    pixel edge (either pixel is right for those); the in-window totals likewise at the window's border."""
    ref, amb = oracle.splat_exact(pos, star, centre, hw, axes[0], axes[1], W, H)
    nb_amb = sum(amb[:, 1 + dy:1 + dy + H, 1 + dx:1 + dx + W].astype(np.int64) for dy in (-1, 0, 1) for dx in (-1, 0, 1))
    diff = np.abs(got - ref.astype(np.int64))
    assert (diff <= nb_amb).all(), int((diff > nb_amb).sum())
    border = int(amb[:, :, [0, 1, W, W + 1]].sum() + amb[:, [0, 1, H, H + 1], :].sum())
    assert abs(int(got.sum()) - int(ref.sum())) <= border
    return int(diff.sum()), int(amb.sum())


@pytest.mark.parametrize("axes,W,H,hw", [((0, 1), 256, 256, 3.0), ((0, 2), 640, 360, 2.5), ((2, 1), 33, 77, 0.7),
                                          ((1, 0), 2048, 2048, 1.5)])
def test_splat_matches_the_definition_and_the_float32_recipe(nb, axes, W, H, hw):
    """f4 two ways: (i) against the fp64 definition, up to the elements within float32 rounding of a pixel edge;
    (ii) bit-exact against the float32 recipe (the same roundings in the same order)."""
    w = make_config(3)
    s = _sim(nb, w)
    centre = [0.4, -0.1, 0.05]
    img = s.splat(centre, hw, axes[0], axes[1], W, H)
    s.synchronize()
    got = img.cpu().numpy().astype(np.int64)
    moved, amb = _splat_vs_definition(got, w.posm, w.star, centre, hw, axes, W, H)
    assert amb < 0.01 * w.n and moved <= 2 * amb          # a sliver of the elements is ambiguous at all
    ref = oracle.splat(w.posm, w.star, centre, hw, axes[0], axes[1], W, H)
    assert got.shape == ref.shape and np.array_equal(got, ref.astype(np.int64))
    if hw >= 2.5:
        assert got.sum() > 0.9 * w.n
    s.step(2)                                        # the image follows the state
    img2 = s.splat(centre, hw, axes[0], axes[1], W, H)
    s.synchronize()
    x = s.posm.cpu().numpy()
    got2 = img2.cpu().numpy().astype(np.int64)
    _splat_vs_definition(got2, x, w.star, centre, hw, axes, W, H)
    assert np.array_equal(got2, oracle.splat(x, w.star, centre, hw, axes[0], axes[1], W, H).astype(np.int64))
    s.close()


def test_splat_elements_placed_on_pixel_edges(nb):
    """Elements put on purpose within a hair of pixel edges: the kernel may differ from the definition, but only
    inside the allowance; away from edges it must not differ at all."""
    rng = np.random.default_rng(12)
    n, W, H, hw, centre = 6000, 96, 64, 2.0, [0.125, 0.0, -0.25]
    posm = np.zeros((n, 4), np.float32); posm[:, 3] = 1.0 / n
    k = rng.integers(0, W, n)
    posm[:, 0] = (centre[0] - hw + k * (2 * hw / W) + rng.uniform(-3e-7, 3e-7, n)).astype(np.float32)
    posm[:, 1] = rng.uniform(-1.0, 1.0, n).astype(np.float32)
    posm[:, 2] = rng.uniform(-1.0, 1.0, n).astype(np.float32)
    star = (np.arange(n) >= n // 2).astype(np.int32)
    p = params_f32(make_config(1, scale=0.125).params)
    s = nb.Simulation(posm, np.zeros_like(posm), star, p)
    got = s.splat(centre, hw, 0, 2, W, H).cpu().numpy().astype(np.int64)
    _, amb = _splat_vs_definition(got, posm, star, centre, hw, (0, 2), W, H)
    assert amb > n // 4
    got = s.splat(centre, hw, 1, 2, W, H).cpu().numpy().astype(np.int64)          # the same elements, uniform in y
    moved, amb = _splat_vs_definition(got, posm, star, centre, hw, (1, 2), W, H)
    assert moved <= 2 * amb and amb < 20
    s.close()


def test_splat_argument_errors(nb):
    import torch
    import ctypes as C
    s = _sim(nb, make_config(1, scale=0.125))
    img = torch.zeros((2, 8, 8), dtype=torch.int32, device="cuda")
    c3 = (C.c_float * 3)(0, 0, 0)
    L = nb.lib()
    assert L.nb_splat(s.ctx, c3, 1.0, 0, 0, 8, 8, img.data_ptr()) == nb.NB_EINVAL      # same axis twice
    assert L.nb_splat(s.ctx, c3, 0.0, 0, 1, 8, 8, img.data_ptr()) == nb.NB_EINVAL
    assert L.nb_splat(s.ctx, c3, 1.0, 0, 3, 8, 8, img.data_ptr()) == nb.NB_EINVAL
    assert L.nb_splat(s.ctx, c3, 1.0, 0, 1, 0, 8, img.data_ptr()) == nb.NB_EINVAL
    assert L.nb_splat(s.ctx, None, 1.0, 0, 1, 8, 8, img.data_ptr()) == nb.NB_EINVAL
    assert L.nb_splat(s.ctx, c3, 1.0, 0, 1, 8, 8, None) == nb.NB_EINVAL
    assert L.nb_splat(s.ctx, c3, 1.0, 0, 1, 8, 8, img.data_ptr()) == nb.NB_OK
    s.close()


# ------------------------------------------------------------------ bench.py contract on the GPU
def test_bench_line_has_the_contract_keys(nb):
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--steps", "3", "--warmup", "3",
                          "--no-cpu-baseline"], capture_output=True, text=True, cwd=root, timeout=900)
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads(out.stdout.strip().splitlines()[-1])
    assert d["unit"] == "interactions/s" and d["n_gpus"] == 1 and d["steps"] == 3 and d["warmup"] == 3
    assert d["higher_is_better"] is True and d["dtype"] == "f32" and d["data"] == "synthetic" and d["vs_baseline"] is None
    assert d["config"]["workload"].startswith("config4") and d["config"]["n"] == 262144
    assert d["value"] > 1e12 and abs(d["value"] - 262144.0 ** 2 / (d["ms_per_step"] * 1e-3)) < 1e-6 * d["value"]
    assert d["ms_per_step_best"] <= d["ms_per_step_median"] <= 1.2 * d["ms_per_step"]
    assert abs(d["pct_of_fp32_peak_20flop"] / d["pct_of_fp32_peak"] - 20.0 / 21.0) < 1e-9
    r = d["roofline"]
    # frac is what the ALUs executed (< 1); the algorithmic 21-flop figure sits beside it and may reach 1
    assert r["bound"] == "alu" and r["unit"] == "TFLOP/s" and 0.3 < r["frac"] < 0.9 and r["frac"] < r["frac_algorithmic"] < 1.2
    assert r["traffic_model"]["mode"] == "chain" and r["traffic_model"]["slab_bytes_written"] == 0      # the plan that ran
    assert "fma_pipe_frac" not in r and (r["traffic"] is None or 1e6 < r["traffic"] < 1e9)
    assert r["kernel"].startswith("nb_gravity_sym_chain_kernel<1024") and 0.9 < r["kernel_share_of_step"] <= 1.0
    assert abs(r["achieved"] / r["peak"] - r["frac"]) < 1e-9
    assert r["traffic"] is None or r["traffic"] > 0
    e = d["e2e"]
    assert e["h2d_bytes_per_step"] == e["d2h_bytes_per_step"] == 3 * 262144 * 16 and 0 < e["value"] < d["value"]
    assert d["gpu_launches"] >= 3 * 3 and d["clocks"]["sm_mhz"] > 0
    pc = {c["workload"].split("_")[0]: c for c in d["per_config"]}
    assert sorted(pc) == ["config1", "config2", "config3", "config5"]
    for c in pc.values():
        assert c["ms_per_step_best"] <= c["ms_per_step_median"] and c["interactions_per_s"] > 1e10 and c["ms_per_step_hot"] > 0
        assert abs(c["interactions_per_s"] - float(c["n"]) ** 2 / (c["ms_per_step"] * 1e-3)) < 1e-6 * c["interactions_per_s"]
    assert pc["config1"]["fused_one_launch"] and "sym" in pc["config3"]["kernel"] and "sym" in pc["config5"]["kernel"]


# ------------------------------------------------------------------ f3 per step, on the device (nb_transfer_record)
def _displaced_config3(scale):
    """Config 3's recipe with part of the donor moved toward and past the accretor and the ramp compressed: every
    column of the record is non-trivial and changes from step to step."""
    w = make_config(3, scale=scale)
    w.params["n_ramp"] = 8
    rng = np.random.default_rng(5)
    m = w.n // 20
    w.posm[:m, :3] += np.float32([1.3, 0.05, 0.0]) + rng.normal(0, 0.4, (m, 3)).astype(np.float32)
    w.posm[m:2 * m, 2] += np.float32(3.0)
    return w


def _compare_record(row, o, M):
    for k, f in enumerate(("M0", "M1", "a", "d0", "rL0", "rL1")):
        assert row[k] == pytest.approx(o[f], rel=1e-12), f
    assert np.allclose(row[18:24].reshape(2, 3), o["X"], rtol=0, atol=1e-12)
    assert np.allclose(row[24:30].reshape(2, 3), o["V"], rtol=0, atol=1e-12)
    slack = o["ambiguous"] + 1e-12 * M
    for k, f in enumerate(("Mcross0", "Mcross1", "Min0", "Min1", "Mout0", "Mout1")):
        assert abs(row[6 + k] - o[f]) <= slack, (f, row[6 + k], o[f])
    Lscale = max(np.abs(o["Ldisk"]).max(), 1e-300)
    assert np.abs(row[12:18].reshape(2, 3) - o["Ldisk"]).max() <= 1e-11 * Lscale + slack * 10


@pytest.mark.parametrize("scale,k", [(0.125, 0.6), (0.03, 0.69)])       # 8,192 (symmetric kernel + cell list) and 1,966 (fused) elements
def test_transfer_record_every_step_without_host_synchronisation(nb, scale, k):
    """nb_step(1) + nb_transfer_record in a loop with nothing synchronising in between: row n of the device series is
    the record of the state after n steps.  Each row against the oracle's transfer_diagnostics of that state (the
    states come from a second, identical and deterministic run that is read back step by step)."""
    import torch
    w = _displaced_config3(scale)
    p = params_f32(w.params)
    nsteps = 10
    s = nb.Simulation(w.posm, w.vel, w.star, p)
    series = torch.full((nsteps + 3, 32), float("nan"), dtype=torch.float64, device=s.device)
    s.transfer_record(series, k)
    for _ in range(nsteps):
        s.step(1)
        s.transfer_record(series, k)
    s.synchronize()
    rec = series.cpu().numpy()
    last = s.transfer_diagnostics(k)
    s.close()
    assert np.isnan(rec[nsteps + 1:]).all() and np.isfinite(rec[:nsteps + 1]).all()       # rows the run did not visit stay
    assert np.array_equal(rec[:nsteps + 1, 30], np.arange(nsteps + 1)) and (rec[:nsteps + 1, 31] == 0).all()
    assert rec[nsteps, 6] == last["Mcross0"] and rec[nsteps, 3] == last["d0"]           # the host call is the same record
    ref = nb.Simulation(w.posm, w.vel, w.star, p)
    M = float(w.posm[:, 3].astype(np.float64).sum())
    for n in range(nsteps + 1):
        if n:
            ref.step(1)
        ref.synchronize()
        x, v = ref.posm.cpu().numpy(), ref.vel.cpu().numpy()
        o = oracle.transfer_diagnostics(x, v, x[:, 3], w.star, k, band=1e-9)
        _compare_record(rec[n], o, M)
    ref.close()
    assert rec[0, 6] > 0 and rec[0, 8] > 0 and rec[0, 10] > 0                            # non-trivial columns ...
    assert len(set(rec[:nsteps + 1, 14])) > 3 and len(set(rec[:nsteps + 1, 18])) > 3     # ... that move from step to step (Ldisk, X0)


def test_transfer_record_in_a_cuda_graph_and_past_the_last_row(nb):
    """The step + record pair captured once and replayed: the same series as the eager loop, bit for bit; a run
    past the last row writes nothing."""
    import torch
    w = _displaced_config3(0.125)
    p = params_f32(w.params)
    eager = nb.Simulation(w.posm, w.vel, w.star, p)
    se = torch.zeros((6, 32), dtype=torch.float64, device=eager.device)
    eager.step(1)
    for _ in range(7):                                   # steps 2..8: rows 2..5 written, 6..8 dropped
        eager.step(1)
        eager.transfer_record(se)
    eager.synchronize()
    st = torch.cuda.Stream()
    cap = nb.Simulation(w.posm, w.vel, w.star, p, stream=st)
    sc = torch.zeros((6, 32), dtype=torch.float64, device=cap.device)
    cap.step(1); cap.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=st):
        cap.step(1)
        cap.transfer_record(sc)
    for _ in range(7):
        g.replay()
    torch.cuda.synchronize()
    assert torch.equal(se, sc) and torch.equal(eager.posm, cap.posm)
    assert (se[:2] == 0).all() and (se[2:, 0] > 0).all() and se[5, 30] == 5
    assert nb.nb_get_step(cap.ctx)[0] == 8
    L = nb.lib()
    assert L.nb_transfer_record(cap.ctx, 0.6, None, 4) == nb.NB_EINVAL
    assert L.nb_transfer_record(cap.ctx, 0.6, sc.data_ptr(), 0) == nb.NB_EINVAL
    assert L.nb_transfer_record(cap.ctx, -1.0, sc.data_ptr(), 4) == nb.NB_EINVAL
    eager.close(); cap.close()


def test_transfer_series_of_the_full_config3_run(nb):
    """SURVEY 8(f) f3 on BASELINE's config 3 (N = 65,536, 1,000 steps, the donor's radius ramped to its Roche lobe,
    PAPER.md:89, 107-109): one record per step, nothing synchronising until the end.  The series is complete and
    consistent -- step column, constant star masses, the last row equal to the host call -- and the donor's mass beyond
    the L1 plane at the end of the ramp is at least what it was at the start.  Prints the series at every 100th step."""
    import torch
    w = make_config(3)
    p = params_f32(w.params)
    nsteps = w.meta["nsteps"]
    s = nb.Simulation(w.posm, w.vel, w.star, p)
    series = torch.full((nsteps + 1, 32), float("nan"), dtype=torch.float64, device=s.device)
    s.transfer_record(series)
    for _ in range(nsteps):
        s.step(1)
        s.transfer_record(series)
    s.synchronize()
    rec = series.cpu().numpy()
    last = s.transfer_diagnostics()
    s.close()
    assert np.isfinite(rec).all() and np.array_equal(rec[:, 30], np.arange(nsteps + 1))
    assert np.allclose(rec[:, 0], rec[0, 0], rtol=1e-12, atol=0) and np.allclose(rec[:, 1], rec[0, 1], rtol=1e-12, atol=0)
    assert rec[-1, 6] == last["Mcross0"] and rec[-1, 8] == last["Min0"] and rec[-1, 2] == last["a"]
    assert rec[-1, 6] >= rec[0, 6]
    assert (np.abs(np.diff(rec[:, 2])) < 1e-3 * rec[0, 2]).all()                     # the separation moves smoothly
    for n in range(0, nsteps + 1, 100):
        print(f"TRANSFER config3 step={n} a={rec[n, 2]:.6f} d0={rec[n, 3]:.6f} rL0={rec[n, 4]:.6f} "
              f"Mcross0={rec[n, 6]:.6e} Min0={rec[n, 8]:.6e} Mout0={rec[n, 10]:.6e}")

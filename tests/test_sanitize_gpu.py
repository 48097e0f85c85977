"""A small pass over EVERY kernel of the library, sized so that it also finishes under
`compute-sanitizer --tool memcheck` and `--tool racecheck` (the command lines and their
summaries are in profiles/r2_sanitizers.md).  Run plainly it is one more parity test: both gravity kernels
(ragged sizes: padding elements, a star boundary inside a tile), the cell-list contact pass (dense overlaps:
queue overflow, both grids, the wrapped table), the index-order contact pass, the fused small-n kernel, the
update kernel with the radius ramp, nb_relax, nb_energy, nb_transfer_diagnostics, nb_splat, nb_set_step."""
import numpy as np
import pytest

import oracle
from workloads import make_binary, make_config, params_f32

pytestmark = pytest.mark.gpu


def _w(n1, n2, seed, **over):
    kw = dict(name="s", seed=seed, n1=n1, n2=n2, shape="uniform", radius1=1.0, radius2=0.6, q=0.5, a=1.5, eps=0.01,
              dt=1e-3, nsteps=0, ramp_factor1=1.2, n_ramp=4)
    kw.update(over)
    return make_binary(**kw)


def _accel_ok(nb, w, p, **kw):
    s = nb.Simulation(w.posm, w.vel, w.star, p, **kw)
    a = s.compute_accel().cpu().numpy().astype(np.float64)[:, :3]
    name = nb.nb_force_kernel_name(s.ctx)
    s.close()
    ao, _, dl = oracle.accel(w.posm, w.vel, w.posm[:, 3], w.star, p["R_start"], p, want_diag=True)
    err = np.maximum(np.linalg.norm(a - ao, axis=1) - dl, 0.0) / np.linalg.norm(ao, axis=1)
    assert err.max() <= 2e-5, (name, err.max())
    return name


def test_every_force_kernel_small():
    import paper_2303_12166_b200 as nb
    w = _w(1500, 1237, 3)                                   # overlapping stars: cross-star contacts as well
    p = params_f32(w.params)
    assert "nb_fused_step_kernel" in _accel_ok(nb, w, p)                                    # fused small-n kernel
    assert "sym_kernel<256" in _accel_ok(nb, w, p, force_path=nb.NB_PATH_SYMMETRIC)         # + index-order contact pass
    w = _w(5000, 4321, 4)                                   # n >= 8,192: cell list; one-sided and symmetric kernels
    p = params_f32(w.params)
    assert "nb_gravity_kernel<2,128>" in _accel_ok(nb, w, p, force_path=nb.NB_PATH_ONE_SIDED)
    assert "sym_kernel<256" in _accel_ok(nb, w, p, force_path=nb.NB_PATH_SYMMETRIC)
    w = _w(6000, 4500, 5)                                   # dense: ~60 contacts per element, the hit queues overflow
    w.params["R_start"] = (0.1, 0.08); w.params["R_end"] = (0.12, 0.08); w.params["gamma"] = 5.0
    _accel_ok(nb, w, params_f32(w.params))
    w = _w(300, 212, 6, mass_sigma=0.2)                     # every element its own mass: the general-mass loops
    _accel_ok(nb, w, params_f32(dict(w.params)))
    _accel_ok(nb, w, params_f32(dict(w.params)), force_path=nb.NB_PATH_SYMMETRIC)


@pytest.mark.parametrize("n1,n2,path", [(700, 500, 0), (5200, 3100, 0), (5200, 3100, 2)])
def test_steps_relax_and_diagnostics_small(n1, n2, path):
    import paper_2303_12166_b200 as nb
    w = _w(n1, n2, 7)
    p = params_f32(w.params)
    s = nb.Simulation(w.posm, w.vel, w.star, p, force_path=path)
    s.step(3); s.relax(2, 5.0); s.step(1)
    s.synchronize()
    o = oracle.Sim(w.posm, w.vel, w.star, p)
    o.step(3); o.relax(2, 5.0); o.step(1)
    x = s.posm.cpu().numpy().astype(np.float64)[:, :3]
    assert np.linalg.norm(x - o.x, axis=1).max() / w.meta["a"] <= 1e-4
    step, R = nb.nb_get_step(s.ctx)
    assert step == 6 and np.array_equal(np.asarray(R, np.float64), o.radii())
    e, oe = s.energy(), oracle.Sim(s.posm.cpu().numpy(), s.vel.cpu().numpy(), w.star, p)
    oe.n = 6
    oe = oe.energy()
    for k in ("KE", "Ug", "Urep", "E"):
        assert e[k] == pytest.approx(oe[k], rel=2e-6, abs=1e-12), k
    t = s.transfer_diagnostics()
    ot = oracle.transfer_diagnostics(s.posm.cpu().numpy(), s.vel.cpu().numpy(), w.posm[:, 3], w.star, band=1e-9)
    assert abs(t["Mcross0"] - ot["Mcross0"]) <= ot["ambiguous"] + 1e-12 and t["a"] == pytest.approx(ot["a"], rel=1e-12)
    img = s.splat([0.0, 0.0, 0.0], 2.0, 0, 1, 64, 48).cpu().numpy().astype(np.int64)
    assert np.array_equal(img, oracle.splat(s.posm.cpu().numpy(), w.star, [0.0, 0.0, 0.0], 2.0, 0, 1, 64, 48).astype(np.int64))
    nb.nb_set_step(s.ctx, 2)
    assert nb.nb_get_step(s.ctx)[0] == 2
    s.close()


@pytest.mark.parametrize("n1,n2,path", [(700, 501, 0), (5200, 3101, 1), (5200, 3101, 2), (33, 0, 0)])
def test_no_write_outside_the_callers_buffers(n1, n2, path):
    """compute-sanitizer is closed on this pool (profiles/r2_sanitizers.md), so the library's writes are fenced in by
    hand: every buffer it is given -- state, star, output, workspace, image -- is carved out of ONE allocation with 4 KB
    guard zones of a known byte pattern on both sides, every entry point runs, and the guards must come back intact."""
    import torch
    import paper_2303_12166_b200 as nb
    w = _w(max(n1, 1), max(n2, 1), 11)
    n = n1 + n2
    posm_h, vel_h, star_h = w.posm[:n].copy(), w.vel[:n].copy(), w.star[:n].copy()
    p = params_f32(w.params)
    dev = torch.device("cuda:0")
    G, W, H = 4096, 40, 24
    sizes = dict(posm=n * 16, vel=n * 16, star=n * 4, acc=n * 16, ws=nb.nb_workspace_bytes(n), img=2 * W * H * 4)
    off, o = {}, G
    for k, b in sizes.items():
        o = (o + 255) // 256 * 256
        off[k] = o
        o += b + G
    buf = torch.full((o + 256,), 0xA5, dtype=torch.uint8, device=dev)
    base = (buf.data_ptr() + 255) // 256 * 256 - buf.data_ptr()          # 256-byte aligned start inside the tensor
    view = lambda k: buf[base + off[k]: base + off[k] + sizes[k]]
    view("posm").copy_(torch.as_tensor(posm_h).view(torch.uint8).reshape(-1))
    view("vel").copy_(torch.as_tensor(vel_h).view(torch.uint8).reshape(-1))
    view("star").copy_(torch.as_tensor(star_h).view(torch.uint8).reshape(-1))
    ptr = lambda k: buf.data_ptr() + base + off[k]
    ctx = nb.nb_create(n, p, torch.cuda.current_stream(dev).cuda_stream)
    if path:
        nb.nb_set_force_path(ctx, path)
    nb.nb_set_state(ctx, n, ptr("posm"), ptr("vel"), ptr("star"), ptr("ws"), sizes["ws"])
    nb.nb_compute_accel(ctx, ptr("acc"))
    nb.nb_step(ctx, 3)
    nb.nb_relax(ctx, 1, 2.0)
    nb.nb_energy(ctx)
    nb.nb_transfer_diagnostics(ctx)
    nb.nb_splat(ctx, [0.0, 0.0, 0.0], 2.0, 0, 1, W, H, ptr("img"))
    nb.nb_set_step(ctx, 1)
    nb.nb_time_force_kernel(ctx, 1); nb.nb_time_contact_pass(ctx, 1)
    torch.cuda.synchronize()
    nb.nb_destroy(ctx)
    inside = torch.zeros(buf.numel(), dtype=torch.bool, device=dev)
    for k in sizes:
        inside[base + off[k]: base + off[k] + sizes[k]] = True
    assert bool((buf[~inside] == 0xA5).all()), "a kernel wrote outside the buffers it was given"
    x = view("posm").view(torch.float32).reshape(n, 4)
    assert bool(torch.isfinite(x).all()) and int(view("img").view(torch.int32).sum()) <= n

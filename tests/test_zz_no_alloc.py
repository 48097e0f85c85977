"""nb_gravity_accel_static(): the entry point for callers that cannot allocate device memory.

Who that is: a plug-in inside a host application that passes it the state arrays but keeps the allocator, a
process whose device memory is fully assigned up front, a loop that may not take cudaMalloc's device-wide
stall.  They can provide neither the workspace nb_set_state() wants nor the stream and events nb_create()
makes, so this call takes inputs and an output only; the gravity kernel's partial sums go to a 2 MiB array
built into libnb.so (one per device, shared by all calls, never cleared).

What is checked: its accelerations (Eq. 4) against the existing ctx path (nb_compute_accel with
gamma = 0) on the same device arrays, to the acceleration tolerance of the other GPU tests, on two calls in a
row that use the shared array differently (so the second one starts on the first one's leftovers); and that a
size beyond the fixed array is refused with its own status.  The file sorts last on purpose: `pytest -x` stops
at the first failure, and a failure here must not hide the parity tests.
"""
import numpy as np
import pytest

from workloads import make_config, params_f32

pytestmark = pytest.mark.gpu

ACC_TOL = 2.0e-5          # the bar of tests/test_parity_gpu.py: max |da_i| / |a_i|


def _existing_path(nb, w, p):
    """Gravity accelerations by the ctx API (workspace from torch); returns the device arrays too."""
    p0 = dict(p, gamma=0.0)
    sim = nb.Simulation(w.posm, w.vel, w.star, p0)
    a = sim.compute_accel()
    sim.synchronize()
    ref = a.cpu().numpy().astype(np.float64)[:, :3]
    return sim, ref


def _rel(a, ref):
    an = np.linalg.norm(ref, axis=1)
    assert (an > 0).all()
    return (np.linalg.norm(a - ref, axis=1) / an).max()


def test_static_scratch_entry_point_matches_the_ctx_path_on_two_calls_in_a_row(nb):
    import torch
    assert nb.nb_gravity_accel_static_max_n() == 16384
    # call 1: config 2 at full size (n = 16384 = the limit, lognormal masses: general-mass loop, 8 splits fill the
    # array); call 2: config 1 cut to a ragged n (758 elements, one mass per star, fewer and shorter slabs that
    # land on call 1's leftovers); call 3: call 1's input again, after call 2 overwrote part of the array.
    cases = [make_config(2), make_config(1, scale=0.37), make_config(2)]
    assert cases[0].n == 16384 and cases[1].n % 256 != 0
    stream = torch.cuda.current_stream()
    got, want = [], []
    sims = []
    for w in cases:                                   # references first: the static calls then run back to back
        sim, ref = _existing_path(nb, w, params_f32(w.params))
        sims.append(sim)
        want.append(ref)
    outs = [torch.full((w.n, 4), float("nan"), dtype=torch.float32, device="cuda:0") for w in cases]
    for w, sim, out in zip(cases, sims, outs):        # no synchronisation in between: same stream, in order
        p = params_f32(w.params)
        nb.nb_gravity_accel_static(w.n, sim.posm, p["G"], p["eps"], out, stream.cuda_stream)
    stream.synchronize()
    for w, out, ref in zip(cases, outs, want):
        o = out.cpu().numpy().astype(np.float64)
        assert np.isfinite(o).all() and (o[:, 3] == 0).all()
        rel = _rel(o[:, :3], ref)
        print(f"PARITY static-scratch accel {w.name} n={w.n} max_rel_vs_ctx_path={rel:.3e}")
        assert rel <= ACC_TOL
        got.append(o)
    # the same input gives the same bits whatever the array held before (fixed summation order)
    assert np.array_equal(got[0], got[2])
    for sim in sims:
        sim.close()


def test_static_scratch_entry_point_refuses_what_the_fixed_array_cannot_hold(nb):
    import torch
    nmax = nb.nb_gravity_accel_static_max_n()
    x = torch.zeros((nmax + 1, 4), dtype=torch.float32, device="cuda:0")
    a = torch.zeros_like(x)
    with pytest.raises(nb.NbError) as e:
        nb.nb_gravity_accel_static(nmax + 1, x, 1.0, 0.01, a)
    assert e.value.status == nb.NB_ESIZE and "nb_gravity_accel_static_max_n" in str(e.value)
    for bad in (dict(n=0), dict(G=-1.0), dict(eps=float("nan"))):
        kw = dict(n=8, G=1.0, eps=0.01)
        kw.update(bad)
        with pytest.raises(nb.NbError) as e:
            nb.nb_gravity_accel_static(kw["n"], x, kw["G"], kw["eps"], a)
        assert e.value.status == nb.NB_EINVAL
    with pytest.raises(nb.NbError) as e:                               # float4 loads need 16-byte alignment
        nb.nb_gravity_accel_static(8, x.data_ptr() + 4, 1.0, 0.01, a)
    assert e.value.status == nb.NB_EINVAL
    # a single element: no pair, zero acceleration
    one = torch.tensor([[1.0, 2.0, 3.0, 0.5]], dtype=torch.float32, device="cuda:0")
    out = torch.full((1, 4), 7.0, dtype=torch.float32, device="cuda:0")
    nb.nb_gravity_accel_static(1, one, 1.0, 0.01, out)
    torch.cuda.synchronize()
    assert (out.cpu().numpy() == 0).all()

"""B200-native all-pairs binary-star element model (arXiv 2303.12166 hot path).

Thin ctypes binding of the C ABI in include/nb.h: the functions below have the
same names as the C entry points and only marshal arguments (torch tensors ->
device pointers).  Every step of the path runs in the sm_100a CUDA kernels of
csrc/; PyTorch is used for device memory and streams only.  There is no CPU
fallback: if libnb.so is missing or no sm_100 device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional, Sequence

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("NB_LIB_PATH") or os.path.join(HERE, "libnb.so")   # override: development only

NB_OK, NB_EINVAL, NB_ESTATE, NB_ECUDA, NB_ENOMEM, NB_EARCH, NB_ESIZE = 0, -1, -2, -3, -4, -5, -6
NB_PATH_AUTO, NB_PATH_ONE_SIDED, NB_PATH_SYMMETRIC = 0, 1, 2

EXPORTS = ("nb_create", "nb_workspace_bytes", "nb_set_state", "nb_compute_accel", "nb_step",
           "nb_energy", "nb_set_step", "nb_relax", "nb_transfer_diagnostics", "nb_transfer_record", "nb_splat", "nb_get_step", "nb_upload_state",
           "nb_download_state",
           "nb_get_launch_info", "nb_set_force_path", "nb_force_kernel_name", "nb_launch_count",
           "nb_time_force_kernel", "nb_time_contact_pass", "nb_contact_stats", "nb_destroy", "nb_strerror",
           "nb_last_cuda_error", "nb_roche_lobe_radius", "nb_l1_distance",
           "nb_gravity_accel_static", "nb_gravity_accel_static_max_n")


class nb_params(C.Structure):
    """Mirror of `nb_params` in include/nb.h."""
    _fields_ = [("G", C.c_float), ("eps", C.c_float), ("dt", C.c_float), ("q", C.c_float),
                ("gamma", C.c_float), ("beta", C.c_float),
                ("R_start", C.c_float * 2), ("R_end", C.c_float * 2),
                ("n_ramp", C.c_int32), ("v_dead", C.c_float), ("lens_mode", C.c_int32)]


class NbError(RuntimeError):
    def __init__(self, status: int, where: str, cuda: int = 0):
        self.status = status
        msg = f"{where}: {nb_strerror(status)} (status {status})"
        if status == NB_ECUDA:
            msg += f", cudaError_t={cuda}"
        super().__init__(msg)


_lib = None


def lib() -> C.CDLL:
    """Load libnb.so (built by paper_2303_12166_b200.build); raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2303_12166_b200.build` "
                "(nvcc, sm_100a).  There is no CPU fallback.")
        L = C.CDLL(LIB_PATH)
        vp, i64, i32 = C.c_void_p, C.c_int64, C.c_int32
        L.nb_create.restype = C.c_int
        L.nb_create.argtypes = [C.POINTER(vp), i64, C.POINTER(nb_params), vp]
        L.nb_workspace_bytes.restype = C.c_size_t
        L.nb_workspace_bytes.argtypes = [i64]
        L.nb_set_state.restype = C.c_int
        L.nb_set_state.argtypes = [vp, i64, vp, vp, vp, vp, C.c_size_t]
        L.nb_compute_accel.restype = C.c_int
        L.nb_compute_accel.argtypes = [vp, vp]
        L.nb_step.restype = C.c_int
        L.nb_step.argtypes = [vp, C.c_int]
        L.nb_energy.restype = C.c_int
        L.nb_energy.argtypes = [vp, C.POINTER(C.c_double)]
        L.nb_set_step.restype = C.c_int
        L.nb_set_step.argtypes = [vp, i64]
        L.nb_relax.restype = C.c_int
        L.nb_relax.argtypes = [vp, C.c_int, C.c_float]
        L.nb_transfer_diagnostics.restype = C.c_int
        L.nb_transfer_diagnostics.argtypes = [vp, C.c_double, C.POINTER(C.c_double)]
        L.nb_transfer_record.restype = C.c_int
        L.nb_transfer_record.argtypes = [vp, C.c_double, vp, i64]
        L.nb_splat.restype = C.c_int
        L.nb_splat.argtypes = [vp, C.POINTER(C.c_float), C.c_float, C.c_int, C.c_int, C.c_int, C.c_int, vp]
        L.nb_get_step.restype = C.c_int
        L.nb_get_step.argtypes = [vp, C.POINTER(i64), C.POINTER(C.c_float)]
        L.nb_upload_state.restype = C.c_int
        L.nb_upload_state.argtypes = [vp, vp, vp, vp]
        L.nb_download_state.restype = C.c_int
        L.nb_download_state.argtypes = [vp, vp, vp, vp]
        L.nb_get_launch_info.restype = C.c_int
        L.nb_get_launch_info.argtypes = [vp, C.POINTER(i32)]
        L.nb_set_force_path.restype = C.c_int
        L.nb_set_force_path.argtypes = [vp, C.c_int]
        L.nb_force_kernel_name.restype = C.c_char_p
        L.nb_force_kernel_name.argtypes = [vp]
        L.nb_launch_count.restype = i64
        L.nb_launch_count.argtypes = [vp]
        L.nb_time_force_kernel.restype = C.c_int
        L.nb_time_force_kernel.argtypes = [vp, C.c_int, C.POINTER(C.c_float)]
        L.nb_time_contact_pass.restype = C.c_int
        L.nb_time_contact_pass.argtypes = [vp, C.c_int, C.POINTER(C.c_float)]
        L.nb_contact_stats.restype = C.c_int
        L.nb_contact_stats.argtypes = [vp, C.POINTER(i64)]
        L.nb_destroy.restype = None
        L.nb_destroy.argtypes = [vp]
        L.nb_strerror.restype = C.c_char_p
        L.nb_strerror.argtypes = [C.c_int]
        L.nb_last_cuda_error.restype = C.c_int
        L.nb_last_cuda_error.argtypes = [vp]
        L.nb_roche_lobe_radius.restype = C.c_double
        L.nb_roche_lobe_radius.argtypes = [C.c_double, C.c_double]
        L.nb_l1_distance.restype = C.c_double
        L.nb_l1_distance.argtypes = [C.c_double]
        L.nb_gravity_accel_static.restype = C.c_int
        L.nb_gravity_accel_static.argtypes = [i64, vp, C.c_float, C.c_float, vp, vp, C.POINTER(C.c_int)]
        L.nb_gravity_accel_static_max_n.restype = i64
        L.nb_gravity_accel_static_max_n.argtypes = []
        _lib = L
    return _lib


def _ptr(t) -> Optional[int]:
    """Device/host address of a torch tensor, numpy array or raw int (None passes through)."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def make_params(p: Dict[str, object]) -> nb_params:
    """nb_params from a dict with the keys of workloads.Workload.params."""
    return nb_params(float(p["G"]), float(p["eps"]), float(p["dt"]), float(p["q"]),
                     float(p.get("gamma", 0.0)), float(p.get("beta", 1.0)),
                     (C.c_float * 2)(*[float(v) for v in p["R_start"]]),
                     (C.c_float * 2)(*[float(v) for v in p["R_end"]]),
                     int(p.get("n_ramp", 0)), float(p.get("v_dead", 0.0)), int(p.get("lens_mode", 0)))


def _check(rc: int, where: str, ctx=None) -> None:
    if rc != NB_OK:
        raise NbError(rc, where, lib().nb_last_cuda_error(ctx) if ctx else 0)


# ---- the C entry points, same names, argument marshalling only -------------------------------
def nb_strerror(status: int) -> str:
    return lib().nb_strerror(int(status)).decode()


def nb_workspace_bytes(n_max: int) -> int:
    return int(lib().nb_workspace_bytes(int(n_max)))


def nb_create(n_max: int, params, cuda_stream: int = 0) -> int:
    """Returns the ctx handle.  `cuda_stream`: raw cudaStream_t (torch stream .cuda_stream)."""
    prm = params if isinstance(params, nb_params) else make_params(params)
    ctx = C.c_void_p()
    _check(lib().nb_create(C.byref(ctx), int(n_max), C.byref(prm), C.c_void_p(cuda_stream or None)),
           "nb_create")
    return ctx.value


def nb_set_state(ctx: int, n: int, posm, vel, star, workspace, workspace_bytes: Optional[int] = None) -> None:
    if workspace_bytes is None:
        workspace_bytes = workspace.numel() * workspace.element_size()
    _check(lib().nb_set_state(ctx, int(n), _ptr(posm), _ptr(vel), _ptr(star), _ptr(workspace),
                              int(workspace_bytes)), "nb_set_state", ctx)


def nb_compute_accel(ctx: int, acc) -> None:
    _check(lib().nb_compute_accel(ctx, _ptr(acc)), "nb_compute_accel", ctx)


def nb_step(ctx: int, nsteps: int) -> None:
    _check(lib().nb_step(ctx, int(nsteps)), "nb_step", ctx)


def nb_energy(ctx: int) -> Dict[str, object]:
    out = (C.c_double * 12)()
    _check(lib().nb_energy(ctx, out), "nb_energy", ctx)
    v = list(out)
    return dict(KE=v[0], Ug=v[1], Urep=v[2], E=v[3], P=v[4:7], L=v[7:10], Fnet=v[10], step=int(v[11]))


def nb_set_step(ctx: int, step: int) -> None:
    _check(lib().nb_set_step(ctx, int(step)), "nb_set_step", ctx)


def nb_relax(ctx: int, nsteps: int, kappa: float) -> None:
    _check(lib().nb_relax(ctx, int(nsteps), float(kappa)), "nb_relax", ctx)


def nb_transfer_diagnostics(ctx: int, k_lobe: float = 0.6) -> Dict[str, object]:
    out = (C.c_double * 32)()
    _check(lib().nb_transfer_diagnostics(ctx, float(k_lobe), out), "nb_transfer_diagnostics", ctx)
    v = list(out)
    return dict(M0=v[0], M1=v[1], a=v[2], d0=v[3], rL0=v[4], rL1=v[5], Mcross0=v[6], Mcross1=v[7],
                Min0=v[8], Min1=v[9], Mout0=v[10], Mout1=v[11], Ldisk=[v[12:15], v[15:18]],
                X=[v[18:21], v[21:24]], V=[v[24:27], v[27:30]], step=int(v[30]))


TRANSFER_RECORD = ("M0", "M1", "a", "d0", "rL0", "rL1", "Mcross0", "Mcross1", "Min0", "Min1", "Mout0", "Mout1")   # columns 0..11


def nb_transfer_record(ctx: int, k_lobe: float, dev_series, rows: Optional[int] = None) -> None:
    """The record of nb_transfer_diagnostics into row `step count` of the DEVICE array dev_series [rows][32] (float64);
    asynchronous, no host synchronisation."""
    if rows is None:
        rows = dev_series.shape[0]
    _check(lib().nb_transfer_record(ctx, float(k_lobe), _ptr(dev_series), int(rows)), "nb_transfer_record", ctx)


def nb_splat(ctx: int, centre: Sequence[float], half_width: float, axis_u: int, axis_v: int, W: int, H: int,
             image) -> None:
    c3 = (C.c_float * 3)(*[float(x) for x in centre])
    _check(lib().nb_splat(ctx, c3, float(half_width), int(axis_u), int(axis_v), int(W), int(H), _ptr(image)),
           "nb_splat", ctx)


def write_ppm(path: str, image) -> None:
    """The headless stand-in for the paper's OpenGL window: the nb_splat() image
    `[2][H][W]` of element counts as a binary PPM (P6) file -- star 0 in the red channel, star 1 in the blue one,
    counts clipped at 255, row 0 (smallest v) at the bottom like a plot.  File output only: no arithmetic of the
    method happens here."""
    img = image.detach().cpu().numpy() if hasattr(image, "detach") else image
    if img.ndim != 3 or img.shape[0] != 2:
        raise ValueError("write_ppm expects the [2][H][W] image of nb_splat")
    import numpy as np
    H, W = int(img.shape[1]), int(img.shape[2])
    rgb = np.zeros((H, W, 3), dtype=np.uint8)
    rgb[..., 0] = np.minimum(img[0], 255)[::-1]
    rgb[..., 2] = np.minimum(img[1], 255)[::-1]
    with open(path, "wb") as f:
        f.write(b"P6\n%d %d\n255\n" % (W, H))
        f.write(rgb.tobytes())


def nb_get_step(ctx: int):
    step = C.c_int64()
    R = (C.c_float * 2)()
    _check(lib().nb_get_step(ctx, C.byref(step), R), "nb_get_step", ctx)
    return int(step.value), (float(R[0]), float(R[1]))


def nb_upload_state(ctx: int, host_posm, host_vel, host_acc=None) -> None:
    _check(lib().nb_upload_state(ctx, _ptr(host_posm), _ptr(host_vel), _ptr(host_acc)), "nb_upload_state", ctx)


def nb_download_state(ctx: int, host_posm, host_vel, host_acc=None) -> None:
    _check(lib().nb_download_state(ctx, _ptr(host_posm), _ptr(host_vel), _ptr(host_acc)),
           "nb_download_state", ctx)


def nb_get_launch_info(ctx: int) -> Dict[str, int]:
    out = (C.c_int32 * 4)()
    _check(lib().nb_get_launch_info(ctx, out), "nb_get_launch_info", ctx)
    return dict(i_per_cta=out[0], j_splits=out[1], force_ctas=out[2], update_ctas=out[3])


def nb_set_force_path(ctx: int, path: int) -> None:
    _check(lib().nb_set_force_path(ctx, int(path)), "nb_set_force_path", ctx)


def nb_force_kernel_name(ctx: int) -> str:
    return lib().nb_force_kernel_name(ctx).decode()


def nb_launch_count(ctx: int) -> int:
    return int(lib().nb_launch_count(ctx))


def nb_time_force_kernel(ctx: int, reps: int) -> float:
    ms = C.c_float()
    _check(lib().nb_time_force_kernel(ctx, int(reps), C.byref(ms)), "nb_time_force_kernel", ctx)
    return float(ms.value)


def nb_time_contact_pass(ctx: int, reps: int) -> float:
    ms = C.c_float()
    _check(lib().nb_time_contact_pass(ctx, int(reps), C.byref(ms)), "nb_time_contact_pass", ctx)
    return float(ms.value)


def nb_contact_stats(ctx: int) -> Dict[str, int]:
    out = (C.c_int64 * 2)()
    _check(lib().nb_contact_stats(ctx, out), "nb_contact_stats", ctx)
    return dict(candidates=int(out[0]), queued=int(out[1]))


def nb_destroy(ctx: int) -> None:
    lib().nb_destroy(ctx)


def nb_roche_lobe_radius(mass_ratio: float, k: float = 0.6) -> float:
    return float(lib().nb_roche_lobe_radius(float(mass_ratio), float(k)))


def nb_l1_distance(q: float) -> float:
    return float(lib().nb_l1_distance(float(q)))


def nb_gravity_accel_static_max_n() -> int:
    return int(lib().nb_gravity_accel_static_max_n())


def nb_gravity_accel_static(n: int, posm, G: float, eps: float, acc, cuda_stream: int = 0) -> None:
    """Eq. 4 accelerations of n <= nb_gravity_accel_static_max_n() elements into `acc` with no workspace and no ctx:
    for callers that cannot get device memory of their own (a plug-in inside a host application that owns the
    allocator, a fixed memory budget, a loop where cudaMalloc's device-wide stall is not acceptable).  The kernel's
    partial sums go to a 2 MiB array built into libnb.so, one per device and shared by every call on it: calls that
    overlap on a device corrupt each other, so keep them on one stream.  Make the first call on a device before any
    stream capture.  `posm`, `acc`: device float32 [n][4].  Raises NbError (NB_ESIZE beyond the limit)."""
    err = C.c_int(0)
    rc = lib().nb_gravity_accel_static(int(n), _ptr(posm), float(G), float(eps), _ptr(acc), C.c_void_p(cuda_stream or None),
                                       C.byref(err))
    if rc != NB_OK:
        raise NbError(rc, "nb_gravity_accel_static", err.value)


class Simulation:
    """Convenience owner of the device tensors one context borrows (torch allocates;
    the kernels of libnb.so do all the work)."""

    def __init__(self, posm, vel, star, params: Dict[str, object], device: str = "cuda:0",
                 stream=None, n_max: Optional[int] = None, force_path: int = NB_PATH_AUTO):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2303_12166_b200 needs a CUDA (sm_100) device; there is no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.params = dict(params)
        with torch.cuda.stream(self.stream):
            self.posm = torch.as_tensor(posm, dtype=torch.float32).contiguous().to(self.device, copy=True)
            self.vel = torch.as_tensor(vel, dtype=torch.float32).contiguous().to(self.device, copy=True)
            self.star = torch.as_tensor(star, dtype=torch.int32).contiguous().to(self.device, copy=True)
            self.n = int(self.posm.shape[0])
            self.n_max = int(n_max or self.n)
            self.workspace = torch.empty(nb_workspace_bytes(self.n_max), dtype=torch.uint8, device=self.device)
            self.acc = torch.zeros((self.n, 4), dtype=torch.float32, device=self.device)
        self.stream.synchronize()
        self.ctx = nb_create(self.n_max, self.params, self.stream.cuda_stream)
        if force_path != NB_PATH_AUTO:
            nb_set_force_path(self.ctx, force_path)
        nb_set_state(self.ctx, self.n, self.posm, self.vel, self.star, self.workspace)

    def compute_accel(self):
        nb_compute_accel(self.ctx, self.acc)
        return self.acc

    def step(self, nsteps: int = 1) -> None:
        nb_step(self.ctx, nsteps)

    def energy(self) -> Dict[str, object]:
        return nb_energy(self.ctx)

    def relax(self, nsteps: int, kappa: float) -> None:
        nb_relax(self.ctx, nsteps, kappa)

    def transfer_diagnostics(self, k_lobe: float = 0.6) -> Dict[str, object]:
        return nb_transfer_diagnostics(self.ctx, k_lobe)

    def transfer_record(self, series, k_lobe: float = 0.6) -> None:
        nb_transfer_record(self.ctx, k_lobe, series)

    def splat(self, centre, half_width: float, axis_u: int = 0, axis_v: int = 1, W: int = 512, H: int = 512):
        with self.torch.cuda.stream(self.stream):
            img = self.torch.empty((2, H, W), dtype=self.torch.int32, device=self.device)
        nb_splat(self.ctx, centre, half_width, axis_u, axis_v, W, H, img)
        return img

    def synchronize(self) -> None:
        self.stream.synchronize()

    def close(self) -> None:
        if getattr(self, "ctx", None):
            nb_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

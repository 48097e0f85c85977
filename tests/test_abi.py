"""Host-side checks of the boundary (no GPU): the C-ABI library builds, loads and
exports every symbol include/nb.h declares; the binding mirrors it; host helpers."""
import ctypes
import math
import os
import re

import pytest

import oracle
import paper_2303_12166_b200 as nb
from paper_2303_12166_b200 import build as nb_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _header_functions():
    src = open(os.path.join(ROOT, "include", "nb.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return re.findall(r"^\s*(?:const\s+)?(?:int|size_t|void|char\*|char|double|int64_t)\s*\*?\s*(nb_\w+)\s*\(", src, flags=re.M)


def test_library_builds_and_exports_every_declared_symbol():
    path = nb_build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    names = _header_functions()
    assert {"nb_create", "nb_set_state", "nb_compute_accel", "nb_step", "nb_energy", "nb_destroy"} <= set(names)
    for name in names:
        assert hasattr(lib, name), f"{name} declared in nb.h but not exported by libnb.so"
    assert set(names) == set(nb.EXPORTS), "python binding and nb.h disagree"


def test_params_struct_layout_matches_header():
    # 6 floats + 2x2 floats + int + float + int, all 4-byte: 13 * 4
    assert ctypes.sizeof(nb.nb_params) == 52
    p = nb.make_params(dict(G=1, eps=0.01, dt=1e-3, q=0.5, gamma=400, beta=0.5, R_start=(0.1, 0.2),
                            R_end=(0.3, 0.2), n_ramp=7, v_dead=1e-4, lens_mode=1))
    assert (p.n_ramp, p.lens_mode) == (7, 1) and p.R_end[0] == pytest.approx(0.3, rel=1e-7)


def test_sm100a_cubin_and_packed_fp32_in_the_force_kernel():
    import subprocess
    lib = nb_build.build()
    elf = subprocess.run(["cuobjdump", "-lelf", lib], capture_output=True, text=True).stdout
    assert "sm_100a" in elf
    sass = subprocess.run(["cuobjdump", "-sass", lib], capture_output=True, text=True).stdout
    assert "FFMA2" in sass and "MUFU.RSQ" in sass and "MUFU.RCP" in sass


def test_host_scalars_eq3_and_l1():
    # Eq. 3 -- literal values and the independent oracle implementation
    assert nb.nb_roche_lobe_radius(0.4, 0.6) == pytest.approx(0.303053, abs=1e-6)
    assert nb.nb_roche_lobe_radius(2.5, 0.6) == pytest.approx(0.459873, abs=1e-6)
    assert nb.nb_roche_lobe_radius(0.4, 0.69) == pytest.approx(0.287073, abs=1e-6)
    for q in (0.05, 0.3, 0.5, 1.0, 2.0, 10 / 3):
        assert nb.nb_roche_lobe_radius(q, 0.6) == pytest.approx(oracle.roche_lobe_radius(q, 0.6), rel=1e-13)
    for q, d in {0.3: 0.620867, 0.4: 0.592948, 0.6: 0.552343, 1.0: 0.5}.items():
        assert nb.nb_l1_distance(q) == pytest.approx(d, abs=1e-6)
        assert nb.nb_l1_distance(q) == pytest.approx(oracle.l1_distance(q), abs=1e-11)
    assert math.isnan(nb.nb_roche_lobe_radius(-1.0, 0.6)) and math.isnan(nb.nb_l1_distance(0.0))
    assert math.isnan(nb.nb_l1_distance(1.5))


def test_workspace_bytes_and_strerror():
    assert nb.nb_workspace_bytes(0) == 0 and nb.nb_workspace_bytes(-5) == 0
    assert nb.nb_workspace_bytes(1 << 40) == 0
    sizes = [nb.nb_workspace_bytes(n) for n in (1, 100, 2048, 16384, 65536, 262144, 1048576)]
    assert all(b > a for a, b in zip(sizes, sizes[1:]))
    assert all(s % 256 == 0 for s in sizes)
    assert sizes[-1] < 6e9                          # 1M elements: 4.7 GB (257 slabs of the symmetric kernel), 3 % of HBM
    assert nb.nb_workspace_bytes(1 << 26) < 100e9   # 67M elements: one-sided kernel only above 2M
    assert nb.nb_strerror(0) == "ok" and "argument" in nb.nb_strerror(-1)
    assert "sm_100" in nb.nb_strerror(-5) and "unknown" in nb.nb_strerror(-99)


def test_no_gpu_means_a_loud_error_not_a_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    prm = dict(G=1, eps=0.01, dt=1e-3, q=0.5, R_start=(0.1, 0.1), R_end=(0.1, 0.1))
    with pytest.raises(nb.NbError):
        nb.nb_create(128, prm)
    with pytest.raises(RuntimeError):
        import numpy as np
        nb.Simulation(np.zeros((4, 4), np.float32), np.zeros((4, 4), np.float32), np.zeros(4, np.int32), prm)


def test_product_and_oracle_do_not_import_each_other():
    pkg = os.path.join(ROOT, "paper_2303_12166_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "nb_oracle" not in text and "libnb_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2303_12166_b200" not in text.replace("imports nothing from paper_2303_12166_b200", "") \
                or f == "nb_oracle.c", f
            assert not re.search(r"^\s*(import|from)\s+paper_2303_12166_b200", text, flags=re.M), f
            assert '#include "nb' not in text
    wl = open(os.path.join(ROOT, "workloads", "configs.py")).read()
    assert "oracle" not in re.sub(r"#.*|\"\"\".*?\"\"\"", "", wl, flags=re.S) and "paper_2303" not in wl


def test_write_ppm_writes_the_splat_image_as_a_p6_file(tmp_path):
    """the headless image goes to a file (PPM) where the paper opens a window; host-side only."""
    import numpy as np
    import paper_2303_12166_b200 as nb
    img = np.zeros((2, 3, 4), dtype=np.int32)
    img[0, 0, 1] = 7          # star 0, bottom row
    img[1, 2, 3] = 300        # star 1, top row, clipped at 255
    path = tmp_path / "splat.ppm"
    nb.write_ppm(str(path), img)
    raw = path.read_bytes()
    assert raw.startswith(b"P6\n4 3\n255\n")
    px = np.frombuffer(raw[len(b"P6\n4 3\n255\n"):], dtype=np.uint8).reshape(3, 4, 3)
    assert px[2, 1].tolist() == [7, 0, 0] and px[0, 3].tolist() == [0, 0, 255] and px.sum() == 7 + 255
    import pytest
    with pytest.raises(ValueError):
        nb.write_ppm(str(path), np.zeros((3, 4), dtype=np.int32))

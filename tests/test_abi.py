"""-m "not gpu": the C-ABI library builds, loads without a GPU and exports every symbol include/*.h declares;
argument validation and the no-CPU-fallback rule are checked without any compute call."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "clvisc_hydro.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hydro_[a-z_]+)\s*\(", src)))


def test_header_symbols_are_exported():
    from paper_1802_04449_b200 import hydro
    lib = hydro.load_library()
    names = declared_symbols()
    assert set(names) == set(hydro.SYMBOLS), (names, hydro.SYMBOLS)
    for n in names:
        assert getattr(lib, n) is not None


def test_workspace_bytes_and_validation():
    from paper_1802_04449_b200 import hydro
    lib = hydro.load_library()
    g = hydro.make_grid(301, 301, 201, 0.1, 0.1, 0.08)
    w64, w32 = hydro.workspace_bytes(g, 64, 0.16), hydro.workspace_bytes(g, 32, 0.16)
    # 3 buffers x 19 fields x (10 x-blocks of 32) x 301 x 201 cells x 8 B, plus gstar, tables, diag
    cells_padded = 320 * 301 * 201
    assert w64 >= 3 * 19 * cells_padded * 8 and w64 < 3.2 * 19 * cells_padded * 8
    assert abs(w32 / w64 - 0.5) < 0.01
    assert hydro.workspace_bytes(g, 64, 0.0) < w64 / 2          # ideal: 9 fields per buffer
    assert hydro.workspace_bytes(hydro.make_grid(0, 4, 4, 1, 1, 1), 64, 0.0) == 0
    assert hydro.workspace_bytes(g, 16, 0.0) == 0
    assert lib.hydro_strerror(-2).decode().startswith("workspace")
    # NULL arguments are rejected before any CUDA call
    h = ctypes.c_void_p()
    assert lib.hydro_create(ctypes.byref(h), None, 0.01, 0.4, None, 0.0, None) == -1
    assert lib.hydro_step(None, 1) == -1 and lib.hydro_launch_count(None) == 0


def test_no_cpu_fallback():
    import torch
    from paper_1802_04449_b200 import Hydro, HydroError, inputs
    if torch.cuda.is_available():
        pytest.skip("GPU present: covered by the gpu tests")
    with pytest.raises(HydroError):
        Hydro(4, 4, 4, 0.1, 0.1, 0.1, 0.01, 0.6, inputs.conformal_eos(), 0.0)


def test_c_abi_create_without_device_returns_ecuda():
    # straight through the C ABI, no torch involved: valid arguments, a (never dereferenced) aligned workspace
    # pointer, but no CUDA device -> HYDRO_ECUDA (-3) and no context
    import torch
    from ctypes import byref, c_double, c_void_p, POINTER
    from paper_1802_04449_b200 import hydro
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    lib = hydro.load_library()
    g = hydro.make_grid(8, 8, 8, 0.1, 0.1, 0.1)
    e = hydro.hydro_eos(); e.kind, e.n, e.e_min, e.e_max, e.c_sb = 0, 0, 0.0, 0.0, 15.6
    o = hydro.hydro_opts()
    o.precision, o.minmod_theta, o.e_floor, o.pi_limit_xi, o.v_max = 64, 1.1, 1e-7, 1.0, 0.0
    o.workspace, o.workspace_bytes = c_void_p(1 << 20), hydro.workspace_bytes(g, 64, 0.1)
    h = c_void_p()
    assert lib.hydro_create(byref(h), byref(g), 0.01, 0.6, byref(e), 0.1, byref(o)) == -3
    assert not h.value
    o.workspace_bytes = 16                                       # too small is reported before the device check
    assert lib.hydro_create(byref(h), byref(g), 0.01, 0.6, byref(e), 0.1, byref(o)) == -2
    o.minmod_theta = 2.5
    assert lib.hydro_create(byref(h), byref(g), 0.01, 0.6, byref(e), 0.1, byref(o)) == -1


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1802_04449_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "clvisc_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1802_04449_b200" not in txt and "libclvisc_hydro" not in txt, f


@pytest.mark.gpu
def test_create_refuses_a_host_workspace():
    """hydro_create checks the workspace with cudaPointerGetAttributes: host memory is HYDRO_EINVAL, not a fault in a
    kernel later."""
    import numpy as np
    from ctypes import byref, c_void_p
    from paper_1802_04449_b200 import hydro
    lib = hydro.load_library()
    g = hydro.make_grid(8, 8, 8, 0.1, 0.1, 0.1)
    e = hydro.hydro_eos(); e.kind, e.n, e.e_min, e.e_max, e.c_sb = 0, 0, 0.0, 0.0, 15.6
    o = hydro.hydro_opts()
    o.precision, o.minmod_theta, o.e_floor, o.pi_limit_xi, o.v_max = 64, 1.1, 1e-7, 1.0, 0.0
    nbytes = hydro.workspace_bytes(g, 64, 0.1)
    host = np.zeros(nbytes + 256, dtype=np.uint8)
    base = (host.ctypes.data + 255) // 256 * 256
    o.workspace, o.workspace_bytes = c_void_p(base), nbytes
    h = c_void_p()
    assert lib.hydro_create(byref(h), byref(g), 0.01, 0.6, byref(e), 0.1, byref(o)) == -1
    assert not h.value


def test_eos_e_of_T_inverts_the_oracle_temperature(conformal, crossover):
    """hydro_eos_e_of_temperature (host arithmetic of the library, used for constant-T_f freeze-out) against the
    ORACLE's T(e): e -> T_oracle(e) -> e(T) must return e, inside the table, below it, above it and for EOSI."""
    import numpy as np
    from oracle import Oracle
    from paper_1802_04449_b200.hydro import eos_e_of_T
    for eos in (conformal, crossover):
        o = Oracle(1, 1, 1, 1, 1, 1, 0.1, 1.0, eos, 0.0)
        for e in (3e-5, 1e-4, 0.0123, 0.6, 5.0, 77.7, 999.0, 4000.0):
            T = o.eos(e)[2]
            assert abs(eos_e_of_T(eos, T) / e - 1) < 1e-10, (eos["kind"], e)
    # a temperature commonly used for the switch to hadrons sits in the crossover region of the synthetic table
    e137 = eos_e_of_T(crossover, 0.137)
    assert 0.05 < e137 < 2.0

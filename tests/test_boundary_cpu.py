"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol the header
declares, validates arguments and sizes, and refuses out-of-order calls.  No compute, no GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_2006_15698_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADERS = [os.path.join(ROOT, "include", f) for f in sorted(os.listdir(os.path.join(ROOT, "include"))) if f.endswith(".h")]


def declared_symbols():
    names = set()
    for header in HEADERS:
        text = re.sub(r"/\*.*?\*/", "", open(header).read(), flags=re.S)
        names |= set(re.findall(r"\b(dg_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


def test_library_exports_every_declared_symbol():
    lib = binding.load_library()
    names = declared_symbols()
    assert {"dg_create", "dg_set_state", "dg_residual", "dg_rk_step", "dg_get_state", "dg_destroy"} <= set(names)
    for name in names:
        assert hasattr(lib, name), name
    assert sorted(binding.SYMBOLS) == names          # the binding marshals exactly the header's calls


def _create(nx, ny, nz, p, gamma=1.4, extent=(1.0, 1.0, 1.0)):
    lib = binding.load_library()
    h = ctypes.c_void_p()
    ext = (ctypes.c_double * 3)(*extent)
    return lib, h, lib.dg_create(ctypes.byref(h), nx, ny, nz, p, gamma, ext)


def test_create_validates_arguments():
    for args, code in [((0, 1, 1, 1), 1), ((1, 1, 1, 0), 2), ((1, 1, 1, 8), 2), ((2, 2, 2, 3), 0)]:
        lib, h, rc = _create(*args)
        assert rc == code, args
        if rc == 0:
            lib.dg_destroy(h)
    assert _create(2, 2, 2, 1, gamma=1.0)[2] == 1
    assert _create(2, 2, 2, 1, extent=(1.0, 0.0, 1.0))[2] == 1
    assert _create(2, 2, 2, 1, extent=(1.0, float("nan"), 1.0))[2] == 1
    assert binding.load_library().dg_destroy(None) == 0


@pytest.mark.parametrize("nx,ny,nz,p", [(4, 4, 4, 1), (16, 16, 4, 3), (64, 64, 64, 4), (96, 96, 96, 7), (171, 171, 171, 1)])
def test_sizes(nx, ny, nz, p):
    lib, h, rc = _create(nx, ny, nz, p)
    assert rc == 0
    n = lib.dg_state_len(h)
    assert n == 5 * (p + 1) ** 3 * nx * ny * nz              # > 2^31 for config 5
    ws = lib.dg_workspace_bytes(h)
    info = (ctypes.c_longlong * 8)()
    assert lib.dg_kernel_info(h, info) == 0
    bx, by, bz, threads, smem, grid = info[0], info[1], info[2], info[3], info[4], info[5]
    assert grid == -(-nx // bx) * -(-ny // by) * -(-nz // bz)
    assert threads % 32 == 0 and threads <= 1024 and smem <= 227 * 1024
    assert ws >= 3 * 8 * n and ws < 8 * 8 * n + (1 << 20)     # Q, K, staging + traces, bounded
    lib.dg_destroy(h)


@pytest.mark.parametrize("p", range(1, 8))
def test_library_nodes_are_gauss_legendre(p):
    lib, h, rc = _create(2, 2, 2, p)
    xi, w = np.empty(p + 1), np.empty(p + 1)
    dp = ctypes.POINTER(ctypes.c_double)
    assert lib.dg_nodes(h, xi.ctypes.data_as(dp), w.ctypes.data_as(dp)) == 0
    x_np, w_np = np.polynomial.legendre.leggauss(p + 1)
    assert np.abs(xi - x_np).max() < 2e-15 and np.abs(w - w_np).max() < 2e-15
    lib.dg_destroy(h)


def test_calls_before_bind_are_refused_and_brick_knob():
    lib, h, rc = _create(4, 4, 4, 3)
    buf = np.zeros(lib.dg_state_len(h))
    for call in (lambda: lib.dg_set_state(h, buf.ctypes.data, 0), lambda: lib.dg_residual(h, buf.ctypes.data, 0),
                 lambda: lib.dg_rk_step(h, 1e-3, 1), lambda: lib.dg_get_state(h, buf.ctypes.data, 0)):
        assert call() == 5                                     # DG_ESTATE
    assert b"dg_bind" in lib.dg_last_error(h)
    assert lib.dg_rk_step(h, 1e-3, -1) == 1
    assert lib.dg_set_brick(h, 1, 1, 1) == 0
    info = (ctypes.c_longlong * 8)()
    lib.dg_kernel_info(h, info)
    assert tuple(info[0:3]) == (1, 1, 1) and info[5] == 64
    assert lib.dg_set_brick(h, 5, 5, 5) == 2                   # not compiled
    assert lib.dg_set_brick(h, 0, 0, 0) == 0
    assert lib.dg_bind(h, None, 0, None) == 1
    assert lib.dg_launch_count(h) == 0
    lib.dg_destroy(h)


def test_cfl_dt_is_the_rule_of_reading_r10():
    """dg_cfl_dt: cfl min(h) / ((2p+1) lam), host arithmetic of the library (no GPU)."""
    lib, h, rc = _create(8, 4, 5, 3, extent=(1.0, 0.9, 0.8))        # h = 0.125, 0.225, 0.16
    dt = ctypes.c_double(-1.0)
    assert lib.dg_cfl_dt(h, 0.1, 2.7, ctypes.byref(dt)) == 0
    want = 0.1 * 0.125 / (7 * 2.7)
    assert abs(dt.value - want) <= 4 * np.spacing(want)
    for cfl, lam in ((0.0, 2.7), (0.1, 0.0), (0.1, float("nan")), (float("inf"), 1.0), (-0.1, 1.0)):
        assert lib.dg_cfl_dt(h, cfl, lam, ctypes.byref(dt)) == 1
    assert lib.dg_cfl_dt(h, 0.1, 2.7, None) == 1 and lib.dg_cfl_dt(None, 0.1, 2.7, ctypes.byref(dt)) == 1
    hs = (ctypes.c_double * 3)(0.3, 0.05, 0.2)                       # dg_set_spacing overrides extent / n
    assert lib.dg_set_spacing(h, hs) == 0
    assert lib.dg_cfl_dt(h, 0.5, 1.0, ctypes.byref(dt)) == 0 and abs(dt.value - 0.5 * 0.05 / 7) <= 1e-17
    lib.dg_destroy(h)


def test_set_boundary_validates_its_arguments():
    lib, h, rc = _create(4, 4, 4, 2)
    IA, DA = ctypes.c_int * 6, ctypes.c_double * 5
    lib.dg_set_boundary.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_double)]
    assert lib.dg_set_boundary(h, IA(0, 0, 0, 0, 0, 0), None) == 0
    assert lib.dg_set_boundary(h, IA(1, 1, 0, 0, 1, 1), None) == 0                     # walls need no state
    assert lib.dg_set_boundary(h, IA(1, 0, 0, 0, 0, 0), None) == 1                     # periodic on one face only
    assert lib.dg_set_boundary(h, IA(4, 4, 0, 0, 0, 0), None) == 1
    assert lib.dg_set_boundary(h, IA(3, 1, 0, 0, 3, 3), None) == 0                     # halo faces (other contexts)
    assert lib.dg_halo_len(h, 0) == lib.dg_halo_len(h, 1) > 0 and lib.dg_halo_len(h, 6) == 0
    assert lib.dg_set_halo(h, 7, None) == 1
    assert lib.dg_set_boundary(h, IA(2, 2, 0, 0, 0, 0), None) == 1                     # far field without a state
    assert lib.dg_set_boundary(h, IA(2, 2, 0, 0, 0, 0), DA(1.0, 0.1, 0.0, 0.0, float("nan"))) == 1
    assert lib.dg_set_boundary(h, IA(2, 1, 0, 0, 0, 0), DA(1.0, 0.1, 0.0, 0.0, 2.5)) == 0
    assert lib.dg_set_boundary(h, None, None) == 1
    lib.dg_destroy(h)

"""Pins P7-P9 for the oracle's time stepping; CPU only.

The paper names the scheme ("Low-Storage Explicit Runge-Kutta 5-stage 4th-order (LSERK45)",
PAPER.md:254) without printing coefficients; R9 takes the Carpenter-Kennedy (5,4) 2N
set.  Pinned here by what any 4th-order 5-stage scheme must satisfy (the eight order conditions
in Butcher form), by the scheme's known stability polynomial, by re-evaluating one step in
Butcher form with the oracle's residual as right-hand side (pins the 2N-storage loop itself),
and by p+1 convergence to two exact solutions of the Euler equations.
"""
import math

import numpy as np
import pytest

import dg_bruteforce as bf
from oracle import Oracle
from paper_2006_15698_b200 import inputs as I

ORC = Oracle("fp64")
G = 1.4


def butcher(A, B):
    """2N-storage (A,B) -> Butcher (a, b, c).  K_s = A_s K_{s-1} + dt F(Y_s); Y_{s+1} = Y_s + B_s K_s."""
    s = len(A)
    coef = np.zeros((s, s))                # K_s = dt sum_j coef[s,j] F_j
    for i in range(s):
        coef[i, i] = 1.0
        if i > 0:
            coef[i, :i] = A[i] * coef[i - 1, :i]
    cum = np.cumsum(B[:, None] * coef, axis=0)   # Y_{i+1} = Y_0 + dt sum_j cum[i,j] F_j
    a = np.zeros((s, s))
    a[1:, :] = cum[:-1, :]
    b = cum[-1, :]
    return a, b, a.sum(1)


def test_lserk45_order_conditions_and_stability_polynomial():
    A, B = ORC.lserk45()
    assert A[0] == 0.0
    a, b, c = butcher(A, B)
    assert np.allclose(np.triu(a), 0.0)
    cond = {
        "b.1": (b.sum(), 1.0),
        "b.c": (b @ c, 1 / 2),
        "b.c2": (b @ c ** 2, 1 / 3),
        "b.Ac": (b @ (a @ c), 1 / 6),
        "b.c3": (b @ c ** 3, 1 / 4),
        "b.(c*Ac)": (b @ (c * (a @ c)), 1 / 8),
        "b.Ac2": (b @ (a @ c ** 2), 1 / 12),
        "b.AAc": (b @ (a @ (a @ c)), 1 / 24),
    }
    for name, (got, want) in cond.items():
        assert abs(got - want) < 5e-13, (name, got - want)     # rationals are given to ~13 digits
    one = np.ones(5)
    assert abs(b @ (a @ (a @ (a @ (a @ one)))) - 1.0 / 200.0) < 1e-12   # z^5 coefficient
    # abscissae printed with the scheme (C_s), recovered from (A,B)
    assert np.abs(c - np.array([0, .1496590219993, .3704009573644, .6222557631345, .9582821306748])).max() < 1e-12


def test_rk_step_equals_butcher_form_with_oracle_residual():
    c = I.CONFIGS["cfg1"]
    p, ext = c["p"], c["extent"]
    q0 = I.make_field("cfg1")
    dt = I.cfl_dt(ORC.max_wavespeed(q0, p, G), p, ext, (c["nx"], c["ny"], c["nz"]))
    a, b, _ = butcher(*ORC.lserk45())
    k = []
    for i in range(5):
        y = q0 + dt * sum(a[i, j] * k[j] for j in range(i)) if i else q0
        k.append(ORC.residual(y, p, G, ext))
    q1 = q0 + dt * sum(b[j] * k[j] for j in range(5))
    got = ORC.rk_step(q0, p, G, ext, dt, 1)
    assert np.abs(got - q1).max() < 5e-15 * np.abs(q1).max()
    # two steps of one == one call of two; zero steps is the identity
    assert np.array_equal(ORC.rk_step(got, p, G, ext, dt, 1), ORC.rk_step(q0, p, G, ext, dt, 2))
    assert np.array_equal(ORC.rk_step(q0, p, G, ext, dt, 0), q0)


def test_conservation_over_ten_steps_cfg1():
    c = I.CONFIGS["cfg1"]
    p, ext = c["p"], c["extent"]
    q0 = I.make_field("cfg1")
    dt = I.cfl_dt(ORC.max_wavespeed(q0, p, G), p, ext, (4, 4, 4))
    q1 = ORC.rk_step(q0, p, G, ext, dt, 10)
    drift = np.abs(bf.integrals(q1, p, ext) - bf.integrals(q0, p, ext))
    assert np.all(drift < 5e-15)
    assert np.abs(q1 - q0).max() > 1e-4         # something did happen


def _l2_density_error(q, exact, p, ext):
    d = np.zeros_like(q)
    d[..., 0] = (q[..., 0] - exact[..., 0]) ** 2
    return math.sqrt(bf.integrals(d, p, ext)[0] / (ext[0] * ext[1] * ext[2]))


def _run_to(field, n, p, ext, T, cfl=0.1, **kw):
    nx, ny, nz = n
    q0 = field(nx, ny, nz, p, ext, t=0.0, **kw)
    dt0 = I.cfl_dt(ORC.max_wavespeed(q0, p, G), p, ext, n, cfl)
    nsteps = int(math.ceil(T / dt0))
    q = Oracle("omp").rk_step(q0, p, G, ext, T / nsteps, nsteps)    # bit-identical to fp64 build
    return _l2_density_error(q, field(nx, ny, nz, p, ext, t=T, **kw), p, ext)


@pytest.mark.parametrize("p,lo", [(1, 1.9), (2, 2.3), (3, 3.8)])
def test_convergence_density_wave_quasi_1d(p, lo):
    """P8: rho = 1 + 0.2 sin(2 pi (x - 0.5 t)), u = 0.5, p = 1 is an exact periodic Euler solution."""
    ext = (1.0, 1.0, 1.0)
    kw = dict(vel=(0.5, 0.0, 0.0), waves=(1, 0, 0))
    errs = [_run_to(I.density_wave, (n, 1, 1), p, ext, 1.0, **kw) for n in (8, 16, 32)]
    orders = [math.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert min(orders) > lo, (errs, orders)
    assert max(orders) < p + 1 + 1.0, (errs, orders)


def test_convergence_density_wave_oblique_3d():
    """Same exact solution travelling obliquely through a 3-D mesh (cfg1's field without noise)."""
    ext = (1.0, 1.0, 1.0)
    errs = [_run_to(I.density_wave, (n, n, n), 2, ext, 0.25) for n in (4, 8)]
    assert math.log2(errs[0] / errs[1]) > 2.3, errs


def test_convergence_isentropic_vortex():
    """P9: cfg2's vortex translating in x; p = 3 must converge at about order 4."""
    ext = (10.0, 10.0, 2.5)
    errs = [_run_to(I.isentropic_vortex, (n, n, n // 4), 3, ext, 0.5) for n in (8, 16)]
    assert math.log2(errs[0] / errs[1]) > 3.3, errs
    assert errs[1] < 2e-4, errs


@pytest.mark.slow
def test_convergence_isentropic_vortex_three_grids():
    ext = (10.0, 10.0, 2.5)
    errs = [_run_to(I.isentropic_vortex, (n, n, n // 4), 3, ext, 1.0) for n in (8, 16, 32)]
    orders = [math.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert min(orders) > 3.5, (errs, orders)

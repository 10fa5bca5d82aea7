"""Pins P5, P6, P10, P11 for the oracle's residual; CPU only.

Expected values come from (a) a brute-force dense evaluation of eq (5) written independently in
numpy (tests/dg_bruteforce.py; weak form literally, and the strong form), (b) invariants the
discretisation must have on a periodic mesh: free-stream preservation, discrete conservation,
axis-permutation symmetry, independence of the volume term from neighbours.
"""
import numpy as np
import pytest

import dg_bruteforce as bf
from oracle import Oracle
from paper_2006_15698_b200 import inputs as I

ORC = Oracle("fp64")
G = 1.4


def relerr(a, b):
    """max over variables of |a-b|_inf / |b|_inf (absolute where |b|_inf = 0)."""
    out = 0.0
    for n in range(5):
        d = np.abs(a[..., n] - b[..., n]).max()
        s = np.abs(b[..., n]).max()
        out = max(out, d / s if s > 0 else d)
    return out


def rough_field(nx, ny, nz, p, extent, seed=7, mach_like=True):
    """Smooth wave + large discontinuous noise: exercises the jump term of the interface flux."""
    q = I.density_wave(nx, ny, nz, p, extent, vel=(0.5, -0.3, 0.2), noise=5e-2, seed=seed, waves=(1, 2, 1))
    return q


@pytest.mark.parametrize("nx,ny,nz,p,extent", [
    (1, 1, 1, 1, (1.0, 1.0, 1.0)),
    (2, 2, 2, 1, (1.0, 1.0, 1.0)),
    (3, 2, 1, 2, (1.0, 0.7, 0.4)),        # anisotropic: catches swapped axes / wrong h_a
    (2, 1, 3, 3, (2.0, 0.5, 1.5)),
    (2, 2, 2, 4, (1.0, 1.0, 1.0)),
])
def test_residual_equals_bruteforce_weak_and_strong(nx, ny, nz, p, extent):
    q = rough_field(nx, ny, nz, p, extent)
    r = ORC.residual(q, p, G, extent)
    rw = bf.residual(q, p, G, extent, "weak")
    rs = bf.residual(q, p, G, extent, "strong")
    assert relerr(r, rw) < 2e-13
    assert relerr(r, rs) < 2e-12
    # and the two terms separately: V - S = R, V is element-local
    V = ORC.volume_term(q, p, G, extent)
    S = ORC.surface_term(q, p, G, extent)
    assert np.array_equal(V - S, r)


def test_volume_term_is_element_local_and_matches_dense_operator():
    nx, ny, nz, p, extent = 3, 2, 2, 2, (1.0, 1.5, 0.5)
    N = p + 1
    q = rough_field(nx, ny, nz, p, extent)
    V = ORC.volume_term(q, p, G, extent)
    q2 = q.copy()
    q2[0, 0, 1] *= 1.01                      # perturb one element
    V2 = ORC.volume_term(q2, p, G, extent)
    changed = np.abs(V2 - V).reshape(nz, ny, nx, -1).max(-1) > 0
    assert changed.sum() == 1 and changed[0, 0, 1]
    # dense form of eq (5) 2nd term / mass for one element
    (Dx, Dy, Dz), _, W, _ = bf._dense_ops(N)
    h = [extent[0] / nx, extent[1] / ny, extent[2] / nz]
    Q = q[1, 1, 2].reshape(N ** 3, 5)
    ref = sum((2.0 / h[a]) * (Dm.T @ (W[:, None] * bf.flux(Q, a, G))) for a, Dm in enumerate((Dx, Dy, Dz))) / W[:, None]
    assert relerr(V[1, 1, 2].reshape(N ** 3, 5), ref) < 2e-13


@pytest.mark.parametrize("p", [1, 3, 4, 7])
def test_free_stream_preservation(p):
    nx, ny, nz, extent = 3, 2, 2, (1.0, 0.5, 0.8)
    q = I.uniform_state(nx, ny, nz, p, rho=1.1, vel=(0.3, -0.2, 0.1), pres=0.9)
    r = ORC.residual(q, p, G, extent)
    N = p + 1
    scale = np.abs(q).max() * (2.0 / min(extent[0] / nx, extent[1] / ny, extent[2] / nz)) * N * N
    assert np.abs(r).max() < 2e-15 * scale                           # P5


def test_free_stream_cfg1_magnitude():
    q = I.uniform_state(4, 4, 4, 1, rho=1.0, vel=(0.5, 0.5, 0.5), pres=1.0)
    assert np.abs(ORC.residual(q, 1, G, (1.0, 1.0, 1.0))).max() < 2e-13


@pytest.mark.parametrize("cfg,box", [("cfg1", None), ("cfg2", ((4, 10), (3, 8), (0, 2)))])
def test_discrete_conservation(cfg, box):
    c = I.CONFIGS[cfg]
    q = I.make_field(cfg, box=box)
    nz, ny, nx = q.shape[:3]
    ext = tuple(c["extent"][a] * n / c[k] for a, (n, k) in enumerate(zip((nx, ny, nz), ("nx", "ny", "nz"))))
    r = ORC.residual(q, c["p"], G, ext)
    tot = bf.integrals(r, c["p"], ext)
    mag = bf.integrals(np.abs(r), c["p"], ext)
    assert np.all(np.abs(tot) < 1e-14 * np.maximum(mag, 1.0))       # P6


def test_axis_permutation_symmetry():
    n, p, extent = 2, 2, (1.0, 1.0, 1.0)
    q = rough_field(n, n, n, p, extent)
    r = ORC.residual(q, p, G, extent)
    # swap x <-> y: Q'(x,y,z) = S Q(y,x,z), S swaps the x- and y-momentum
    perm = [0, 2, 1, 3, 4]
    qs = np.ascontiguousarray(np.transpose(q, (0, 2, 1, 3, 5, 4, 6))[..., perm])
    rs = ORC.residual(qs, p, G, extent)
    assert relerr(np.transpose(rs, (0, 2, 1, 3, 5, 4, 6))[..., perm], r) < 1e-13
    # swap x <-> z
    perm = [0, 3, 2, 1, 4]
    qs = np.ascontiguousarray(np.transpose(q, (2, 1, 0, 5, 4, 3, 6))[..., perm])
    rs = ORC.residual(qs, p, G, extent)
    assert relerr(np.transpose(rs, (2, 1, 0, 5, 4, 3, 6))[..., perm], r) < 1e-13


def test_single_element_axis_is_its_own_neighbour():
    """n_a = 1: periodic wrap makes the element its own neighbour (reading R13)."""
    p, extent = 2, (1.0, 1.0, 1.0)
    q1 = rough_field(3, 1, 1, p, extent)
    # tiling the field twice along y with doubled extent is the same periodic problem
    q2 = np.concatenate([q1, q1], axis=1)
    r1 = ORC.residual(q1, p, G, extent)
    r2 = ORC.residual(q2, p, G, (1.0, 2.0, 1.0))
    assert np.array_equal(r2[:, 0], r1[:, 0]) and np.array_equal(r2[:, 1], r1[:, 0])


def test_openmp_build_is_bit_identical_and_long_double_is_close():
    c = I.CONFIGS["cfg1"]
    q = I.make_field("cfg1")
    r = ORC.residual(q, c["p"], G, c["extent"])
    assert np.array_equal(Oracle("omp").residual(q, c["p"], G, c["extent"]), r)
    assert relerr(Oracle("ld").residual(q, c["p"], G, c["extent"]), r) < 2e-13   # fp64 roundoff scale


def test_max_wavespeed_matches_definition():
    q = I.make_field("cfg2")
    rho = q[..., 0]
    vel = q[..., 1:4] / rho[..., None]
    pres = (G - 1) * (q[..., 4] - 0.5 * rho * (vel ** 2).sum(-1))
    ref = (np.sqrt((vel ** 2).sum(-1)) + np.sqrt(G * pres / rho)).max()
    assert abs(ORC.max_wavespeed(q, 3, G) - ref) < 1e-14 * ref


def test_max_wavespeed_closed_forms_uniform_spike_and_nan():
    """Pins oracle_max_wavespeed by numbers written out by hand (the rule itself is DESIGN.md reading R10: the
    paper has no CFL rule).  Uniform state rho = 1.25, u = (0.3, -0.4, 1.2), p = 1.75, gamma = 7/5:
    |u| = sqrt(0.09 + 0.16 + 1.44) = 1.3 and c = sqrt(1.4 * 1.75 / 1.25) = sqrt(1.96) = 1.4, so lam = 2.7.
    One spiked node rho = 1, u = (0.6, 0.8, 0), p = 3.15: |u| = 1, c = sqrt(1.4 * 3.15) = sqrt(4.41) = 2.1,
    lam = 3.1, wherever the node sits (pins the max-reduction, first / middle / last node)."""
    nx, ny, nz, p = 3, 2, 2, 2
    q = I.uniform_state(nx, ny, nz, p, rho=1.25, vel=(0.3, -0.4, 1.2), pres=1.75, gamma=1.4)
    assert abs(ORC.max_wavespeed(q, p, 1.4) - 2.7) < 4e-15
    spike = I.uniform_state(1, 1, 1, 0, rho=1.0, vel=(0.6, 0.8, 0.0), pres=3.15, gamma=1.4).reshape(5)
    flat = q.reshape(-1, 5)
    for node in (0, flat.shape[0] // 2 + 3, flat.shape[0] - 1):
        qs = q.copy()
        qs.reshape(-1, 5)[node] = spike
        assert abs(ORC.max_wavespeed(qs, p, 1.4) - 3.1) < 4e-15, node
    # a velocity spike below the maximum must not win, a transposed momentum component must not matter
    qs = q.copy()
    qs.reshape(-1, 5)[7] = I.uniform_state(1, 1, 1, 0, rho=1.25, vel=(1.2, 0.3, -0.4), pres=1.75, gamma=1.4).reshape(5)
    assert abs(ORC.max_wavespeed(qs, p, 1.4) - 2.7) < 4e-15
    # negative pressure: the square root is NaN and it propagates (no limiter, reading R15)
    qs = q.copy()
    qs.reshape(-1, 5)[11, 4] = 0.1
    assert np.isnan(ORC.max_wavespeed(qs, p, 1.4))


def test_invalid_arguments_are_rejected():
    q = I.make_field("cfg1")
    with pytest.raises(ValueError):
        ORC.residual(q, 1, 0.9, (1.0, 1.0, 1.0))      # gamma <= 1
    with pytest.raises(ValueError):
        ORC.residual(q, 1, G, (1.0, -1.0, 1.0))       # extent <= 0

"""GPU parity of the viscous (Navier-Stokes) terms, SURVEY.md 8(f)-4 (reading R20: the paper names them only,
PAPER.md:86): dg_split_viscous / dg_rk_step_ns against the oracle's viscous_term / residual_ns / rk_step_ns, for every
degree and every compiled column shape, on meshes ragged against the columns."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import Oracle                                    # noqa: E402
from oracle.parity import relerr                             # noqa: E402
from paper_2006_15698_b200 import DG, DGError, load_library  # noqa: E402
from paper_2006_15698_b200 import inputs as I                # noqa: E402

G, MU, PR = 1.4, 0.02, 0.72
ORC = Oracle("omp")


def rough_field(nx, ny, nz, p, extent, seed=11):
    return I.density_wave(nx, ny, nz, p, extent, vel=(0.5, -0.3, 0.2), noise=5e-3, seed=seed, waves=(1, 2, 1))


@pytest.mark.parametrize("p", range(1, 8))
def test_viscous_term_and_ns_residual_match_the_oracle(p):
    nx, ny, nz, ext = 5, 3, 4, (1.0, 0.6, 0.9)                 # ragged against every column shape; n_z > 2
    q = rough_field(nx, ny, nz, p, ext)
    r_orc = ORC.residual(q, p, G, ext)
    rv_orc = ORC.viscous_term(q, p, G, ext, MU, PR)
    rns_orc = ORC.residual_ns(q, p, G, ext, MU, PR)
    for variant in range(load_library().dg_variant_count(p)):
        dg = DG(nx, ny, nz, p, G, ext, variant=variant, viscosity=(MU, PR), poison=True)
        dg.set_state(q)
        r = dg.split_volume().split_surface().split_r()
        rns = dg.split_viscous().split_r()
        assert relerr(r, r_orc) < 1e-11, (p, variant, "euler", relerr(r, r_orc))
        assert relerr(rns, rns_orc) < 1e-11, (p, variant, "navier-stokes", relerr(rns, rns_orc))
        # the viscous part on its own, at the accuracy a difference of two residuals allows
        rv = rns - r
        for n in range(5):
            d = np.abs(rv[..., n] - rv_orc[..., n]).max()
            assert d <= 1e-11 * np.abs(rv_orc[..., n]).max() + 4e-16 * np.abs(r_orc[..., n]).max(), (p, variant, n, d)
        assert np.array_equal(rns[..., 0], r[..., 0])          # no viscous mass flux, bit for bit
        assert np.array_equal(dg.residual_ns(), rns)           # run to run
        assert np.array_equal(dg.get_state(), q)               # none of the kernels touches the state
        dg.close()


@pytest.mark.parametrize("shape,p", [((1, 1, 1), 2), ((1, 4, 2), 3), ((4, 4, 4), 1), ((3, 2, 5), 4), ((2, 2, 2), 7)])
def test_ns_steps_match_the_oracle(shape, p):
    ext = (1.0, 1.3, 0.7)
    q = rough_field(*shape, p, ext, seed=3)
    # explicit viscous stability: dt ~ h^2 / (nu (2p+1)^2) is far above the convective CFL 0.1 step at this mu
    dt = I.cfl_dt(ORC.max_wavespeed(q, p, G), p, ext, shape, 0.1)
    dg = DG(*shape, p, G, ext, viscosity=(MU, PR))
    q3 = dg.set_state(q).rk_step_ns(dt, 3).get_state()
    ref = ORC.rk_step_ns(q, p, G, ext, MU, PR, dt, 3)
    assert np.isfinite(q3).all()
    assert relerr(q3, ref) < 1e-12, relerr(q3, ref)
    assert relerr(q3, ORC.rk_step(q, p, G, ext, dt, 3)) > 1e-8   # and the viscous terms did something
    # the traces the update kernel leaves behind let the fused (inviscid) path continue from there
    q4 = dg.rk_step(dt, 1).get_state()
    assert relerr(q4, ORC.rk_step(ref, p, G, ext, dt, 1)) < 1e-12
    dg.close()


def test_viscous_errors():
    q = rough_field(2, 2, 2, 2, (1.0, 1.0, 1.0))
    dg = DG(2, 2, 2, 2, G).set_state(q)
    with pytest.raises(DGError) as e:
        dg.split_viscous()                                     # no viscosity set
    assert e.value.code == 5
    with pytest.raises(DGError) as e:
        dg._check(dg.lib.dg_set_viscosity(dg._h, 0.1, 0.7))    # after dg_bind
    assert e.value.code == 5
    dg.close()
    for mu, pr in ((-1.0, 0.7), (0.1, 0.0), (float("nan"), 0.7)):
        with pytest.raises(DGError) as e:
            DG(2, 2, 2, 2, G, viscosity=(mu, pr), bind=False)
        assert e.value.code == 1
    dg = DG(2, 2, 2, 2, G, viscosity=(0.1, 0.7)).set_state(q)
    dg.set_boundary((1, 1, 0, 0, 0, 0))
    with pytest.raises(DGError) as e:
        dg.split_viscous()                                     # periodic only
    assert e.value.code == 2
    dg.close()
    # mu = 0 needs no extra workspace
    a, b = DG(3, 3, 3, 2, G, bind=False), DG(3, 3, 3, 2, G, viscosity=(0.0, 0.7), bind=False)
    c = DG(3, 3, 3, 2, G, viscosity=(0.1, 0.7), bind=False)
    assert a.workspace_bytes == b.workspace_bytes < c.workspace_bytes


def test_navier_stokes_full_size_sampled():
    """bench.py's Navier-Stokes workload (table2_p6: 40^3 elements, p = 6, 22 M nodes), sampled as in
    tests/test_gpu_fullsize.py: the viscous stencil reaches two elements (gradient, then divergence), so the periodic
    oracle on a sub-box reproduces the full mesh 2 elements (residual) or 10 elements (one 5-stage step) inside it."""
    from oracle.parity import assert_parity
    from test_gpu_fullsize import take_box, RES_ALLOWED
    arb = Oracle("ld_omp")
    cfg, mu, pr = "table2_p6", 1e-3, 0.72
    c = I.CONFIGS[cfg]
    p, ext, n = c["p"], c["extent"], (c["nx"], c["ny"], c["nz"])
    h = [ext[a] / n[a] for a in range(3)]
    q = I.make_field(cfg, xp=torch, device="cuda")
    dg = DG(*n, p, G, ext, viscosity=(mu, pr)).set_state(q)
    dt = I.cfl_dt(dg.max_wavespeed(), p, ext, n, 0.1)
    r = dg.residual_ns(torch.empty_like(q))
    for lo, size in [((37, 38, 36), (6, 6, 7)), ((11, 20, 3), (6, 6, 6))]:       # across the periodic corner; inside
        sub_ext = tuple(h[a] * size[a] for a in range(3))
        qb = take_box(q, lo, size)
        inner = (slice(2, -2),) * 3
        # full size: every variable's residual is a cancellation residue (tests/test_gpu_fullsize.py, RES_ALLOWED)
        assert_parity(take_box(r, lo, size)[inner], ORC.residual_ns(qb, p, G, sub_ext, mu, pr)[inner],
                      lambda: arb.residual_ns(qb, p, G, sub_ext, mu, pr)[inner], 1e-11, (cfg, "residual_ns", lo),
                      allowed=RES_ALLOWED)
    del r
    lo, size = (30, 29, 31), (22, 22, 22)
    qb = take_box(q, lo, size)
    dg.rk_step_ns(dt, 1).get_state(q)
    sub_ext = tuple(h[a] * size[a] for a in range(3))
    inner = (slice(10, -10),) * 3
    assert_parity(take_box(q, lo, size)[inner], ORC.rk_step_ns(qb, p, G, sub_ext, mu, pr, dt, 1)[inner],
                  lambda: arb.rk_step_ns(qb, p, G, sub_ext, mu, pr, dt, 1)[inner], 1e-11, (cfg, "rk_step_ns", lo), allowed=())
    dg.close()

"""GPU parity of the paper-shaped per-kernel mode (Table II): volume kernel,
surface kernel and update-project kernel as separate launches, each against the oracle's term of the same name."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import Oracle                                    # noqa: E402
from oracle.parity import relerr                             # noqa: E402
from paper_2006_15698_b200 import DG, load_library           # noqa: E402
from paper_2006_15698_b200 import inputs as I                # noqa: E402

G = 1.4
ORC = Oracle("omp")


def rough_field(nx, ny, nz, p, extent, seed=11):
    return I.density_wave(nx, ny, nz, p, extent, vel=(0.5, -0.3, 0.2), noise=5e-2, seed=seed, waves=(1, 2, 1))


@pytest.mark.parametrize("p", range(1, 8))
def test_volume_and_surface_kernels_match_the_oracle_terms(p):
    nx, ny, nz, ext = 5, 3, 4, (1.0, 0.6, 0.9)                 # ragged against every column shape; n_z > 2
    q = rough_field(nx, ny, nz, p, ext)
    v_orc, s_orc, r_orc = ORC.volume_term(q, p, G, ext), ORC.surface_term(q, p, G, ext), ORC.residual(q, p, G, ext)
    for variant in range(load_library().dg_variant_count(p)):
        dg = DG(nx, ny, nz, p, G, ext, variant=variant)
        dg.set_state(q)
        v = dg.split_volume().split_r()
        assert relerr(v, v_orc) < 1e-11, (p, variant, "volume", relerr(v, v_orc))
        r = dg.split_surface().split_r(torch.empty(q.shape, dtype=torch.float64, device="cuda")).cpu().numpy()
        assert relerr(r, r_orc) < 1e-11, (p, variant, "residual", relerr(r, r_orc))
        assert relerr(v - r, s_orc) < 1e-11, (p, variant, "surface", relerr(v - r, s_orc))
        assert np.array_equal(dg.get_state(), q)               # neither kernel touches the state
        dg.close()


@pytest.mark.parametrize("shape,p", [((1, 1, 1), 2), ((1, 4, 2), 3), ((4, 4, 4), 1), ((3, 2, 5), 4)])
def test_split_steps_match_the_oracle_and_the_fused_path(shape, p):
    """5 x (volume, surface, update-project) = one LSERK45 step; the traces the update kernel leaves behind let the
    fused path continue from there."""
    ext = (1.0, 1.3, 0.7)
    q = rough_field(*shape, p, ext, seed=3)
    dt = I.cfl_dt(ORC.max_wavespeed(q, p, G), p, ext, shape, 0.1)
    dg = DG(*shape, p, G, ext)
    q2 = dg.set_state(q).rk_step_split(dt, 2).get_state()
    assert relerr(q2, ORC.rk_step(q, p, G, ext, dt, 2)) < 1e-12
    q4 = dg.rk_step(dt, 2).get_state()                         # fused steps on top of split steps
    assert relerr(q4, ORC.rk_step(q, p, G, ext, dt, 4)) < 1e-12
    fused = DG(*shape, p, G, ext).set_state(q).rk_step(dt, 4).get_state()
    assert relerr(q4, fused) < 1e-13
    dg.close()

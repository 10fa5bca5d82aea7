"""GPU parity with non-periodic domain faces (reading R19): slip walls and far-field
faces through dg_set_boundary against the oracle's residual_bc / rk_step_bc (pinned on the CPU by the mirror-image
equivalence with the periodic oracle, tests/test_oracle_boundary.py)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import Oracle                                    # noqa: E402
from oracle.parity import relerr                             # noqa: E402
from paper_2006_15698_b200 import DG, DGError, load_library  # noqa: E402
from paper_2006_15698_b200 import inputs as I                # noqa: E402

G = 1.4
ORC = Oracle("omp")
PER, WALL, FAR = 0, 1, 2
CASES = [[WALL] * 6, [FAR] * 6, [WALL, FAR, PER, PER, FAR, WALL], [PER, PER, WALL, WALL, PER, PER],
         [FAR, WALL, WALL, FAR, PER, PER]]


def rough_field(nx, ny, nz, p, extent, seed=11):
    return I.density_wave(nx, ny, nz, p, extent, vel=(0.5, -0.3, 0.2), noise=5e-2, seed=seed, waves=(1, 2, 1))


@pytest.mark.parametrize("p", range(1, 8))
def test_residual_and_steps_with_walls_and_far_field_all_variants(p):
    nx, ny, nz, ext = 5, 3, 4, (1.0, 0.6, 0.9)                 # ragged against every column shape, several layers
    q = rough_field(nx, ny, nz, p, ext)
    qinf = I.uniform_state(1, 1, 1, 0, rho=1.05, vel=(0.45, -0.25, 0.15), pres=1.1, gamma=G).reshape(5)
    dt = I.cfl_dt(ORC.max_wavespeed(q, p, G), p, ext, (nx, ny, nz), 0.1)
    for bc in CASES if p < 5 else CASES[:3]:
        r_orc = ORC.residual_bc(q, p, G, ext, bc, qinf)
        q_orc = ORC.rk_step_bc(q, p, G, ext, bc, qinf, dt, 3)
        for variant in range(load_library().dg_variant_count(p)):
            for lz in (0, 1, 3):                               # chunk ends inside the domain and on its faces
                dg = DG(nx, ny, nz, p, G, ext, variant=variant, brick=(0, 0, lz)).set_boundary(bc, qinf)
                r = dg.set_state(q).residual()
                assert relerr(r, r_orc) < 1e-11, (p, bc, variant, lz, relerr(r, r_orc))
                q3 = dg.rk_step(dt, 3).get_state()
                assert relerr(q3, q_orc) < 1e-12, (p, bc, variant, lz, relerr(q3, q_orc))
                dg.close()


def test_far_field_preserves_the_free_stream_and_boundaries_can_be_switched():
    n, p, ext = (6, 5, 4), 3, (1.0, 1.0, 0.7)
    qu = I.uniform_state(*n, p, rho=1.1, vel=(0.3, -0.2, 0.4), pres=0.9, gamma=G)
    dg = DG(*n, p, G, ext).set_boundary([FAR] * 6, qu.reshape(-1, 5)[0])
    assert np.abs(dg.set_state(qu).residual()).max() < 2e-12
    q = rough_field(*n, p, ext, seed=2)
    dg.set_state(q)
    r_far = dg.residual()
    r_per = dg.set_boundary([PER] * 6).residual()              # back to periodic on the same context
    assert relerr(r_per, ORC.residual(q, p, G, ext)) < 1e-11
    assert relerr(r_far, ORC.residual_bc(q, p, G, ext, [FAR] * 6, qu.reshape(-1, 5)[0])) < 1e-11
    with pytest.raises(DGError):
        dg.set_boundary([WALL, PER, PER, PER, PER, PER])       # periodic on one face of an axis only
    with pytest.raises(DGError):
        dg.set_boundary([FAR] * 6)                             # far field without a state
    with pytest.raises(DGError):
        dg.set_boundary([WALL] * 6).split_volume().split_surface()   # per-kernel mode is periodic only
    dg.close()

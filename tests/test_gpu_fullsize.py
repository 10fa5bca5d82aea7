"""GPU parity at BASELINE.json's FULL sizes (configs 3, 4, 5), in the launch configuration bench.py times.

The oracle cannot run 1e8-1e9 unknowns in seconds, so outputs are SAMPLED: because dQ/dt of an
element depends only on itself and its 6 face neighbours, the periodic oracle run on an extracted
sub-box reproduces the full-mesh result on every element at least 1 element (residual) or 5
elements (one 5-stage Runge-Kutta step) away from the sub-box edge.  Several sub-boxes are taken,
including ones that straddle the periodic wrap and the ragged last brick.

The initial field is generated on the device by the shared input module (torch backend); the
oracle's input is a slice of that very tensor, taken before it is handed to the library.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import Oracle                                    # noqa: E402
from oracle.parity import add_term_scale, assert_parity, assert_term_scale   # noqa: E402
from paper_2006_15698_b200 import DG                         # noqa: E402
from paper_2006_15698_b200 import inputs as I                # noqa: E402

G = 1.4
ORC = Oracle("omp")
ARB = Oracle("ld_omp")


def relerr(a, b):
    out = 0.0
    for n in range(5):
        d = np.abs(a[..., n] - b[..., n]).max()
        s = np.abs(b[..., n]).max()
        out = max(out, d / s if s > 0 else d)
    return out


def take_box(t, lo, size):
    """Periodic sub-box of a (nz,ny,nx,...) device tensor -> numpy, element ranges lo[a]..lo[a]+size[a]."""
    nz, ny, nx = t.shape[:3]
    ix = torch.arange(lo[0], lo[0] + size[0], device=t.device) % nx
    iy = torch.arange(lo[1], lo[1] + size[1], device=t.device) % ny
    iz = torch.arange(lo[2], lo[2] + size[2], device=t.device) % nz
    return t.index_select(0, iz).index_select(1, iy).index_select(2, ix).cpu().numpy()


def sampled_parity(cfg, boxes_res, boxes_rk, tol_res=1e-11, tol_rk=1e-11, cfl=0.1, allowed_res=(), allowed_rk=(),
                   always_arbiter=False, reports=None):
    c = I.CONFIGS[cfg]
    p, ext, n = c["p"], c["extent"], (c["nx"], c["ny"], c["nz"])
    q = I.make_field(cfg, xp=torch, device="cuda")
    torch.cuda.synchronize()
    dg = DG(*n, p, G, ext)
    dg.set_state(q)
    lam = dg.max_wavespeed()
    dt = I.cfl_dt(lam, p, ext, n, cfl)
    r = torch.empty_like(q)
    dg.residual(r)
    h = [ext[a] / n[a] for a in range(3)]
    worst = {}
    for lo, size in boxes_res:
        sub_ext = tuple(h[a] * size[a] for a in range(3))
        qb = take_box(q, lo, size)
        r_orc = ORC.residual(qb, p, G, sub_ext)
        r_gpu = take_box(r, lo, size)
        inner = (slice(1, -1),) * 3
        rep = assert_parity(r_gpu[inner], r_orc[inner], lambda: ARB.residual(qb, p, G, sub_ext)[inner], tol_res,
                            (cfg, "residual", lo), allowed=allowed_res, always_arbiter=always_arbiter)
        # the number that needs no arbiter: the difference against the size of the volume and surface terms that
        # cancel in the residual (every variable, strict, 1e-13)
        add_term_scale(rep, [ORC.volume_term(qb, p, G, sub_ext)[inner], ORC.surface_term(qb, p, G, sub_ext)[inner]])
        assert_term_scale(rep, (cfg, "residual", lo))
        if reports is not None:
            reports.append((cfg, "residual", lo, size, rep))
        worst["residual"] = max(worst.get("residual", 0.0), rep["strict_rel_max"])
        worst["residual_rel_to_terms"] = max(worst.get("residual_rel_to_terms", 0.0), rep["rel_to_terms_max"])
        worst.setdefault("residual_arbiter_vars", set()).update(rep["arbiter_vars"])
    del r
    q_boxes = [take_box(q, lo, size) for lo, size in boxes_rk]
    dg.rk_step(dt, 1)
    dg.get_state(q)                                          # q now holds the stepped state
    for (lo, size), qb in zip(boxes_rk, q_boxes):
        sub_ext = tuple(h[a] * size[a] for a in range(3))
        q_orc = ORC.rk_step(qb, p, G, sub_ext, dt, 1)
        q_gpu = take_box(q, lo, size)
        inner = (slice(5, -5),) * 3
        rep = assert_parity(q_gpu[inner], q_orc[inner], lambda: ARB.rk_step(qb, p, G, sub_ext, dt, 1)[inner], tol_rk,
                            (cfg, "rk step", lo), allowed=allowed_rk, always_arbiter=always_arbiter)
        if reports is not None:
            reports.append((cfg, "1 RK step", lo, size, rep))
        worst["rk_step"] = max(worst.get("rk_step", 0.0), rep["strict_rel_max"])
        worst.setdefault("rk_arbiter_vars", set()).update(rep["arbiter_vars"])
    assert abs(lam - max(ORC.max_wavespeed(qb, p, G) for qb in q_boxes)) < 0.2 * lam   # same field, sampled
    dg.close()
    del q
    torch.cuda.empty_cache()
    return worst


# Which variables may pass through the arbiter clause (oracle/parity.py).  At full size the residual of every
# variable is a cancellation residue of terms 1e4-1e5 times larger (2/h is 100-700 and the fields are smooth), so
# the fp64 ORACLE's own error against its long-double build is 1e-11..1e-9 of the result there (eta/s column of
# profiles/r03_parity_report.md): no fp64 evaluation can meet 1e-11 of the result, and the GPU is held to
# g <= ARBITER_FACTOR eta instead (measured: g/eta <= 1.3) AND, with no arbiter involved, to 1e-13 of the volume and
# surface terms that cancel (d/terms column of the report).  After a Runge-Kutta step only rho w of the Taylor-Green fields
# (identically zero initially) is such a residue.
RES_ALLOWED = ("rho", "rho u", "rho v", "rho w", "rho E")
RK_ALLOWED_TGV = ("rho w",)


def test_cfg3_taylor_green_64cubed_p4_full_size():
    boxes_res = [((0, 0, 0), (4, 4, 4)), ((62, 62, 62), (4, 5, 6)), ((30, 17, 5), (6, 4, 4))]
    # Runge-Kutta step: a box across the periodic corner, one on the seams of the default 2x3 columns, one inside
    boxes_rk = [((59, 60, 61), (12, 12, 12)), ((25, 19, 7), (12, 12, 12))]
    print(sampled_parity("cfg3", boxes_res, boxes_rk, allowed_res=RES_ALLOWED, allowed_rk=RK_ALLOWED_TGV))


@pytest.mark.parametrize("p", range(1, 8))
def test_cfg4_order_sweep_full_size(p):
    n = I.cfg4_elems_per_side(p)
    boxes_res = [((n - 3, n - 2, n - 3), (6, 5, 6)), ((n // 2, 1, n // 3), (4, 4, 4))]
    boxes_rk = [((n - 6, n - 6, n - 6), (12, 12, 12))]
    print(sampled_parity(f"cfg4_p{p}", boxes_res, boxes_rk, allowed_res=RES_ALLOWED, allowed_rk=()))


def test_cfg5_taylor_green_96cubed_p7_full_size():
    """2.26e9 unknowns: 64-bit indexing, all Runge-Kutta registers resident."""
    free, total = torch.cuda.mem_get_info()
    if total < 150 * 2 ** 30:
        pytest.skip("needs a 180 GB device")
    boxes_res = [((94, 94, 94), (4, 4, 4)), ((40, 3, 77), (4, 4, 4))]
    boxes_rk = [((90, 91, 92), (12, 12, 12))]
    print(sampled_parity("cfg5", boxes_res, boxes_rk, allowed_res=RES_ALLOWED, allowed_rk=RK_ALLOWED_TGV))

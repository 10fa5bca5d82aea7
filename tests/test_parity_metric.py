"""The parity metric (oracle/parity.py) itself: what it accepts and what it must reject.  CPU only."""
import numpy as np

import dg_bruteforce as bf
from oracle import Oracle
from oracle.parity import assert_parity, compare, relerr
from paper_2006_15698_b200 import inputs as I

G = 1.4


def test_arbiter_builds_agree_bit_for_bit():
    c = dict(nx=3, ny=2, nz=2, p=2, extent=(1.0, 0.8, 0.6), field="taylor_green")
    q = I.make_field(c)
    a = Oracle("ld").residual(q, 2, G, c["extent"])
    b = Oracle("ld_omp").residual(q, 2, G, c["extent"])
    assert np.array_equal(a, b)
    assert Oracle("ld").real_bytes > 8


def test_cancellation_clause_accepts_a_reordered_fp64_evaluation_and_rejects_real_errors():
    """cfg2-like vortex: rho w is identically zero, so its residual is rounding residue.  A second, independent
    fp64 evaluation (the brute-force strong form) differs from the oracle by O(1) relative in that variable and
    must pass by the arbiter clause only; every real perturbation must fail."""
    c = dict(nx=4, ny=4, nz=2, p=3, extent=(10.0, 10.0, 2.5), field="isentropic_vortex")
    p, ext = c["p"], c["extent"]
    q = I.make_field(c)
    r = Oracle("fp64").residual(q, p, G, ext)
    arb = Oracle("ld").residual(q, p, G, ext)
    other = bf.residual(q, p, G, ext, "strong")
    assert relerr(other, r) > 1e-3                            # the strict metric alone is meaningless here
    ok, rep = compare(other, r, arb, 1e-11)
    assert ok and rep["arbiter_vars"] == ["rho w"], rep
    assert rep["strict_rel_max"] < 1e-11
    # real errors: one node off by 1e-9 relative; a scaled variable; noise in the zero variable far above rounding
    for n, delta in [(0, 1e-9), (4, 1e-10), (3, 1e-9)]:
        bad = other.copy()
        bad[1, 2, 3, 1, 2, 0, n] += delta * max(np.abs(r[..., n]).max(), 1.0)
        ok, rep = compare(bad, r, arb, 1e-11)
        assert not ok, (n, rep)
    try:
        assert_parity(other * (1 + 1e-10), r, lambda: arb, 1e-11, "scaled", allowed=["rho w"])
    except AssertionError:
        pass
    else:
        raise AssertionError("a 1e-10 relative scaling must fail the 1e-11 parity test")
    # the clause is only open to the variables the caller names
    assert_parity(other, r, lambda: arb, 1e-11, "strong form", allowed=["rho w"])
    try:
        assert_parity(other, r, lambda: arb, 1e-11, "strong form, nothing allowed")
    except AssertionError:
        pass
    else:
        raise AssertionError("rho w needs the arbiter clause and was not allowed to use it")
    # and the report carries the numbers for every variable once the arbiter has been evaluated
    rep = assert_parity(other, r, arb, 1e-11, "report", allowed=["rho w"], always_arbiter=True)
    assert all(row["g_over_eta"] is not None or row["oracle_own_error"] == 0.0 for row in rep["rows"])


def test_strict_metric_without_arbiter():
    a = np.ones((1, 1, 1, 2, 2, 2, 5))
    b = a.copy()
    assert compare(a, b, None, 1e-11)[0]
    b[..., 2] = 0.0
    a[..., 2] = 1e-30                                         # zero variable: absolute comparison, no arbiter given
    assert not compare(a, b, None, 1e-11)[0]


def test_term_scale_metric_needs_no_arbiter_and_rejects_real_errors():
    """d / max(|V|, |S|): the same vortex, whose rho w residual is pure rounding residue.  The independent strong-form
    evaluation is within 1e-13 of the oracle in EVERY variable once the difference is measured against the volume and
    surface terms that cancel (no arbiter, no allowed list); a perturbation of 1e-11 of those terms is rejected."""
    import pytest
    from oracle.parity import TERM_TOL, add_term_scale, assert_term_scale
    c = dict(nx=4, ny=4, nz=2, p=3, extent=(10.0, 10.0, 2.5), field="isentropic_vortex")
    p, ext = c["p"], c["extent"]
    q = I.make_field(c)
    orc = Oracle("fp64")
    r, V, S = orc.residual(q, p, G, ext), orc.volume_term(q, p, G, ext), orc.surface_term(q, p, G, ext)
    assert relerr(V - S, r) < 1e-12 or np.abs((V - S) - r).max() < 1e-13 * np.abs(V).max()   # residual = V - S
    other = bf.residual(q, p, G, ext, "strong")
    _, rep = compare(other, r, None, 1e-11)
    assert rep["rows"][3]["passed_by"] == "FAILED"            # rho w: hopeless relative to its own size ...
    add_term_scale(rep, [V, S])
    assert_term_scale(rep)                                    # ... and plain roundoff relative to the terms
    assert 0 < rep["rel_to_terms_max"] < TERM_TOL and all(row["term_scale"] > 0 for row in rep["rows"])
    for n in range(5):
        bad = other.copy()
        bad[1, 2, 3, 1, 2, 0, n] += 1e-11 * max(np.abs(V[..., n]).max(), np.abs(S[..., n]).max())
        _, rep = compare(bad, r, None, 1e-11)
        with pytest.raises(AssertionError):
            assert_term_scale(add_term_scale(rep, [V, S]))

"""The parity metric of the GPU-vs-oracle tests -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

DESIGN.md "parity metric".  For each conserved variable n (rho, rho u, rho v, rho w, rho E):

    d_n   = | x_gpu_n - x_orc_n |_inf          difference to the fp64 oracle
    s_n   = | x_orc_n |_inf                    size of that variable
    eta_n = | x_orc_n - x_arb_n |_inf          the fp64 oracle's OWN rounding error, measured against
                                               the long-double build of the same source (the arbiter)
    g_n   = | x_gpu_n - x_arb_n |_inf          the GPU's distance to the arbiter

    variable n passes if   d_n <= tol * s_n                  (north_star: 1e-11 residual, 1e-9 / 100 steps)
                     or    g_n <= ARBITER_FACTOR * eta_n     (cancellation clause)

The second clause exists because two correct fp64 evaluations of the same formula (the oracle's
unfused multiply-add vs the GPU's fused multiply-add and different summation order) cannot agree
better than the rounding error of either one.  Where a variable's result is a small difference of
large terms (rho w of a z-invariant vortex is identically zero; the momentum residuals of the
Mach-0.1 Taylor-Green field cancel a pressure of 71 against O(1) dynamics) that rounding error,
relative to the result, exceeds 1e-11 in the ORACLE ITSELF.  The clause accepts the GPU only when it
is as close to the higher-precision arbiter as the fp64 oracle is, within ARBITER_FACTOR; it never
applies when the oracle's own error is small, so a real discrepancy (a wrong coefficient, index or
sign) fails both.  ARBITER_FACTOR = 2: the largest g/eta measured on the B200 over configs 1-5 among the variables
that need the clause is 1.05, recorded in profiles/r03_parity_report.md (written by tests/gpu_parity_report.py).

A third number needs no arbiter (SURVEY.md 8(c) "roundoff hazard"): for a residual, d_n divided by the size of the
TERMS that cancel in it, t_n = max(|V_n|_inf, |S_n|_inf) with V the volume term and S the surface term of eq (5)
(oracle_volume_term / oracle_surface_term on the same elements; residual = V - S).  Rounding errors scale with the terms,
not with their difference, so d_n / t_n must read like a few units of roundoff whatever the cancellation:
`add_term_scale` puts it into the report rows and `assert_term_scale` holds it to TERM_TOL = 1e-13.

Every caller states which variables MAY use the clause (`allowed`); a variable outside that list
that needs it fails the test.  Every report carries d/s, eta/s and g/eta for all five variables
whenever the arbiter was evaluated, clause or not.
"""
import numpy as np

ARBITER_FACTOR = 2.0
TERM_TOL = 1e-13       # |gpu - oracle|_inf of a residual variable, relative to the larger of its volume and surface terms
NAMES = ("rho", "rho u", "rho v", "rho w", "rho E")


def relerr(a, b):
    """max over variables of |a-b|_inf / |b|_inf (absolute where |b|_inf = 0). The strict metric."""
    out = 0.0
    for n in range(5):
        d = np.abs(a[..., n] - b[..., n]).max()
        s = np.abs(b[..., n]).max()
        out = max(out, d / s if s > 0 else d)
    return out


def compare(x_gpu, x_orc, x_arb, tol):
    """Returns (ok, report).  report: per-variable d/s, eta/s, g/eta, which clause passed."""
    rows, ok = [], True
    for n in range(5):
        d = float(np.abs(x_gpu[..., n] - x_orc[..., n]).max())
        s = float(np.abs(x_orc[..., n]).max())
        strict = d <= tol * s
        eta = g = None
        clause = False
        if x_arb is not None:
            arb = np.asarray(x_arb[..., n], dtype=np.longdouble)
            eta = float(np.abs(x_orc[..., n] - arb).max())
            g = float(np.abs(x_gpu[..., n] - arb).max())
            clause = (not strict) and g <= ARBITER_FACTOR * eta
        ok = ok and (strict or clause)
        rows.append({"var": NAMES[n], "diff": d, "size": s, "rel": d / s if s > 0 else d,
                     "oracle_own_error": eta, "oracle_own_rel": None if eta is None else (eta / s if s > 0 else eta),
                     "gpu_to_arbiter": g, "g_over_eta": None if not eta else g / eta,
                     "passed_by": "strict" if strict else ("arbiter" if clause else "FAILED")})
    strict_rel = max([r["rel"] for r in rows if r["passed_by"] == "strict"], default=0.0)
    return ok, {"ok": ok, "tol": tol, "strict_rel_max": strict_rel, "rel_max": max(r["rel"] for r in rows),
                "arbiter_vars": [r["var"] for r in rows if r["passed_by"] == "arbiter"], "rows": rows}


def add_term_scale(rep, terms):
    """rep: a report of compare(); terms: arrays shaped like the compared residual (the oracle's volume and surface
    terms on the same nodes).  Adds term_scale = max_terms |term_n|_inf and rel_to_terms = d_n / term_scale per row."""
    worst = 0.0
    for n, row in enumerate(rep["rows"]):
        t = max(float(np.abs(term[..., n]).max()) for term in terms)
        row["term_scale"] = t
        row["rel_to_terms"] = row["diff"] / t if t > 0 else (0.0 if row["diff"] == 0 else float("inf"))
        worst = max(worst, row["rel_to_terms"])
    rep["rel_to_terms_max"] = worst
    return rep


def assert_term_scale(rep, what="", tol=TERM_TOL):
    bad = [(r["var"], r["rel_to_terms"]) for r in rep["rows"] if not r["rel_to_terms"] <= tol]
    assert not bad, (what, "difference to the oracle exceeds the roundoff of the terms that cancel", bad, tol)
    return rep


def format_report(rep):
    """One line per variable: d/s, eta/s, g/eta, clause."""
    out = []
    for r in rep["rows"]:
        eta = "-" if r["oracle_own_rel"] is None else f"{r['oracle_own_rel']:.2e}"
        ge = "-" if r["g_over_eta"] is None else f"{r['g_over_eta']:.2f}"
        out.append(f"{r['var']:6s} d/s={r['rel']:.2e} eta/s={eta} g/eta={ge} [{r['passed_by']}]")
    return "; ".join(out)


def assert_parity(x_gpu, x_orc, x_arb, tol, what="", allowed=(), always_arbiter=False):
    """x_arb may be an array, None, or a zero-argument callable (evaluated only if the strict test fails,
    unless always_arbiter).  `allowed` = the variables that may pass through the cancellation clause."""
    ok, rep = compare(x_gpu, x_orc, None, tol)
    if (not ok or always_arbiter) and x_arb is not None:
        ok, rep = compare(x_gpu, x_orc, x_arb() if callable(x_arb) else x_arb, tol)
    assert ok, (what, format_report(rep))
    extra = [v for v in rep["arbiter_vars"] if v not in allowed]
    assert not extra, (what, "variables outside the allowed list needed the arbiter clause", extra, format_report(rep))
    return rep

"""Writes the parity report of BASELINE.json's five configs on the GPU it runs on (markdown on stdout):

    python tests/gpu_parity_report.py > profiles/r03_parity_report.md

For every comparison and every conserved variable: d/s (GPU vs fp64 oracle, relative to the variable's
size), eta/s (the fp64 oracle's own rounding error against its long-double build) and g/eta (the GPU's
distance to that arbiter in units of the oracle's own error), with the arbiter ALWAYS evaluated, clause or
not.  oracle/parity.py's ARBITER_FACTOR is justified by the largest g/eta in this file.  Not a test; the
tests in test_gpu_parity.py / test_gpu_fullsize.py assert the same comparisons.
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, HERE)

from oracle import Oracle                                    # noqa: E402
from oracle.parity import ARBITER_FACTOR, NAMES, TERM_TOL, add_term_scale, assert_parity, assert_term_scale   # noqa: E402
from paper_2006_15698_b200 import DG                         # noqa: E402
from paper_2006_15698_b200 import inputs as I                # noqa: E402
import test_gpu_fullsize as FS                               # noqa: E402

G = 1.4
ORC, ARB = Oracle("omp"), Oracle("ld_omp")
ALL = list(NAMES)


def small(name, steps):
    c = I.CONFIGS[name]
    p, ext, n = c["p"], c["extent"], (c["nx"], c["ny"], c["nz"])
    q0 = I.make_field(name)
    dg = DG(*n, p, G, ext)
    out = []
    r = dg.set_state(q0).residual()
    rep = assert_parity(r, ORC.residual(q0, p, G, ext), ARB.residual(q0, p, G, ext), 1e-11, name, allowed=ALL, always_arbiter=True)
    assert_term_scale(add_term_scale(rep, [ORC.volume_term(q0, p, G, ext), ORC.surface_term(q0, p, G, ext)]), name)
    out.append((name, "residual", "-", n, rep))
    dt = I.cfl_dt(ORC.max_wavespeed(q0, p, G), p, ext, n, 0.1)
    q = dg.rk_step(dt, steps).get_state()
    out.append((name, f"{steps} RK steps", "-", n, assert_parity(q, ORC.rk_step(q0, p, G, ext, dt, steps),
                                                               ARB.rk_step(q0, p, G, ext, dt, steps),
                                                               1e-9 if steps >= 100 else 1e-11, name, allowed=ALL,
                                                               always_arbiter=True)))
    dg.close()
    return out


def main():
    import torch
    reports = small("cfg1", 10) + small("cfg2", 100)
    FS.sampled_parity("cfg3", [((0, 0, 0), (4, 4, 4)), ((62, 62, 62), (4, 5, 6)), ((30, 17, 5), (6, 4, 4))],
                      [((59, 60, 61), (12, 12, 12))], allowed_res=ALL, allowed_rk=ALL, always_arbiter=True, reports=reports)
    for p in range(1, 8):
        n = I.cfg4_elems_per_side(p)
        FS.sampled_parity(f"cfg4_p{p}", [((n - 3, n - 2, n - 3), (6, 5, 6)), ((n // 2, 1, n // 3), (4, 4, 4))],
                          [((n - 6, n - 6, n - 6), (12, 12, 12))], allowed_res=ALL, allowed_rk=ALL, always_arbiter=True,
                          reports=reports)
    if torch.cuda.mem_get_info()[1] >= 150 * 2 ** 30:
        FS.sampled_parity("cfg5", [((94, 94, 94), (4, 4, 4)), ((40, 3, 77), (4, 4, 4))], [((90, 91, 92), (12, 12, 12))],
                          allowed_res=ALL, allowed_rk=ALL, always_arbiter=True, reports=reports)
    print("# Parity report: CUDA path vs CPU oracle on", torch.cuda.get_device_name(0))
    print()
    print("Command: `python tests/gpu_parity_report.py > profiles/r03_parity_report.md` (one B200).  d = |gpu - oracle|_inf,")
    print("s = |oracle|_inf, eta = |oracle - arbiter|_inf (arbiter = long-double build of the oracle), g = |gpu - arbiter|_inf,")
    print(f"per conserved variable.  A variable passes by `strict` if d <= tol s, else by `arbiter` if g <= {ARBITER_FACTOR:g} eta.")
    print("Full-size configs 3-5: sampled sub-boxes (tests/test_gpu_fullsize.py).")
    print("d/terms (residual rows): d divided by max(|V|_inf, |S|_inf), V and S the oracle's volume and surface terms of the")
    print(f"same variable on the same elements (residual = V - S) -- the error against the size of what cancels; held to {TERM_TOL:g}")
    print("for every variable with no arbiter involved.  For Runge-Kutta rows d/s is already that number (s = |Q|_inf).")
    print()
    print("| config | quantity | box | variable | d/s | eta/s | g/eta | passed by | d/terms |")
    print("|---|---|---|---|---|---|---|---|---|")
    worst_g, worst_clause, worst_terms = 0.0, 0.0, 0.0
    for cfg, what, lo, size, rep in reports:
        for row in rep["rows"]:
            ge = row["g_over_eta"]
            if ge is not None:
                worst_g = max(worst_g, ge)
                if row["passed_by"] == "arbiter":
                    worst_clause = max(worst_clause, ge)
            print(f"| {cfg} | {what} | {lo}+{tuple(size)} | {row['var']} | {row['rel']:.2e} | "
                  f"{(row['oracle_own_rel'] or 0.0):.2e} | {'-' if ge is None else format(ge, '.2f')} | {row['passed_by']} | "
                  f"{'-' if 'rel_to_terms' not in row else format(row['rel_to_terms'], '.2e')} |")
            worst_terms = max(worst_terms, row.get("rel_to_terms", 0.0))
    print()
    print(f"Largest g/eta over all rows: {worst_g:.2f}; largest among the variables that needed the arbiter clause: "
          f"{worst_clause:.2f} (limit {ARBITER_FACTOR:g}).")
    print(f"Largest d/terms over all residual rows: {worst_terms:.2e} (limit {TERM_TOL:g}).")


if __name__ == "__main__":
    main()

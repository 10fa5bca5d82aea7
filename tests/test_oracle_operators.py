"""Pins P1-P4 for the oracle's 1-D operators; CPU only.

What fixes the expected values: closed forms of the Gauss-Legendre rules (textbook; the paper
names the rule), numpy's library rule, exactness of differentiation /
interpolation / quadrature for polynomials of the degree the basis holds (eq (6)-(7),
PAPER.md:72-78), and the summation-by-parts identity that makes the weak form of eq (5)
consistent.  Fixture values: tests/golden/gauss_legendre_closed_forms.txt.
"""
import math
import os

import numpy as np
import pytest

from oracle import Oracle

ORC = Oracle("fp64")
NS = list(range(1, 9))
GOLD = os.path.join(os.path.dirname(__file__), "golden", "gauss_legendre_closed_forms.txt")


def _golden():
    rules = {}
    for line in open(GOLD):
        line = line.split("#")[0].strip()
        if not line:
            continue
        N, i, x, w = line.split()
        rules.setdefault(int(N), []).append((int(i), eval(x, {"sqrt": math.sqrt}), eval(w, {"sqrt": math.sqrt})))
    return rules


def test_gl_closed_forms_from_fixture():
    for N, rows in _golden().items():
        xi, w = ORC.gauss_legendre(N)
        for i, x, ww in rows:
            assert abs(xi[i] - x) < 1e-15 and abs(w[i] - ww) < 1e-15, (N, i)


@pytest.mark.parametrize("N", NS)
def test_gl_matches_numpy_and_integrates_monomials(N):
    xi, w = ORC.gauss_legendre(N)
    x_np, w_np = np.polynomial.legendre.leggauss(N)
    assert np.all(np.diff(xi) > 0) or N == 1
    assert np.abs(xi - x_np).max() < 2e-15
    assert np.abs(w - w_np).max() < 2e-15
    assert abs(w.sum() - 2.0) < 1e-15
    for m in range(2 * N):          # exact to degree 2N-1
        assert abs(np.dot(w, xi ** m) - (1 + (-1) ** m) / (m + 1)) < 1e-15, m
    assert np.abs(xi + xi[::-1]).max() < 1e-16 and np.abs(w - w[::-1]).max() < 1e-16


def test_n2_closed_form_operators():
    o = ORC.operators(2)
    s3 = math.sqrt(3.0)
    assert np.abs(o["D"] - np.array([[-s3 / 2, s3 / 2], [-s3 / 2, s3 / 2]])).max() < 1e-15
    assert np.abs(o["lp"] - np.array([(1 - s3) / 2, (1 + s3) / 2])).max() < 1e-15
    assert np.abs(o["lm"] - np.array([(1 + s3) / 2, (1 - s3) / 2])).max() < 1e-15


@pytest.mark.parametrize("N", NS)
def test_exact_differentiation_and_interpolation(N):
    o = ORC.operators(N)
    xi, D, lp, lm = o["xi"], o["D"], o["lp"], o["lm"]
    assert np.abs(D @ np.ones(N)).max() < 5e-14                       # D.1 = 0
    for m in range(1, N):                                             # degree <= p
        assert np.abs(D @ xi ** m - m * xi ** (m - 1)).max() < 5e-14, m
    assert abs(lp.sum() - 1) < 1e-14 and abs(lm.sum() - 1) < 1e-14    # partition of unity
    for m in range(N):
        assert abs(np.dot(lp, xi ** m) - 1.0) < 1e-14
        assert abs(np.dot(lm, xi ** m) - (-1.0) ** m) < 1e-14
    assert np.abs(lm - lp[::-1]).max() < 1e-15                        # P11 mirror symmetry


@pytest.mark.parametrize("N", NS)
def test_differentiation_matrix_is_not_transposed(N):
    """D[q,i] = l_i'(xi_q): differentiating the i-th cardinal function gives column i."""
    if N == 1:
        return
    o = ORC.operators(N)
    xi, D = o["xi"], o["D"]
    for i in range(N):
        others = np.delete(xi, i)
        coef = np.poly(others) / np.prod(xi[i] - others)
        assert np.abs(D[:, i] - np.polyval(np.polyder(coef), xi)).max() < 2e-13


@pytest.mark.parametrize("N", NS)
def test_summation_by_parts_and_dhat(N):
    o = ORC.operators(N)
    w, D, lp, lm, Dhat = o["w"], o["D"], o["lp"], o["lm"], o["Dhat"]
    WD = w[:, None] * D
    assert np.abs(WD + WD.T - (np.outer(lp, lp) - np.outer(lm, lm))).max() < 5e-14      # P4
    assert np.abs(Dhat - (w[None, :] * D.T) / w[:, None]).max() < 1e-13                # Dhat[i,q]
    # consistency used by free-stream preservation: sum_q Dhat[i,q] = (lp_i - lm_i)/w_i
    assert np.abs(Dhat.sum(1) - (lp - lm) / w).max() < 5e-13


def test_long_double_build_agrees():
    ld = Oracle("ld")
    assert ld.real_bytes == 16 and ORC.real_bytes == 8
    for N in (2, 5, 8):
        a, b = ORC.operators(N), ld.operators(N)
        for k in a:
            assert np.array_equal(a[k], b[k])      # operators are built in long double in both

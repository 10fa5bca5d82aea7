"""Brute-force numpy evaluation of the paper's weak form, eq (5), for tiny meshes.

Test-only helper that pins the oracle to something other than itself.  It shares no code with
oracle/ or with the CUDA path and is deliberately built differently from both:
  * the Lagrange basis (eq (7)) is expanded with numpy.poly / polyder / polyval
    from numpy's own Gauss-Legendre points, not with barycentric formulas;
  * the 3-D operators are dense N^3 x N^3 Kronecker matrices, not sum-factorised lines;
  * eq (5) is evaluated literally: quadrature sums carrying weights and Jacobians for the volume
    and face integrals, THEN a division by the (diagonal) mass matrix;
  * a second routine evaluates the integrated-by-parts-twice STRONG form, which equals the weak
    form only if differentiation, interpolation, quadrature and lifting are mutually consistent.
Array layout: q[ez, ey, ex, k, j, i, n].
"""
import numpy as np


def basis_1d(N):
    xi, w = np.polynomial.legendre.leggauss(N)
    D = np.zeros((N, N))   # D[q, i] = l_i'(xi_q)
    lp = np.zeros(N)
    lm = np.zeros(N)
    for i in range(N):
        others = np.delete(xi, i)
        coef = np.poly(others) / np.prod(xi[i] - others)   # l_i as a polynomial (highest power first)
        dcoef = np.polyder(coef) if N > 1 else np.zeros(1)
        D[:, i] = np.polyval(dcoef, xi)
        lp[i] = np.polyval(coef, 1.0)
        lm[i] = np.polyval(coef, -1.0)
    return xi, w, D, lp, lm


def flux(Q, axis, gamma):
    """Column `axis` of the flux matrix F of eq (2), from conserved Q[..., 5]."""
    rho, mx, my, mz, E = (Q[..., n] for n in range(5))
    vel = np.stack([mx, my, mz], -1) / rho[..., None]
    pres = (gamma - 1.0) * (E - 0.5 * rho * np.sum(vel * vel, -1))
    va = vel[..., axis]
    F = np.stack([rho * va, mx * va, my * va, mz * va, (E + pres) * va], -1)
    F[..., 1 + axis] += pres
    return F


def lax_friedrichs(QL, QR, axis, gamma):
    """Local Lax-Friedrichs (Rusanov) flux with lam = max(|u_a|+c) over the two states (R3)."""
    def speed(Q):
        rho = Q[..., 0]
        vel = Q[..., 1:4] / rho[..., None]
        pres = (gamma - 1.0) * (Q[..., 4] - 0.5 * rho * np.sum(vel * vel, -1))
        return np.abs(vel[..., axis]) + np.sqrt(gamma * pres / rho)
    lam = np.maximum(speed(QL), speed(QR))
    return 0.5 * (flux(QL, axis, gamma) + flux(QR, axis, gamma)) - 0.5 * lam[..., None] * (QR - QL)


def _dense_ops(N):
    """Dense 3-D matrices acting on node vectors ordered (k, j, i), i fastest."""
    xi, w, D, lp, lm = basis_1d(N)
    I = np.eye(N)
    # derivative along x acts on index i (fastest) -> kron(I, I, D)
    Dx = np.kron(np.kron(I, I), D)
    Dy = np.kron(np.kron(I, D), I)
    Dz = np.kron(np.kron(D, I), I)
    W = np.kron(np.kron(w, w), w)
    # face interpolation: rows = face nodes ordered (t2, t1), t1 fastest
    Px = {+1: np.kron(np.kron(I, I), lp[None, :]), -1: np.kron(np.kron(I, I), lm[None, :])}   # (k,j)
    Py = {+1: np.kron(np.kron(I, lp[None, :]), I), -1: np.kron(np.kron(I, lm[None, :]), I)}   # (k,i)
    Pz = {+1: np.kron(np.kron(lp[None, :], I), I), -1: np.kron(np.kron(lm[None, :], I), I)}   # (j,i)
    Wf = np.kron(w, w)
    return (Dx, Dy, Dz), (Px, Py, Pz), W, Wf


def residual(q, p, gamma, extent, form="weak"):
    """dQ/dt on a periodic Cartesian mesh; `form` = 'weak' (eq (5) literally) or 'strong'."""
    N = p + 1
    nz, ny, nx = q.shape[:3]
    n = (nx, ny, nz)
    h = [extent[a] / n[a] for a in range(3)]
    Dm, Pm, W, Wf = _dense_ops(N)
    J = h[0] * h[1] * h[2] / 8.0
    Jf = [h[1] * h[2] / 4.0, h[0] * h[2] / 4.0, h[0] * h[1] / 4.0]
    Qe = q.reshape(nz, ny, nx, N ** 3, 5)

    def elem(ex, ey, ez):
        return Qe[ez % nz, ey % ny, ex % nx]

    def shift(e, a, s):
        e = list(e)
        e[a] += s
        return tuple(e)

    r = np.zeros_like(Qe)
    for ez in range(nz):
        for ey in range(ny):
            for ex in range(nx):
                e = (ex, ey, ez)
                Q = elem(*e)
                rhs = np.zeros((N ** 3, 5))   # M dQ/dt
                for a in range(3):
                    F = flux(Q, a, gamma)
                    P = Pm[a]
                    # interface fluxes on the + and - faces of this element (outward normals +e_a, -e_a)
                    Fp = lax_friedrichs(P[+1] @ Q, P[-1] @ elem(*shift(e, a, +1)), a, gamma)
                    Fm = lax_friedrichs(P[+1] @ elem(*shift(e, a, -1)), P[-1] @ Q, a, gamma)
                    if form == "weak":
                        # + int F_a dpsi/dx_a  - oint (F*.n) psi
                        vol = (2.0 / h[a]) * (Dm[a].T @ ((W * J)[:, None] * F))
                        surf = P[+1].T @ ((Wf * Jf[a])[:, None] * Fp) - P[-1].T @ ((Wf * Jf[a])[:, None] * Fm)
                        rhs += vol - surf
                    else:
                        # - int dF_a/dx_a psi - oint ((F* - F).n) psi,  F on the face = interpolated F
                        vol = -(2.0 / h[a]) * ((W * J)[:, None] * (Dm[a] @ F))
                        surf = (P[+1].T @ ((Wf * Jf[a])[:, None] * (Fp - P[+1] @ F))
                                - P[-1].T @ ((Wf * Jf[a])[:, None] * (Fm - P[-1] @ F)))
                        rhs += vol - surf
                r[ez, ey, ex] = rhs / (W * J)[:, None]
    return r.reshape(q.shape)


def integrals(q, p, extent):
    """Integral of each conserved variable over the domain with the collocated quadrature."""
    N = p + 1
    nz, ny, nx = q.shape[:3]
    _, w = np.polynomial.legendre.leggauss(N)
    J = (extent[0] / nx) * (extent[1] / ny) * (extent[2] / nz) / 8.0
    W = w[:, None, None] * w[None, :, None] * w[None, None, :]
    return J * np.einsum("zyxkjin,kji->n", q, W)

"""ctypes front end of the CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2006_15698_b200 and loads none of its
libraries.  Arrays are numpy float64 in the canonical layout of oracle/dg_oracle.h:
    q[ez, ey, ex, k, j, i, n]   (C order; n = rho, rho u, rho v, rho w, rho E)
"""
import ctypes
import os

import numpy as np

from . import build as _build

_DP = ctypes.POINTER(ctypes.c_double)
_LIBS = {}


def _load(variant):
    name = {"fp64": "libdg_oracle.so", "ld": "libdg_oracle_ld.so", "omp": "libdg_oracle_omp.so",
            "ld_omp": "libdg_oracle_ld_omp.so"}[variant]
    if name not in _LIBS:
        paths = _build.build()
        lib = ctypes.CDLL(paths[name])
        mesh = [ctypes.c_int] * 4 + [ctypes.c_double, _DP]
        lib.oracle_gauss_legendre.argtypes = [ctypes.c_int, _DP, _DP]
        lib.oracle_operators.argtypes = [ctypes.c_int] + [_DP] * 6
        lib.oracle_lserk45.argtypes = [_DP, _DP]
        lib.oracle_lserk45.restype = None
        for f in (lib.oracle_volume_term, lib.oracle_surface_term, lib.oracle_residual):
            f.argtypes = mesh + [_DP, _DP]
        lib.oracle_rk_step.argtypes = mesh + [_DP, ctypes.c_double, ctypes.c_int]
        _IP = ctypes.POINTER(ctypes.c_int)
        lib.oracle_residual_bc.argtypes = mesh + [_IP, _DP, _DP, _DP]
        lib.oracle_rk_step_bc.argtypes = mesh + [_IP, _DP, _DP, ctypes.c_double, ctypes.c_int]
        lib.oracle_max_wavespeed.argtypes = [ctypes.c_int] * 4 + [ctypes.c_double, _DP, _DP]
        lib.oracle_gradient.argtypes = [ctypes.c_int] * 4 + [_DP, ctypes.c_int, _DP, _DP]
        visc = mesh + [ctypes.c_double, ctypes.c_double]
        lib.oracle_viscous_term.argtypes = visc + [_DP, _DP]
        lib.oracle_residual_ns.argtypes = visc + [_DP, _DP]
        lib.oracle_rk_step_ns.argtypes = visc + [_DP, ctypes.c_double, ctypes.c_int]
        _LIBS[name] = lib
    return _LIBS[name]


def _p(a):
    return a.ctypes.data_as(_DP)


def _check(rc, what):
    if rc != 0:
        raise ValueError(f"oracle: {what} rejected its arguments (rc={rc})")


class Oracle:
    """One build variant of the oracle: 'fp64' (parity), 'ld' (long-double arbiter), 'omp', 'ld_omp'."""

    def __init__(self, variant="fp64"):
        self.variant = variant
        self.lib = _load(variant)

    @property
    def real_bytes(self):
        return self.lib.oracle_real_bytes()

    @property
    def threads(self):
        return self.lib.oracle_threads()

    def gauss_legendre(self, N):
        xi = np.empty(N)
        w = np.empty(N)
        _check(self.lib.oracle_gauss_legendre(N, _p(xi), _p(w)), "gauss_legendre")
        return xi, w

    def operators(self, N):
        """xi, w, D[q,i] = l_i'(xi_q), lp, lm, Dhat[i,q] = w_q D[q,i] / w_i."""
        xi, w, lp, lm = (np.empty(N) for _ in range(4))
        D = np.empty((N, N))
        Dhat = np.empty((N, N))
        _check(self.lib.oracle_operators(N, _p(xi), _p(w), _p(D), _p(lp), _p(lm), _p(Dhat)), "operators")
        return dict(xi=xi, w=w, D=D, lp=lp, lm=lm, Dhat=Dhat)

    def lserk45(self):
        A = np.empty(5)
        B = np.empty(5)
        self.lib.oracle_lserk45(_p(A), _p(B))
        return A, B

    @staticmethod
    def _mesh(q, p):
        q = np.ascontiguousarray(q, dtype=np.float64)
        N = p + 1
        if q.ndim != 7 or q.shape[3:] != (N, N, N, 5):
            raise ValueError(f"q must have shape (nz,ny,nx,{N},{N},{N},5), got {q.shape}")
        nz, ny, nx = q.shape[:3]
        return q, nx, ny, nz

    def _term(self, fn, q, p, gamma, extent):
        q, nx, ny, nz = self._mesh(q, p)
        ext = np.asarray(extent, dtype=np.float64)
        r = np.empty_like(q)
        _check(fn(nx, ny, nz, p, float(gamma), _p(ext), _p(q), _p(r)), "residual term")
        return r

    def volume_term(self, q, p, gamma, extent):
        return self._term(self.lib.oracle_volume_term, q, p, gamma, extent)

    def surface_term(self, q, p, gamma, extent):
        return self._term(self.lib.oracle_surface_term, q, p, gamma, extent)

    def residual(self, q, p, gamma, extent):
        return self._term(self.lib.oracle_residual, q, p, gamma, extent)

    def rk_step(self, q, p, gamma, extent, dt, nsteps):
        q, nx, ny, nz = self._mesh(q, p)
        q = q.copy()
        ext = np.asarray(extent, dtype=np.float64)
        _check(self.lib.oracle_rk_step(nx, ny, nz, p, float(gamma), _p(ext), _p(q), float(dt), int(nsteps)),
               "rk_step")
        return q

    @staticmethod
    def _bc(bc, qinf):
        b = (ctypes.c_int * 6)(*[int(v) for v in bc])
        qi = np.ascontiguousarray(qinf if qinf is not None else np.zeros(5), dtype=np.float64)
        return b, qi

    def residual_bc(self, q, p, gamma, extent, bc, qinf=None):
        """dQ/dt with non-periodic faces: bc = (x-, x+, y-, y+, z-, z+), 0 periodic, 1 slip wall, 2 far field."""
        q, nx, ny, nz = self._mesh(q, p)
        ext = np.asarray(extent, dtype=np.float64)
        b, qi = self._bc(bc, qinf)
        r = np.empty_like(q)
        _check(self.lib.oracle_residual_bc(nx, ny, nz, p, float(gamma), _p(ext), b, _p(qi), _p(q), _p(r)), "residual_bc")
        return r

    def rk_step_bc(self, q, p, gamma, extent, bc, qinf, dt, nsteps):
        q, nx, ny, nz = self._mesh(q, p)
        q = q.copy()
        ext = np.asarray(extent, dtype=np.float64)
        b, qi = self._bc(bc, qinf)
        _check(self.lib.oracle_rk_step_bc(nx, ny, nz, p, float(gamma), _p(ext), b, _p(qi), _p(q), float(dt), int(nsteps)),
               "rk_step_bc")
        return q

    def max_wavespeed(self, q, p, gamma):
        q, nx, ny, nz = self._mesh(q, p)
        lam = np.zeros(1)
        _check(self.lib.oracle_max_wavespeed(nx, ny, nz, p, float(gamma), _p(q), _p(lam)), "max_wavespeed")
        return float(lam[0])

    # ---- viscous (Navier-Stokes) terms, SURVEY.md 8(f)-4 (reading R20) ----
    def gradient(self, q, p, extent, axis):
        """BR1 gradient d_axis Q of the five conserved variables (central interface value)."""
        q, nx, ny, nz = self._mesh(q, p)
        ext = np.asarray(extent, dtype=np.float64)
        s = np.empty_like(q)
        _check(self.lib.oracle_gradient(nx, ny, nz, p, _p(ext), int(axis), _p(q), _p(s)), "gradient")
        return s

    def _visc(self, fn, q, p, gamma, extent, mu, prandtl):
        q, nx, ny, nz = self._mesh(q, p)
        ext = np.asarray(extent, dtype=np.float64)
        r = np.empty_like(q)
        _check(fn(nx, ny, nz, p, float(gamma), _p(ext), float(mu), float(prandtl), _p(q), _p(r)), "viscous term")
        return r

    def viscous_term(self, q, p, gamma, extent, mu, prandtl):
        """div Fv(Q, grad Q): the viscous part of dQ/dt."""
        return self._visc(self.lib.oracle_viscous_term, q, p, gamma, extent, mu, prandtl)

    def residual_ns(self, q, p, gamma, extent, mu, prandtl):
        return self._visc(self.lib.oracle_residual_ns, q, p, gamma, extent, mu, prandtl)

    def rk_step_ns(self, q, p, gamma, extent, mu, prandtl, dt, nsteps):
        q, nx, ny, nz = self._mesh(q, p)
        q = q.copy()
        ext = np.asarray(extent, dtype=np.float64)
        _check(self.lib.oracle_rk_step_ns(nx, ny, nz, p, float(gamma), _p(ext), float(mu), float(prandtl), _p(q),
                                          float(dt), int(nsteps)), "rk_step_ns")
        return q

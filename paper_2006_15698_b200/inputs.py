"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs 1-5).

This module serves BOTH the CUDA path's tests/bench and the oracle's tests, and therefore
holds none of the method's arithmetic: no differentiation, no flux, no Runge-Kutta, and no
operator construction of its own.  Node coordinates come from numpy's library routine
`numpy.polynomial.legendre.leggauss` (the paper's "Gauss-Legendre quadrature" points,
PAPER.md:80); primitive -> conserved is the definition of the state vector (PAPER.md:45-50,
eq (2)-(3)), needed to state an initial condition at all.  It imports neither `oracle` nor the
CUDA binding.

The paper says only "a periodic domain" about its benchmark field; the fields
below are the synthetic stand-ins fixed in SURVEY.md section 8(d) / DESIGN.md "input recipe".

Arrays are float64 with shape (nz, ny, nx, N, N, N, 5) in C order = the canonical layout
`q[((((e*N+k)*N+j)*N+i)*5+n]`, e = ex + nx*(ey + ny*ez)  (include/dg_b200.h).

Every generator takes `box=((x0,x1),(y0,y1),(z0,z1))` (element index ranges, periodic wrap) to
produce a sub-box of the full periodic field: node coordinates and per-node random numbers are
those of the full mesh, so a sub-box equals the corresponding slice of the full field.
`xp` may be numpy (default) or torch (with `device=`) for the analytic fields.
"""
import math

import numpy as np

GAMMA = 1.4


def gl_nodes(N):
    """N Gauss-Legendre points on [-1,1], ascending (numpy library routine)."""
    xi, _ = np.polynomial.legendre.leggauss(N)
    return xi


# ------------------------------------------------------------------------------------------
# mesh helpers
# ------------------------------------------------------------------------------------------
def _elem_indices(n, rng):
    if rng is None:
        return np.arange(n, dtype=np.int64)
    lo, hi = rng
    return np.mod(np.arange(lo, hi, dtype=np.int64), n)


def _as_xp(a, xp, device):
    if xp is np:
        return a
    return xp.as_tensor(a, dtype=xp.float64, device=device)


def node_coords(nx, ny, nz, p, extent, box=None, xp=np, device=None):
    """Broadcastable node coordinates X (1,1,nx',1,1,N), Y (1,ny',1,1,N,1), Z (nz',1,1,N,1,1)."""
    N = p + 1
    xi = gl_nodes(N)
    out = []
    shapes = [(1, 1, -1, 1, 1, N), (1, -1, 1, 1, N, 1), (-1, 1, 1, N, 1, 1)]
    for a, n in enumerate((nx, ny, nz)):
        idx = _elem_indices(n, None if box is None else box[a])
        h = extent[a] / n
        c = (idx[:, None].astype(np.float64) + 0.5 * (xi[None, :] + 1.0)) * h
        out.append(_as_xp(c.reshape(shapes[a]), xp, device))
    return out


def primitive_to_conserved(rho, u, v, w, p, gamma=GAMMA, xp=np):
    """Q = (rho, rho u, rho v, rho w, rho E), rho E = p/(gamma-1) + rho (u^2+v^2+w^2)/2  (eq 3)."""
    rho, u, v, w, p = xp.broadcast_arrays(rho, u, v, w, p) if xp is np else xp.broadcast_tensors(rho, u, v, w, p)
    E = p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w)
    return xp.stack([rho, rho * u, rho * v, rho * w, E], -1)


def uniform_state(nx, ny, nz, p, rho=1.0, vel=(0.3, 0.2, 0.1), pres=1.0, gamma=GAMMA):
    """Free stream: the same conserved vector at every node."""
    N = p + 1
    one = np.ones((nz, ny, nx, N, N, N))
    return np.ascontiguousarray(
        primitive_to_conserved(rho * one, vel[0] * one, vel[1] * one, vel[2] * one, pres * one, gamma))


# ------------------------------------------------------------------------------------------
# counter-based random numbers (splitmix64): value id -> U[0,1)
# ------------------------------------------------------------------------------------------
def splitmix64(x):
    """One splitmix64 output per 64-bit input counter (numpy uint64, wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = x.astype(np.uint64) + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def _unit(x):
    return (x >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def node_noise(nx, ny, nz, p, seed, amplitude, box=None):
    """i.i.d. U(-amplitude, amplitude) per conserved value, keyed by the GLOBAL value index."""
    N = p + 1
    ix = _elem_indices(nx, None if box is None else box[0]).astype(np.uint64)
    iy = _elem_indices(ny, None if box is None else box[1]).astype(np.uint64)
    iz = _elem_indices(nz, None if box is None else box[2]).astype(np.uint64)
    e = (ix[None, None, :] + np.uint64(nx) * (iy[None, :, None] + np.uint64(ny) * iz[:, None, None]))
    loc = np.arange(N * N * N * 5, dtype=np.uint64).reshape(N, N, N, 5)
    ids = e[..., None, None, None, None] * np.uint64(N * N * N * 5) + loc
    with np.errstate(over="ignore"):
        key = splitmix64(np.asarray([seed], dtype=np.uint64))[0]
        u = _unit(splitmix64(ids ^ key))
    return (2.0 * u - 1.0) * amplitude


# ------------------------------------------------------------------------------------------
# config 1: advecting density wave + seeded noise   (exact Euler solution without the noise)
# ------------------------------------------------------------------------------------------
def density_wave(nx, ny, nz, p, extent=(1.0, 1.0, 1.0), t=0.0, vel=(0.5, 0.5, 0.5), amp=0.2,
                 noise=0.0, seed=1, gamma=GAMMA, box=None, waves=(1, 1, 1)):
    """rho = 1 + amp sin(2 pi (kx x/Lx + ky y/Ly + kz z/Lz - (k.vel/L) t)), u=v=w=const, p=1."""
    X, Y, Z = node_coords(nx, ny, nz, p, extent, box)
    ph = (waves[0] * (X - vel[0] * t) / extent[0] + waves[1] * (Y - vel[1] * t) / extent[1]
          + waves[2] * (Z - vel[2] * t) / extent[2])
    rho = 1.0 + amp * np.sin(2.0 * math.pi * ph)
    one = np.ones_like(rho)
    q = primitive_to_conserved(rho, vel[0] * one, vel[1] * one, vel[2] * one, one, gamma)
    if noise:
        q = q + node_noise(nx, ny, nz, p, seed, noise, box)
    return np.ascontiguousarray(q)


# ------------------------------------------------------------------------------------------
# config 2: isentropic vortex extruded in z          (exact Euler solution, translating in x)
# ------------------------------------------------------------------------------------------
def isentropic_vortex(nx, ny, nz, p, extent=(10.0, 10.0, 2.5), t=0.0, beta=5.0, u0=0.5,
                      centre=(5.0, 5.0), gamma=GAMMA, box=None):
    X, Y, Z = node_coords(nx, ny, nz, p, extent, box)
    xc = centre[0] + u0 * t
    dx = X - xc
    dx = dx - extent[0] * np.round(dx / extent[0])  # nearest periodic image
    dy = Y - centre[1]
    dy = dy - extent[1] * np.round(dy / extent[1])
    r2 = dx * dx + dy * dy + 0.0 * Z
    f = beta / (2.0 * math.pi) * np.exp(0.5 * (1.0 - r2))
    T = 1.0 - (gamma - 1.0) * beta * beta / (8.0 * gamma * math.pi ** 2) * np.exp(1.0 - r2)
    rho = T ** (1.0 / (gamma - 1.0))
    pres = rho ** gamma
    u = u0 - f * dy
    v = f * dx
    return np.ascontiguousarray(primitive_to_conserved(rho, u, v, 0.0 * rho, pres, gamma))


# ------------------------------------------------------------------------------------------
# configs 3 and 5: Taylor-Green vortex at Mach 0.1 (rho uniform)
# ------------------------------------------------------------------------------------------
def taylor_green(nx, ny, nz, p, extent=None, mach=0.1, gamma=GAMMA, box=None, xp=np, device=None):
    if extent is None:
        extent = (2.0 * math.pi,) * 3
    X, Y, Z = node_coords(nx, ny, nz, p, extent, box, xp, device)
    p0 = 1.0 / (gamma * mach * mach)
    u = xp.sin(X) * xp.cos(Y) * xp.cos(Z)
    v = -xp.cos(X) * xp.sin(Y) * xp.cos(Z)
    pres = p0 + (xp.cos(2.0 * X) + xp.cos(2.0 * Y)) * (xp.cos(2.0 * Z) + 2.0) / 16.0
    rho = xp.ones_like(pres)
    q = primitive_to_conserved(rho, u, v, 0.0 * rho, pres, gamma, xp)
    return np.ascontiguousarray(q) if xp is np else q.contiguous()


# ------------------------------------------------------------------------------------------
# config 4: free stream + seeded sum of 8 low-wavenumber Fourier modes per variable
# ------------------------------------------------------------------------------------------
def fourier_mode_table(seed=4, nmodes=8):
    """(k[5,nmodes,3] integer wavevectors in {-2..2}^3 \\ {0}, phi[5,nmodes] in [0,2pi))."""
    ctr = np.uint64(0)
    key = splitmix64(np.asarray([seed], dtype=np.uint64))[0]

    def draw():
        nonlocal ctr
        with np.errstate(over="ignore"):
            val = _unit(splitmix64(np.asarray([ctr], dtype=np.uint64) ^ key))[0]
            ctr = ctr + np.uint64(1)
        return val

    k = np.zeros((5, nmodes, 3), dtype=np.int64)
    phi = np.zeros((5, nmodes))
    for n in range(5):
        for m in range(nmodes):
            while True:
                kv = [int(draw() * 5.0) - 2 for _ in range(3)]
                if any(kv):
                    break
            k[n, m] = kv
            phi[n, m] = 2.0 * math.pi * draw()
    return k, phi


def fourier_modes(nx, ny, nz, p, extent=(1.0, 1.0, 1.0), seed=4, amplitude=1e-2, nmodes=8,
                  rho=1.0, vel=(0.3, 0.2, 0.1), pres=1.0, gamma=GAMMA, box=None, xp=np, device=None):
    """Q_n = Qinf_n + (amplitude/nmodes) sum_m cos(2 pi k_nm . x/L + phi_nm); |delta| <= amplitude."""
    X, Y, Z = node_coords(nx, ny, nz, p, extent, box, xp, device)
    k, phi = fourier_mode_table(seed, nmodes)
    qinf = primitive_to_conserved(*(np.float64(c) for c in (rho, vel[0], vel[1], vel[2], pres)), gamma)
    two_pi = 2.0 * math.pi
    shape = (Z.shape[0], Y.shape[1], X.shape[2], Z.shape[3], Y.shape[4], X.shape[5])
    fields = []
    for n in range(5):
        acc = xp.zeros(shape, dtype=xp.float64) if xp is np else xp.zeros(shape, dtype=xp.float64, device=device)
        for m in range(nmodes):
            # cos(a+b+c+phi) expanded so that only 1-D factors meet the transcendental functions
            a = two_pi * float(k[n, m, 0]) / extent[0] * X
            b = two_pi * float(k[n, m, 1]) / extent[1] * Y
            c = two_pi * float(k[n, m, 2]) / extent[2] * Z + float(phi[n, m])
            cab = xp.cos(a) * xp.cos(b) - xp.sin(a) * xp.sin(b)
            sab = xp.sin(a) * xp.cos(b) + xp.cos(a) * xp.sin(b)
            acc = acc + (cab * xp.cos(c) - sab * xp.sin(c))
        fields.append(float(qinf[n]) + (amplitude / nmodes) * acc)
    q = xp.stack(fields, -1)
    return np.ascontiguousarray(q) if xp is np else q.contiguous()


# ------------------------------------------------------------------------------------------
# the five BASELINE.json configurations
# ------------------------------------------------------------------------------------------
def cfg4_elems_per_side(p):
    """round((2e8 / (5 (p+1)^3))^(1/3))  ->  171,114,85,68,57,49,43 for p = 1..7."""
    return int(round((2.0e8 / (5.0 * (p + 1) ** 3)) ** (1.0 / 3.0)))


CONFIGS = {
    "cfg1": dict(nx=4, ny=4, nz=4, p=1, extent=(1.0, 1.0, 1.0), field="density_wave", steps=10),
    "cfg2": dict(nx=16, ny=16, nz=4, p=3, extent=(10.0, 10.0, 2.5), field="isentropic_vortex", steps=100),
    "cfg3": dict(nx=64, ny=64, nz=64, p=4, extent=(2.0 * math.pi,) * 3, field="taylor_green", steps=50),
    "cfg5": dict(nx=96, ny=96, nz=96, p=7, extent=(2.0 * math.pi,) * 3, field="taylor_green", steps=10),
}
# per-GPU share of the paper's Table II run: 512 x 512 x 768 elements at p = 6 over 3,072 GPUs
# = 65,536 elements = 22.5 M nodes per GPU; 40^3 = 64,000 elements (21.95 M nodes) stands in for it
CONFIGS["table2_p6"] = dict(nx=40, ny=40, nz=40, p=6, extent=(1.0, 1.0, 1.0), field="fourier_modes", steps=10)
for _p in range(1, 8):
    _n = cfg4_elems_per_side(_p)
    CONFIGS[f"cfg4_p{_p}"] = dict(nx=_n, ny=_n, nz=_n, p=_p, extent=(1.0, 1.0, 1.0), field="fourier_modes", steps=20)


def make_field(cfg, box=None, xp=np, device=None, override=None):
    """Initial state of a named config (or of a dict with the same keys); optional sub-box."""
    c = dict(CONFIGS[cfg]) if isinstance(cfg, str) else dict(cfg)
    if override:
        c.update(override)
    nx, ny, nz, p, ext, field = c["nx"], c["ny"], c["nz"], c["p"], c["extent"], c["field"]
    if field == "density_wave":
        return density_wave(nx, ny, nz, p, ext, noise=1e-3, seed=1, box=box)
    if field == "isentropic_vortex":
        return isentropic_vortex(nx, ny, nz, p, ext, box=box)
    if field == "taylor_green":
        return taylor_green(nx, ny, nz, p, ext, box=box, xp=xp, device=device)
    if field == "fourier_modes":
        return fourier_modes(nx, ny, nz, p, ext, seed=4, box=box, xp=xp, device=device)
    raise KeyError(field)


def cfl_dt(lam_max, p, extent, n, cfl=0.1):
    """dt = CFL min(h_a) / ((2p+1) lam_max)   (reading R10; harness-side, not parity)."""
    h = min(extent[a] / n[a] for a in range(3))
    return cfl * h / ((2 * p + 1) * lam_max)

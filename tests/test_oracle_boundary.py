"""Pins of the oracle's non-periodic boundary conditions (reading R19 -- the paper has
none, "periodic domain").  CPU only.  The PERIODIC oracle is pinned elsewhere (brute force, conservation,
convergence); these tests tie the wall / far-field code to it and to what the mathematics fixes:

* slip wall == mirror image: a state that is mirror-symmetric about a plane (normal momentum odd, everything else
  even) has, on the periodic mesh of doubled length, exactly the ghost state "interior trace with the normal momentum
  negated" on the other side of that plane.  So the residual of the half mesh with walls on that axis must equal the
  periodic residual of the doubled mesh restricted to the half, for each axis and for all three at once;
* far field: a uniform state with the same state as exterior gives a zero residual (free-stream preservation), on
  every face; and a far-field exterior equal to the wall ghost of a mirror-symmetric state reproduces the wall result;
* conservation: with walls on all six faces mass and energy integrals of dQ/dt vanish to roundoff (no flux through a
  wall: the interface flux of a state and its mirror image has zero mass and energy components), momentum does not;
* LSERK45 with boundaries: the mirrored periodic run and the wall run stay equal over several steps.
"""
import numpy as np
import pytest

import dg_bruteforce as bf
from oracle import Oracle
from paper_2006_15698_b200 import inputs as I

G = 1.4
ORC = Oracle("fp64")
PER, WALL, FAR = 0, 1, 2


def relerr(a, b):
    return max(np.abs(a[..., n] - b[..., n]).max() / max(np.abs(b[..., n]).max(), 1e-300) for n in range(5))


def mirror(q, axis):
    """Mirror image of a canonical state array (nz,ny,nx,k,j,i,n) about the high face of `axis` (0 x, 1 y, 2 z):
    elements and nodes reversed along the axis (Gauss-Legendre nodes are symmetric), normal momentum negated."""
    elem_ax, node_ax = {0: (2, 5), 1: (1, 4), 2: (0, 3)}[axis]
    m = np.flip(np.flip(q, elem_ax), node_ax).copy()
    m[..., 1 + axis] *= -1.0
    return m


def doubled(q, axis):
    elem_ax = {0: 2, 1: 1, 2: 0}[axis]
    return np.ascontiguousarray(np.concatenate([q, mirror(q, axis)], axis=elem_ax))


def field(nx, ny, nz, p, ext, seed=4):
    return I.density_wave(nx, ny, nz, p, ext, vel=(0.4, -0.3, 0.2), noise=3e-2, seed=seed, waves=(1, 1, 2))


@pytest.mark.parametrize("p", [1, 2, 4])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_slip_wall_equals_the_periodic_residual_of_the_mirrored_mesh(p, axis):
    n, ext = [3, 2, 4], [1.0, 0.7, 1.3]
    q = field(*n, p, ext)
    bc = [PER] * 6
    bc[2 * axis] = bc[2 * axis + 1] = WALL
    r_wall = ORC.residual_bc(q, p, G, ext, bc)
    ext2 = list(ext)
    ext2[axis] *= 2
    r_per = ORC.residual(doubled(q, axis), p, G, ext2)
    half = [slice(None)] * 7
    half[{0: 2, 1: 1, 2: 0}[axis]] = slice(0, n[axis])
    assert relerr(r_wall, r_per[tuple(half)]) < 1e-13, (p, axis)
    assert relerr(r_wall, ORC.residual(q, p, G, ext)) > 1e-3      # and the wall is not the periodic neighbour


def test_walls_on_all_axes_and_runge_kutta_steps_match_the_mirrored_periodic_run():
    p, n, ext = 2, [2, 3, 2], [1.0, 1.2, 0.8]
    q = field(*n, p, ext, seed=9)
    big = doubled(doubled(doubled(q, 0), 1), 2)
    ext2 = [2 * e for e in ext]
    sl = (slice(0, n[2]), slice(0, n[1]), slice(0, n[0]))
    assert relerr(ORC.residual_bc(q, p, G, ext, [WALL] * 6), ORC.residual(big, p, G, ext2)[sl]) < 1e-13
    dt = 2e-3
    q_wall = ORC.rk_step_bc(q, p, G, ext, [WALL] * 6, None, dt, 5)
    assert relerr(q_wall, ORC.rk_step(big, p, G, ext2, dt, 5)[sl]) < 1e-13


@pytest.mark.parametrize("p", [1, 3])
def test_far_field_free_stream_and_far_field_as_wall_ghost(p):
    n, ext = [3, 3, 2], [1.0, 1.0, 0.5]
    qu = I.uniform_state(*n, p, rho=1.1, vel=(0.3, -0.2, 0.4), pres=0.9, gamma=G)
    qinf = qu.reshape(-1, 5)[0].copy()
    for bc in ([FAR] * 6, [FAR, FAR, PER, PER, WALL, WALL], [PER, PER, FAR, FAR, PER, PER]):
        if WALL in bc:            # a wall is not transparent to a free stream with a normal velocity: use w = 0 there
            quw = I.uniform_state(*n, p, rho=1.1, vel=(0.3, -0.2, 0.0), pres=0.9, gamma=G)
            r = ORC.residual_bc(quw, p, G, ext, bc, quw.reshape(-1, 5)[0].copy())
        else:
            r = ORC.residual_bc(qu, p, G, ext, bc, qinf)
        assert np.abs(r).max() < 5e-13, (p, bc, np.abs(r).max())
    # a far field whose state differs from the interior produces a residual only in the boundary elements
    q = field(*n, p, ext)
    r_far = ORC.residual_bc(q, p, G, ext, [FAR, FAR, PER, PER, PER, PER], qinf)
    r_per = ORC.residual(q, p, G, ext)
    assert np.array_equal(r_far[:, :, 1:-1], r_per[:, :, 1:-1])
    assert relerr(r_far[:, :, :1], r_per[:, :, :1]) > 1e-3


@pytest.mark.parametrize("p", [1, 3])
@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("side", [0, 1])
def test_far_field_equal_to_the_wall_ghost_reproduces_the_wall(p, axis, side):
    """The far-field branch with an exterior state that DIFFERS from the interior, pinned by the wall branch: for a
    state that varies along one axis only, the trace on a face of that axis is one and the same state at every face
    node, so its wall ghost (normal momentum negated) can be handed over as q_inf.  Far field on that face (low and
    high in turn), wall on the opposite one, must then give the residual of walls on both."""
    n, ext = [3, 2, 4], [1.0, 0.7, 1.3]
    q3 = field(*n, p, ext, seed=7)
    elem_ax, node_ax = {0: (2, 5), 1: (1, 4), 2: (0, 3)}[axis]
    keep = [slice(0, 1)] * 6 + [slice(None)]
    keep[elem_ax] = keep[node_ax] = slice(None)
    q = np.ascontiguousarray(np.broadcast_to(q3[tuple(keep)], q3.shape))       # varies along `axis` only
    _, _, _, lp, lm = bf.basis_1d(p + 1)                                          # l_i(+1), l_i(-1): numpy, not the oracle's
    line = np.moveaxis(q, (elem_ax, node_ax), (0, 1))[:, :, 0, 0, 0, 0, :]       # (element, node, variable) along the axis
    trace = lp @ line[-1] if side else lm @ line[0]
    ghost = trace.copy()
    ghost[1 + axis] *= -1.0
    bc_far, bc_wall = [PER] * 6, [PER] * 6
    bc_wall[2 * axis] = bc_wall[2 * axis + 1] = WALL
    bc_far[2 * axis + side], bc_far[2 * axis + 1 - side] = FAR, WALL
    r_far = ORC.residual_bc(q, p, G, ext, bc_far, ghost)
    r_wall = ORC.residual_bc(q, p, G, ext, bc_wall)
    assert relerr(r_far, r_wall) < 1e-13, (p, axis, side, relerr(r_far, r_wall))
    # and the pin bites: the un-negated trace as exterior state (a transparent face) gives another residual
    assert relerr(ORC.residual_bc(q, p, G, ext, bc_far, trace), r_wall) > 1e-3


@pytest.mark.parametrize("p", [1, 3])
def test_walls_conserve_mass_and_energy(p):
    n, ext = [3, 2, 3], [1.0, 0.8, 1.1]
    q = field(*n, p, ext, seed=2)
    r = ORC.residual_bc(q, p, G, ext, [WALL] * 6)
    tot = bf.integrals(r, p, ext)
    scale = bf.integrals(np.abs(r), p, ext)
    assert abs(tot[0]) < 1e-14 * scale[0] and abs(tot[4]) < 1e-14 * scale[4]
    assert max(abs(tot[1]), abs(tot[2]), abs(tot[3])) > 1e-6 * scale[1]      # walls do exert a force


def test_boundary_arguments_are_validated():
    q = field(2, 2, 2, 1, [1.0] * 3)
    with pytest.raises(ValueError):
        ORC.residual_bc(q, 1, G, [1.0] * 3, [WALL, PER, PER, PER, PER, PER])       # periodic on one face only
    with pytest.raises(ValueError):
        ORC.residual_bc(q, 1, G, [1.0] * 3, [3, 3, PER, PER, PER, PER])
    assert np.array_equal(ORC.residual_bc(q, 1, G, [1.0] * 3, [PER] * 6), ORC.residual(q, 1, G, [1.0] * 3))

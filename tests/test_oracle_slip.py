"""Pins of the oracle's full-slip walls (reading G37: specular reflection at halfway walls).

W1 a box closed by slip walls in y and z IS the mirror-extended periodic box: the fluid cells of the slip box after n steps equal,
   to rounding, the corresponding cells of a wall-free periodic run on the 2(ny-2) x 2(nz-2) mirror image of the initial state
   (streaming of that run is pinned against numpy.roll) -- fixes the reflected index, the source cell, edges and corners;
W2 free slip: tangential momentum and mass of a slip channel are conserved, the wall-normal momentum is not;
W3 uniform flow along slip walls is a fixed point (bounce-back walls would brake it); a wall at the reflected source falls back
   to bounce-back.
CPU only."""
import numpy as np
import pytest

import lbm_inputs as I
from oracle import oracle as O

NT = min(8, O.max_threads())


def _slip_box(nz, ny, nx):
    flags = np.zeros((nz, ny, nx), dtype=np.uint8)
    flags[0] = flags[-1] = I.SLIPWALL
    flags[:, 0] = flags[:, -1] = I.SLIPWALL
    return flags


def _mirror_perm(Q, axis):
    c, w, opp = O.lattice(Q)
    perm = np.empty(Q, dtype=int)
    for i in range(Q):
        m = c[i].copy()
        m[axis] = -m[axis]
        perm[i] = next(j for j in range(Q) if (c[j] == m).all())
    return perm


@pytest.mark.parametrize("Q", [19, 27])
@pytest.mark.parametrize("coll", [0, 1])
def test_W1_slip_box_is_the_mirror_extended_periodic_box(Q, coll):
    nz, ny, nx = 8, 7, 10
    hz, hy = nz - 2, ny - 2
    rng = np.random.Generator(np.random.PCG64(7 + Q))
    rho = 1.0 + 0.02 * rng.standard_normal((hz, hy, nx))
    u = 0.04 * rng.standard_normal((3, hz, hy, nx))
    f_in = O.init_equilibrium(Q, rho, u) * (1 + 0.01 * rng.standard_normal((Q, hz, hy, nx)))
    # slip box: walls around the hz x hy fluid core
    flags = _slip_box(nz, ny, nx)
    f = np.tile(O.feq(Q, 1.0, [0, 0, 0])[:, None, None, None], (1, nz, ny, nx)).astype(float)
    f[:, 1:-1, 1:-1, :] = f_in
    par = dict(tau0=0.62, cs_smago=0.1, collision=coll, sigma=0.6)
    got = O.step(f, flags=flags, nsteps=6, **par)[:, 1:-1, 1:-1, :]
    # mirror extension: y' in [0, 2 hy): cells hy..2hy-1 are the mirror image (y -> 2 hy - 1 - y, c_y -> -c_y); the same in z
    py, pz = _mirror_perm(Q, 1), _mirror_perm(Q, 2)
    ext = np.concatenate([f_in, f_in[py][:, :, ::-1, :]], axis=2)
    ext = np.concatenate([ext, ext[pz][:, ::-1, :, :]], axis=1)
    ref = O.step(ext, flags=None, nsteps=6, **par)[:, :hz, :hy, :]
    if coll == 0:
        assert np.abs(got - ref).max() <= 1e-15
    else:
        # HRR: the FD stencil of the slip box sees u^ = 0 on the wall cells where the mirror box sees the mirrored neighbour
        # (G30): cells next to the walls differ at O(sigma-blend of the strain); the core of the equivalence is the BGK case
        assert np.isfinite(got).all()


def test_W2_free_slip_conserves_tangential_momentum():
    nz, ny, nx = 10, 12, 16
    flags = np.zeros((nz, ny, nx), dtype=np.uint8)
    flags[0] = flags[-1] = I.SLIPWALL                       # slip floor and top, periodic in x and y
    rng = np.random.Generator(np.random.PCG64(11))
    rho = 1.0 + 0.02 * rng.standard_normal(flags.shape)
    u = 0.04 * rng.standard_normal((3,) + flags.shape)
    u[2] += 0.02
    f = O.init_equilibrium(19, rho, u)
    t0 = O.totals(f, flags)
    g = O.step(f, flags=flags, nsteps=40, nthreads=NT, tau0=0.6, cs_smago=0.12)
    t1 = O.totals(g, flags)
    assert abs(t1[0] / t0[0] - 1.0) <= 1e-13
    assert abs(t1[1] - t0[1]) <= 1e-12 * t0[0] and abs(t1[2] - t0[2]) <= 1e-12 * t0[0]
    assert abs(t1[3] - t0[3]) > 1e-3 * abs(t0[3])           # the walls do take up normal momentum
    # the same channel with bounce-back walls loses tangential momentum
    fb = np.where(flags == I.SLIPWALL, I.SOLID, flags).astype(np.uint8)
    f2 = O.init_equilibrium(19, np.ones(flags.shape), np.broadcast_to(np.array([0.03, 0, 0])[:, None, None, None], (3,) + flags.shape).copy())
    tb0 = O.totals(f2, fb)
    tb = O.totals(O.step(f2, flags=fb, nsteps=40, nthreads=NT, tau0=0.6), fb)
    assert tb[1] < 0.97 * tb0[1]


@pytest.mark.parametrize("Q", [19, 27])
def test_W3_uniform_flow_fixed_point_and_fallback(Q):
    nz, ny, nx = 7, 6, 8
    flags = np.zeros((nz, ny, nx), dtype=np.uint8)
    flags[0] = flags[-1] = I.SLIPWALL
    uu = np.zeros((3,) + flags.shape)
    uu[0], uu[1] = 0.05, -0.02                              # tangential to the z walls
    f = O.init_equilibrium(Q, np.ones(flags.shape), uu)
    g = O.step(f, flags=flags, nsteps=25, tau0=0.7)
    fluid = ~I.is_wall(flags)
    assert np.abs(g[:, fluid] - f[:, fluid]).max() <= 1e-15
    # a SOLID block standing on the slip floor: where the reflected source is the block, the link bounces back; mass is kept
    flags[1:3, 2:4, 3:5] = I.SOLID
    f = O.init_equilibrium(Q, np.ones(flags.shape), np.where(I.is_wall(flags), 0.0, uu))
    t0 = O.totals(f, flags)
    t1 = O.totals(O.step(f, flags=flags, nsteps=30, tau0=0.7), flags)
    assert abs(t1[0] / t0[0] - 1.0) <= 1e-13 and t1[1] < t0[1]


@pytest.mark.parametrize("Q", [19, 27])
@pytest.mark.parametrize("coll", [0, 1])
def test_W4_wall_cells_are_inert_whatever_populations_they_hold(Q, coll):
    """Readings R5 / G30 / G37: SOLID and SLIPWALL cells are inert -- nothing a fluid cell computes may depend on the populations
    stored in them; in the HRR form the FD stencil sees u^ = 0 there (a resting wall), not the moment of those stored values.
    (Found by the GPU parity test from a non-equilibrium start: the oracle took u^ of SLIPWALL cells from their own populations,
    which only shows once those populations carry momentum.)"""
    nz, ny, nx = 9, 8, 12
    rng = np.random.Generator(np.random.PCG64(40 + Q + coll))
    flags = _slip_box(nz, ny, nx)
    flags[2:4, 2:4, 5:8] = I.SOLID
    rho = 1.0 + 0.02 * rng.standard_normal(flags.shape)
    u = 0.04 * rng.standard_normal((3,) + flags.shape)
    f = O.init_equilibrium(Q, rho, u) * (1 + 0.01 * rng.standard_normal((Q,) + flags.shape))
    wall = I.is_wall(flags)
    par = dict(tau0=0.58, cs_smago=0.1, collision=coll, sigma=0.5)
    a = O.step(f, flags=flags, nsteps=5, **par)
    g = f.copy()
    g[:, wall] = O.feq(Q, 1.3, [0.1, -0.2, 0.15])[:, None] * (1 + 0.3 * rng.uniform(-1, 1, size=(Q, int(wall.sum()))))
    b = O.step(g, flags=flags, nsteps=5, **par)
    assert np.array_equal(a[:, ~wall], b[:, ~wall])
    assert np.array_equal(b[:, wall], g[:, wall])                # and they keep what they hold

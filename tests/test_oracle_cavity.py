"""Pins of the oracle's moving-wall bounce-back (the lid of the paper's lid-driven cavity benchmark,
PAPER.md l.214; reading G33: g_i(x) = f*_opp(i)(x) + 2 w_i rho_w (c_i.u_w)/c_s^2, rho_w = 1, c_i from the wall into the fluid).

M1 plane Couette flow: the steady state between a resting and a moving halfway wall is the exact linear profile;
M2 one step from rest, written out from the hand-typed golden tables (which populations change, by how much);
M3 tangential momentum fed per wall cell and step = rho_w u_w / 3 (= c_s^2 rho_w u_w: lattice isotropy, both lattices);
M4 a wall moving along its normal feeds mass rho_w u_n per wall cell and step;
M5 the wall is inert and a resting MOVINGWALL (u_w = 0) is exactly a SOLID cell;
M6 HRR form next to the lid (the FD stencil sees u^ = u_w on the wall cell): Couette profile within 2 %.
Nothing here calls the oracle's own formulas for the expected values.  CPU only."""
import os

import numpy as np
import pytest

import lbm_inputs as I
from oracle import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")
NT = min(8, O.max_threads())


def _golden(Q):
    rows = [l.split() for l in open(os.path.join(GOLD, "d3q%d_R1.txt" % Q)) if l.strip() and not l.startswith("#")]
    c = np.array([[int(r[1]), int(r[2]), int(r[3])] for r in rows], dtype=int)
    w = np.array([int(r[4]) / int(r[5]) for r in rows])
    return c, w


def _channel(nz, ny=4, nx=4):
    """periodic in x, y; resting wall at z = 0, moving wall at z = nz-1"""
    flags = np.zeros((nz, ny, nx), dtype=np.uint8)
    flags[0] = I.SOLID
    flags[-1] = I.MOVINGWALL
    return flags


def _rest(Q, shape):
    return O.init_equilibrium(Q, np.ones(shape), np.zeros((3,) + shape))


@pytest.mark.parametrize("Q", [19, 27])
@pytest.mark.parametrize("tau", [0.8, 0.56])
def test_M1_couette_profile_is_exactly_linear(Q, tau):
    nz = 14
    flags = _channel(nz)
    uw = (0.04, -0.015, 0.0)
    f = _rest(Q, flags.shape)
    H = nz - 2
    nu = (tau - 0.5) / 3.0
    steps = int(32 * H * H / nu / 9.87) + 200            # 32 decay times of the slowest mode, exp(-nu pi^2 t / H^2)
    f = O.step(f, flags=flags, nsteps=steps, nthreads=NT, tau0=tau, u_wall=uw)
    rho, u = O.moments(f)
    z = np.arange(1, nz - 1)
    for a in (0, 1):
        want = uw[a] * (z - 0.5) / H                      # walls half a cell outside the last fluid nodes
        got = u[a, 1:-1].mean(axis=(1, 2))
        assert np.abs(got - want).max() <= 2e-9 * abs(uw[a]) + 1e-13
        assert np.abs(u[a, 1:-1] - got[:, None, None]).max() <= 1e-13
    assert np.abs(u[2, 1:-1]).max() <= 1e-13
    assert np.abs(rho[1:-1] - 1.0).max() <= 1e-10          # rounding of ~1e5 steps


@pytest.mark.parametrize("Q", [19, 27])
def test_M2_one_step_from_rest_by_hand(Q):
    c, w = _golden(Q)
    nz = 6
    flags = _channel(nz)
    uw = np.array([0.03, 0.02, -0.01])
    f0 = _rest(Q, flags.shape)
    f1 = O.step(f0, flags=flags, nsteps=1, tau0=0.7, u_wall=tuple(uw))
    # rest equilibrium is a fixed point of collide and of plain bounce-back; only the populations that return from the
    # lid (c_i = wall -> fluid, c_z = -1) in the lid-adjacent plane z = nz-2 change, by 6 w_i (c_i . u_w)
    want = np.broadcast_to(w[:, None, None, None], f0.shape).copy()
    for i in range(Q):
        if c[i, 2] == -1:
            want[i, nz - 2] += 6.0 * w[i] * float(c[i] @ uw)
    fluid = ~I.is_wall(flags)
    assert np.abs(f1[:, fluid] - want[:, fluid]).max() <= 1e-16
    assert np.array_equal(f1[:, ~fluid], f0[:, ~fluid])   # walls inert


@pytest.mark.parametrize("Q", [19, 27])
def test_M3_M4_momentum_and_mass_fed_per_wall_cell(Q):
    nz = 6
    flags = _channel(nz, ny=5, nx=6)
    ncells = 5 * 6
    f0 = _rest(Q, flags.shape)
    t0 = O.totals(f0, flags)
    # tangential: momentum rho_w u_w / 3 per wall cell, no mass
    f1 = O.step(f0, flags=flags, nsteps=1, tau0=0.9, u_wall=(0.06, -0.03, 0.0))
    t1 = O.totals(f1, flags)
    assert abs(t1[0] - t0[0]) <= 1e-12
    assert abs((t1[1] - t0[1]) / ncells - 0.06 / 3.0) <= 1e-13
    assert abs((t1[2] - t0[2]) / ncells + 0.03 / 3.0) <= 1e-13
    assert abs(t1[3] - t0[3]) <= 1e-13
    # normal: the lid moves into the fluid (-z) with speed 0.01: mass rho_w u_n per wall cell
    f2 = O.step(f0, flags=flags, nsteps=1, tau0=0.9, u_wall=(0.0, 0.0, -0.01))
    t2 = O.totals(f2, flags)
    assert abs((t2[0] - t0[0]) / ncells - 0.01) <= 1e-13


def test_M5_resting_moving_wall_is_a_solid_wall():
    cfg = I.make_config(6, shape=(10, 9, 8))
    rng = np.random.Generator(np.random.PCG64(5))
    rho = 1.0 + 0.01 * rng.standard_normal(cfg["shape"])
    u = 0.03 * rng.standard_normal((3,) + cfg["shape"])
    f = O.init_equilibrium(19, rho, u)
    solid = np.where(I.is_wall(cfg["flags"]), I.SOLID, I.FLUID).astype(np.uint8)
    a = O.step(f, flags=cfg["flags"], nsteps=5, tau0=0.6, cs_smago=0.1, u_wall=(0.0, 0.0, 0.0))
    b = O.step(f, flags=solid, nsteps=5, tau0=0.6, cs_smago=0.1)
    assert np.array_equal(a, b)
    # and with the lid moving, the closed box keeps its mass (tangential lid) while the fluid starts to follow the lid
    c = O.step(f, flags=cfg["flags"], nsteps=50, tau0=0.6, cs_smago=0.1, u_wall=(0.05, 0.0, 0.0))
    t0, t1 = O.totals(f, cfg["flags"]), O.totals(c, cfg["flags"])
    assert abs(t1[0] / t0[0] - 1.0) <= 1e-13
    _, uc = O.moments(c)
    assert uc[0, -2, 2:-2, 2:-2].mean() > 0.01           # the layer under the lid moves WITH the lid (sign of the term)


@pytest.mark.parametrize("sigma", [1.0, 0.0])
def test_M6_hrr_couette(sigma):
    nz = 18
    flags = _channel(nz)
    f = _rest(19, flags.shape)
    f = O.step(f, flags=flags, nsteps=6000, nthreads=NT, tau0=0.8, u_wall=(0.04, 0.0, 0.0), collision=1, sigma=sigma)
    _, u = O.moments(f)
    z = np.arange(1, nz - 1)
    want = 0.04 * (z - 0.5) / (nz - 2)
    got = u[0, 1:-1].mean(axis=(1, 2))
    assert np.isfinite(got).all()
    assert np.abs(got - want).max() <= 0.02 * 0.04

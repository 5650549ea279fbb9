"""Pins of the CPU oracle: prescribed solid velocity field u^B(x,t) of Eq. 12 (the moving porous bodies of
Fig. 1; O2b, reading G39) and time-varying porosity d(x,t).

U1 uniform periodic field: u(t) - u^B = (1 - d/tau)^t (u(0) - u^B), rho constant (closed form; BGK form and HRR form at sigma = 1);
U2 one body cell (d = 1, tau = 1) in a fluid at rest, junk u^B elsewhere under d = 0: after one step the total momentum is
   rho u^B of exactly that cell and the populations around it are f^eq(rho, u^B) streamed (fixes the cell index, the component
   order and that u^B enters with weight d);
U3 u^B = 0, or any u^B under d = 0, or use_hlbm = 0: bit-identical to the pinned plain step;
U4 WALLMODEL cells keep the wall model's u^B (reading G39): junk u_body on them changes nothing;
U5 shear flow between moving porous plates (d = 1, u^B = +-U): steady profile linear between the plates, extrapolating to +-U there;
U6 a body that moves (d(x,t), u^B(x,t) re-set every step) drags the fluid along: the momentum it feeds per step is the closed
   form sum_x d (u^B - u) rho / tau over the body cells (Eq. 12 in Eq. 6), step by step.
CPU only.
"""
import numpy as np
import pytest

import lbm_inputs as I
from oracle import oracle as O


@pytest.mark.parametrize("Q", [19, 27])
@pytest.mark.parametrize("collision", [0, 1])
def test_U1_uniform_relaxation_towards_solid_velocity(Q, collision):
    shape = (3, 4, 5)
    d0, tau0 = 0.3, 0.7
    rho0, u0, ub = 1.03, np.array([0.03, -0.02, 0.01]), np.array([-0.01, 0.025, 0.015])
    rho = np.full(shape, rho0)
    u = np.broadcast_to(u0[:, None, None, None], (3,) + shape).copy()
    f = O.init_equilibrium(Q, rho, u)
    d = np.full(shape, d0)
    u_body = np.broadcast_to(ub[:, None, None, None], (3,) + shape).copy()
    for n in range(1, 7):
        f = O.step(f, d=d, nsteps=1, u_body=u_body, tau0=tau0, use_hlbm=1, collision=collision, sigma=1.0)
        r, v = O.moments(f)
        assert np.abs(r - rho0).max() < 1e-14
        want = ub + (1.0 - d0 / tau0) ** n * (u0 - ub)
        assert np.abs(v - want[:, None, None, None]).max() < 1e-14


@pytest.mark.parametrize("Q", [19, 27])
def test_U2_single_body_cell_indexing_and_components(Q):
    c, w, _ = O.lattice(Q)
    nz, ny, nx = 5, 6, 7
    shape = (nz, ny, nx)
    cz, cy, cx = 1, 4, 2
    rng = np.random.default_rng(21)
    rho0 = 1.02
    f = O.init_equilibrium(Q, np.full(shape, rho0), np.zeros((3,) + shape))
    d = np.zeros(shape)
    d[cz, cy, cx] = 1.0
    u_body = 0.05 * rng.standard_normal((3,) + shape)        # junk everywhere (weight d = 0) ...
    ub = np.array([0.011, -0.023, 0.037])
    u_body[:, cz, cy, cx] = ub                               # ... except at the body cell
    got = O.step(f, d=d, nsteps=1, u_body=u_body, tau0=1.0, use_hlbm=1)
    t = O.totals(got)
    assert abs(t[0] - rho0 * nz * ny * nx) < 1e-12
    assert np.abs(t[1:4] - rho0 * ub).max() < 1e-13          # a sum over 210 cells
    # tau = 1, d = 1: the cell's post-collision state is f^eq(rho, u^B); one streaming step spreads it over the neighbours
    feq = O.feq(Q, rho0, ub)
    for i in range(Q):
        z, y, x = (cz + c[i][2]) % nz, (cy + c[i][1]) % ny, (cx + c[i][0]) % nx
        assert abs(got[i, z, y, x] - feq[i]) < 1e-16
    rest = O.feq(Q, rho0, np.zeros(3))
    changed = np.argwhere(np.abs(got - rest[:, None, None, None]) > 1e-15)
    assert len(changed) <= Q


def _channel(rng):
    nz, ny, nx = 7, 5, 10
    shape = (nz, ny, nx)
    flags = np.zeros(shape, dtype=np.uint8)
    flags[0] = I.SOLID
    flags[nz - 1] = I.SOLID
    flags[1:nz - 1, :, 0] = I.INLET
    flags[1:nz - 1, :, nx - 1] = I.OUTLET
    flags[1, :, 1:nx - 1] = I.WM_FLOOR
    d = np.zeros(shape)
    d[1, :, 1:nx - 1] = 1.0
    d[2:5, 1:4, 4:7] = rng.uniform(0.2, 1.0, size=(3, 3, 3))
    rho = 1.0 + 0.01 * rng.standard_normal(shape)
    u = 0.02 * rng.standard_normal((3,) + shape)
    u[0] += 0.04
    f = O.init_equilibrium(19, rho, u)
    par = dict(tau0=0.53, cs_smago=0.1, use_hlbm=1, u_in=(0.05, 0.0, 0.0), wm_enable=1)
    return shape, flags, d, f, par


@pytest.mark.parametrize("collision", [0, 1])
def test_U3_zero_solid_velocity_or_zero_porosity_is_the_plain_step(collision):
    rng = np.random.default_rng(22)
    shape, flags, d, f, par = _channel(rng)
    par = dict(par, collision=collision, sigma=0.7)
    plain = O.step(f, d=d, flags=flags, nsteps=4, **par)
    assert np.array_equal(O.step(f, d=d, flags=flags, nsteps=4, u_body=np.zeros((3,) + shape), **par), plain)
    junk = 0.05 * rng.standard_normal((3,) + shape)
    junk[:, d > 0] = 0.0                                     # u^B only where d = 0
    assert np.array_equal(O.step(f, d=d, flags=flags, nsteps=4, u_body=junk, **par), plain)
    par0 = dict(par, use_hlbm=0)
    junk = 0.05 * rng.standard_normal((3,) + shape)
    assert np.array_equal(O.step(f, d=d, flags=flags, nsteps=4, u_body=junk, **par0),
                          O.step(f, d=d, flags=flags, nsteps=4, **par0))
    # and a non-zero u^B inside the porous block does change the flow
    ub = np.zeros((3,) + shape)
    ub[1, 2:5, 1:4, 4:7] = 0.03
    assert np.abs(O.step(f, d=d, flags=flags, nsteps=4, u_body=ub, **par) - plain).max() > 1e-4


def test_U4_wallmodel_cells_keep_the_wall_models_velocity():
    rng = np.random.default_rng(23)
    shape, flags, d, f, par = _channel(rng)
    ub = np.zeros((3,) + shape)
    ub[0, 2:5, 1:4, 4:7] = -0.02
    ref = O.step(f, d=d, flags=flags, nsteps=3, u_body=ub, **par)
    ub2 = ub.copy()
    wm = (flags & 15) == I.WALLMODEL
    ub2[:, wm] = 0.05 * rng.standard_normal((3, int(wm.sum())))
    assert np.array_equal(O.step(f, d=d, flags=flags, nsteps=3, u_body=ub2, **par), ref)
    # with the wall model off those cells are ordinary porous cells and do see u_body
    off = dict(par, wm_enable=0)
    assert np.abs(O.step(f, d=d, flags=flags, nsteps=3, u_body=ub2, **off) - O.step(f, d=d, flags=flags, nsteps=3, u_body=ub, **off)).max() > 1e-4


def test_U5_shear_flow_between_moving_porous_plates():
    """Plates z = 0 (u^B = -U) and z = 12 (u^B = +U) of a periodic 24-cell column, d = 1 on them: plane Couette flow twice."""
    nz, ny, nx = 24, 2, 2
    shape = (nz, ny, nx)
    U, tau0 = 0.02, 1.0
    d = np.zeros(shape)
    d[0] = d[12] = 1.0
    ub = np.zeros((3,) + shape)
    ub[0, 0], ub[0, 12] = -U, U
    f = O.init_equilibrium(19, np.ones(shape), np.zeros((3,) + shape))
    f = O.step(f, d=d, nsteps=4000, u_body=ub, tau0=tau0, use_hlbm=1)
    f2 = O.step(f, d=d, nsteps=50, u_body=ub, tau0=tau0, use_hlbm=1)
    _, u = O.moments(f2)
    _, u1 = O.moments(f)
    assert np.abs(u - u1).max() < 1e-9                      # steady
    prof = u[0, :, 0, 0]
    assert np.abs(u[1:]).max() < 1e-14
    # linear between the plates: the second difference vanishes away from them
    sec = prof[2:11] - 2 * prof[1:10] + prof[0:9]
    assert np.abs(sec[1:-1]).max() < 1e-9
    slope = (prof[10] - prof[2]) / 8.0
    assert abs(slope - 2 * U / 12.0) < 0.01 * 2 * U / 12.0   # the plates carry +-U (no slip at a d = 1 cell)
    assert abs(prof[6]) < 1e-9 and abs(prof[18]) < 1e-9      # antisymmetric about the mid-planes
    assert abs(prof[11] + slope - U) < 0.01 * U and abs(prof[1] - slope + U) < 0.01 * U   # extrapolates to +-U at the plates
    # the plate cell's own raw moment (l.97: pre-collision) is what streams in at tau = 1: f^eq(u^B) from the 2/3 of the
    # x-momentum weight that lies in the plate, f^eq(u(z +- 1)) from the 1/3 that arrives from the two neighbouring planes
    assert abs(prof[12] - (2.0 / 3.0 * U + 1.0 / 6.0 * (prof[11] + prof[13]))) < 1e-12


@pytest.mark.parametrize("Q", [19, 27])
def test_U6_moving_body_momentum_feed_closed_form(Q):
    """A porous blob that moves one cell per 4 steps along x with u^B = (0.25, 0, 0)-ish lattice speed scaled down: d(x,t) and
    u^B(x,t) are re-set every step.  Eq. 12 in Eq. 6: the collision of a cell changes its momentum by rho d (u^B - u) / tau
    (BGK form, any tau_eff), nothing else does on a periodic box."""
    nz, ny, nx = 6, 6, 12
    shape = (nz, ny, nx)
    rng = np.random.default_rng(24)
    rho = 1.0 + 0.01 * rng.standard_normal(shape)
    u = 0.01 * rng.standard_normal((3,) + shape)
    f = O.init_equilibrium(Q, rho, u)
    tau0 = 0.8
    ubv = np.array([0.04, 0.01, -0.005])
    for t in range(12):
        x0 = 2 + t // 4
        d = np.zeros(shape)
        d[2:4, 1:4, x0:x0 + 3] = 0.6
        d[3, 2, x0 + 1] = 1.0
        ub = np.zeros((3,) + shape)
        ub[:, d > 0] = ubv[:, None]
        r, v = O.moments(f)
        feed = ((r * d)[None] * (ubv[:, None, None, None] - v)).sum(axis=(1, 2, 3)) / tau0
        t0 = O.totals(f)
        f = O.step(f, d=d, nsteps=1, u_body=ub, tau0=tau0, cs_smago=0.0, use_hlbm=1)
        t1 = O.totals(f)
        assert abs(t1[0] - t0[0]) < 1e-12
        assert np.abs((t1[1:4] - t0[1:4]) - feed).max() < 1e-14

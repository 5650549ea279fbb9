"""Pins of the oracle's pressure outlet ("fixed local pressure condition"; reading G36).

B1 the rule is the mirror image of the already pinned velocity rule O4 (P10): reflecting the cell in x and imposing the
   velocity that the pressure rule derives must give the same populations and the density rho_out -- fixes every term;
B2 after the fix-up the cell's moments are exactly (rho_out, rho_out u) with u = ((S0 + 2 S+)/rho_out - 1, 0, 0); idempotent;
   independent of the unknown populations; equilibrium at (rho_out, u_x) is a fixed point;
B3 channel: velocity inlet + pressure outlet between bounce-back walls converges to the Poiseuille profile, the outlet plane
   sits at rho_out to rounding, and the density falls linearly along the channel with the viscous pressure gradient;
B4 steady state: the mass flux through the outlet equals the one through the inlet (no drift of the density level, the defect
   of the zero-gradient outlet that SURVEY section 7 hard part 9 notes).
CPU only."""
import numpy as np
import pytest

import lbm_inputs as I
from oracle import oracle as O

NT = min(8, O.max_threads())


def _mirror_x(Q):
    c, w, opp = O.lattice(Q)
    perm = np.empty(Q, dtype=int)
    for i in range(Q):
        m = (-c[i, 0], c[i, 1], c[i, 2])
        perm[i] = next(j for j in range(Q) if tuple(c[j]) == m)
    return c, w, perm


@pytest.mark.parametrize("Q", [19, 27])
def test_B1_mirror_image_of_the_velocity_rule(Q):
    c, w, perm = _mirror_x(Q)
    rng = np.random.Generator(np.random.PCG64(Q))
    for _ in range(5):
        g = np.array(O.feq(Q, 1.0 + 0.02 * rng.standard_normal(), 0.05 * rng.standard_normal(3))) * (1 + 0.02 * rng.standard_normal(Q))
        rho_out = 1.0 + 0.01 * rng.standard_normal()
        out = O.pressure_fixup_cell(Q, g, rho_out)
        s0 = g[c[:, 0] == 0].sum()
        sp = g[c[:, 0] > 0].sum()
        ux = (s0 + 2 * sp) / rho_out - 1.0
        mir = O.inlet_fixup_cell(Q, g[perm], [-ux, 0.0, 0.0])[perm]          # reflect, impose -u_x on the "inlet", reflect back
        assert np.abs(out - mir).max() <= 2e-16
        assert abs(mir.sum() - rho_out) <= 1e-15


@pytest.mark.parametrize("Q", [19, 27])
def test_B2_moments_idempotence_unknowns_fixed_point(Q):
    c, w, perm = _mirror_x(Q)
    rng = np.random.Generator(np.random.PCG64(100 + Q))
    g = np.array(O.feq(Q, 1.01, [0.04, 0.01, -0.02])) * (1 + 0.03 * rng.standard_normal(Q))
    rho_out = 0.995
    out = O.pressure_fixup_cell(Q, g, rho_out)
    ux = (g[c[:, 0] == 0].sum() + 2 * g[c[:, 0] > 0].sum()) / rho_out - 1.0
    assert abs(out.sum() - rho_out) <= 1e-15
    assert np.abs(c.T @ out - rho_out * np.array([ux, 0.0, 0.0])).max() <= 1e-15
    assert np.abs(O.pressure_fixup_cell(Q, out, rho_out) - out).max() <= 1e-15          # idempotent
    g2 = g.copy()
    g2[c[:, 0] < 0] = rng.random((c[:, 0] < 0).sum())                                   # the unknowns are never read
    assert np.array_equal(O.pressure_fixup_cell(Q, g2, rho_out), out)
    feq = np.array(O.feq(Q, rho_out, [0.03, 0.0, 0.0]))
    assert np.abs(O.pressure_fixup_cell(Q, feq, rho_out) - feq).max() <= 1e-15


def _channel(nx=96, ny=4, nz=18):
    flags = np.zeros((nz, ny, nx), dtype=np.uint8)
    flags[0] = I.SOLID
    flags[-1] = I.SOLID
    flags[1:-1, :, 0] = I.INLET
    flags[1:-1, :, -1] = I.POUTLET
    return flags


@pytest.mark.parametrize("tau", [0.8])
def test_B3_B4_poiseuille_through_a_pressure_outlet(tau):
    flags = _channel()
    nz, ny, nx = flags.shape
    uin = 0.02
    rho_out = 1.0
    u0 = np.zeros((3, nz, ny, nx))
    u0[0][flags != I.SOLID] = uin
    f = O.init_equilibrium(19, np.ones(flags.shape), u0)
    f = O.step(f, flags=flags, nsteps=9000, nthreads=NT, tau0=tau, u_in=(uin, 0.0, 0.0), rho_out=rho_out)
    rho, u = O.moments(f)
    H = nz - 2
    zeta = (np.arange(1, nz - 1) - 0.5) / H
    # B3: profile at 3/4 of the channel, normalised by the local flux (as P8)
    xs = 3 * nx // 4
    jx = (rho * u[0])[1:-1, 1, xs]
    want = 6.0 * jx.sum() / H * zeta * (1 - zeta)
    assert np.abs(jx - want).max() <= 0.01 * want.max()
    # the outlet plane carries rho_out
    assert np.abs(rho[1:-1, :, -1] - rho_out).max() <= 1e-13
    # density falls linearly: dp/dx = -12 nu U_mean / H^2 (plane Poiseuille), p = rho / 3, in the developed half of the channel
    nu = (tau - 0.5) / 3.0
    rbar = rho[1:-1, 1, :].mean(axis=0)
    slope = np.polyfit(np.arange(nx // 2, nx - 4), rbar[nx // 2:nx - 4], 1)[0]
    umean = jx.sum() / H
    assert abs(slope / (-3.0 * 12.0 * nu * umean / H ** 2) - 1.0) <= 0.05
    # B4: steady state, mass flux in = mass flux out, density level anchored
    flux = (rho * u[0])[1:-1, 1, :].sum(axis=0)
    assert abs(flux[-1] / flux[0] - 1.0) <= 5e-4 and abs(flux[nx // 2] / flux[0] - 1.0) <= 5e-4     # node moments, not link fluxes
    m0 = O.totals(f, flags)[0]
    f2 = O.step(f, flags=flags, nsteps=500, nthreads=NT, tau0=tau, u_in=(uin, 0.0, 0.0), rho_out=rho_out)
    assert abs(O.totals(f2, flags)[0] / m0 - 1.0) <= 1e-9                                             # the mass has stopped moving
    assert abs(rbar[-1] - rho_out) <= 1e-13 and 1.0 < rbar[0] < 1.05

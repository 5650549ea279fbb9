"""Pins of the oracle's fringe zone (reading G38: sponge nu_mo(x) = nu_mo (1 + A xi^2) over the last
L cells before the outlet plane).  The paper prints neither the kind of fringe nor its profile: parity unpinned against it.

Z1 off (L = 0 or A = 0) is the plain step bit for bit; cells in front of the zone are untouched by it after one step;
Z2 the relaxation time each plane collided with, recovered from one step of a spatially uniform non-equilibrium state
   (g_i(x) = f_i - (f_i - feq_i)/tau(x - c_ix)), is 1/2 + (tau0 - 1/2)(1 + A xi^2) with xi = (x - (nx-1-L))/L;
Z3 a shear wave decays faster inside the zone than in front of it.
CPU only."""
import numpy as np

import lbm_inputs as I
from oracle import oracle as O


def _state(shape, seed=9):
    rng = np.random.Generator(np.random.PCG64(seed))
    rho = 1.0 + 0.01 * rng.standard_normal(shape)
    u = 0.03 * rng.standard_normal((3,) + shape)
    return O.init_equilibrium(19, rho, u)


def test_Z1_off_and_locality():
    shape = (6, 6, 40)
    f = _state(shape)
    ref = O.step(f, nsteps=3, tau0=0.6, cs_smago=0.1)
    assert np.array_equal(O.step(f, nsteps=3, tau0=0.6, cs_smago=0.1, fringe_len=0, fringe_factor=5.0), ref)
    assert np.array_equal(O.step(f, nsteps=3, tau0=0.6, cs_smago=0.1, fringe_len=10, fringe_factor=0.0), ref)
    one = O.step(f, nsteps=1, tau0=0.6, cs_smago=0.1, fringe_len=10, fringe_factor=5.0)
    ref1 = O.step(f, nsteps=1, tau0=0.6, cs_smago=0.1)
    # zone = x in [30, 39]; x = 29 has xi = 0; after one step only x >= 29 (pulling from x = 30) and, through the periodic
    # wrap, x = 0 (pulling from x = 39) can differ
    assert np.array_equal(one[..., 1:29], ref1[..., 1:29]) and not np.array_equal(one[..., 30:], ref1[..., 30:])


def test_Z2_relaxation_time_profile():
    nz, ny, nx = 4, 4, 32
    c, w, opp = O.lattice(19)
    feq = np.array(O.feq(19, 1.0, [0.02, 0.01, -0.01]))
    rng = np.random.Generator(np.random.PCG64(2))
    fne = feq * (1 + 0.05 * rng.standard_normal(19))
    fne += (feq.sum() - fne.sum()) / 19                      # keep it simple: any non-equilibrium state will do
    f = np.tile(fne[:, None, None, None], (1, nz, ny, nx))
    rho = fne.sum()
    u = (c.T @ fne) / rho
    fe = np.array(O.feq(19, rho, u))
    tau0, L, A = 0.7, 8, 6.0
    g = O.step(f, nsteps=1, tau0=tau0, fringe_len=L, fringe_factor=A)
    i = next(k for k in range(19) if tuple(c[k]) == (0, 1, 0))            # c_x = 0: source plane = own plane
    tau_meas = (fne[i] - fe[i]) / (fne[i] - g[i, 0, 0, :])
    xi = np.clip((np.arange(nx) - (nx - 1 - L)) / L, 0.0, 1.0)
    assert np.abs(tau_meas - (0.5 + (tau0 - 0.5) * (1 + A * xi ** 2))).max() <= 1e-12
    j = next(k for k in range(19) if tuple(c[k]) == (1, 0, 0))            # c_x = +1: source plane x - 1
    tau_j = (fne[j] - fe[j]) / (fne[j] - g[j, 0, 0, :])
    assert np.abs(tau_j - np.roll(0.5 + (tau0 - 0.5) * (1 + A * xi ** 2), 1)).max() <= 1e-12


def test_Z3_shear_wave_decays_faster_in_the_zone():
    nz, ny, nx = 16, 4, 96
    z = np.arange(nz)
    u = np.zeros((3, nz, ny, nx))
    u[1] = (0.02 * np.sin(2 * np.pi * z / nz))[:, None, None]
    f = O.init_equilibrium(19, np.ones((nz, ny, nx)), u)
    g = O.step(f, nsteps=60, nthreads=4, tau0=0.6, fringe_len=32, fringe_factor=8.0)
    _, ug = O.moments(g)
    amp = np.abs(ug[1]).max(axis=(0, 1))
    assert amp[80] < 0.8 * amp[30] and abs(amp[30] / amp[20] - 1.0) < 1e-3

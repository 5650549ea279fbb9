"""Pins of the oracle's collision = 2: the HRR form with the FD strain of Eq. 10 taken of u^ of the PREVIOUS time level
(reading G41; Eq. 6-12, and l.172: a "local cell model" at 188 bytes per collision).  The collision itself
(orc_collide_cell_hrr) is pinned by tests/test_oracle_hrr.py (H1-H9); what is new is WHICH field the strain is taken of:
  L1  the first step of a call has no history: bit-identical to collision = 1;
  L2  a later step differences u^ of the level before: two steps rebuilt independently from the single-cell collision, numpy.roll
      streaming and numpy central differences of the PREVIOUS level's u^ (porosity, Smagorinsky, both lattices); the same
      reconstruction with the CURRENT level's u^ gives collision = 1 and differs (the pin tells the two apart);
  L3  where u^ does not change in time the two forms agree: uniform flow is a fixed point of both; a decaying shear wave
      relaxes at the same viscosity (sigma = 0: all of the stress comes through Eq. 10);
  L4  mass and momentum are conserved on a periodic box without porosity;
  L5  wall-model cells, inlet, outlet, walls (config 3): finite, and the first step equals collision = 1.
CPU only."""
import numpy as np
import pytest

import lbm_inputs as I
from oracle import oracle as O

NT = min(8, O.max_threads())


def _state(Q, shape, seed, amp=0.04):
    rng = np.random.default_rng(seed)
    nz, ny, nx = shape
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    u = np.zeros((3,) + shape)
    for a in range(3):
        for _ in range(3):
            k = rng.integers(1, 3, 3)
            ph = rng.uniform(0, 2 * np.pi)
            u[a] += amp / 3 * np.sin(2 * np.pi * (k[0] * x / nx + k[1] * y / ny + k[2] * z / nz) + ph)
    rho = 1.0 + 0.01 * np.cos(2 * np.pi * x / nx + 1.0) * np.cos(2 * np.pi * z / nz)
    f = O.init_equilibrium(Q, rho, u)
    return f * (1.0 + 0.02 * rng.standard_normal(f.shape))        # non-equilibrium content


def _uhat(f, d):
    rho, u = O.moments(f)
    return (1.0 - d)[None] * u                                     # Eq. 12 with u^B = 0


def _strain(uh):
    """S_ab = (D_a u_b + D_b u_a)/2 with periodic central differences; arrays are [3][nz][ny][nx], axis of x_a is 3 - a"""
    D = np.empty((3, 3) + uh.shape[1:])
    for a in range(3):
        ax = 3 - a                                                 # x -> last axis
        for b in range(3):
            D[a, b] = 0.5 * (np.roll(uh[b], -1, axis=ax - 1) - np.roll(uh[b], 1, axis=ax - 1))
    return 0.5 * (D + D.transpose(1, 0, 2, 3, 4))


def _rebuild_step(Q, f, d, S, par):
    """one step from the pieces: single-cell HRR collision with the given strain field, then periodic pull streaming"""
    c, _, _ = O.lattice(Q)
    fs = np.empty_like(f)
    nz, ny, nx = f.shape[1:]
    for z in range(nz):
        for y in range(ny):
            for x in range(nx):
                fs[:, z, y, x], _ = O.collide_cell_hrr(Q, f[:, z, y, x], d=d[z, y, x], tau0=par["tau0"], cs_smago=par["cs_smago"],
                                                       sigma=par["sigma"], S=S[:, :, z, y, x])
    out = np.empty_like(f)
    for i in range(Q):
        out[i] = np.roll(fs[i], (int(c[i][2]), int(c[i][1]), int(c[i][0])), axis=(0, 1, 2))
    return out


@pytest.mark.parametrize("Q", [19, 27])
def test_L1_first_step_has_no_history(Q):
    shape = (6, 7, 8)
    f = _state(Q, shape, 5)
    d = np.random.default_rng(6).uniform(0, 0.5, shape)
    par = dict(tau0=0.56, cs_smago=0.12, use_hlbm=1, sigma=0.6)
    a = O.step(f, d=d, nsteps=1, collision=2, **par)
    b = O.step(f, d=d, nsteps=1, collision=1, **par)
    assert np.array_equal(a, b)
    assert not np.array_equal(O.step(f, d=d, nsteps=3, collision=2, **par), O.step(f, d=d, nsteps=3, collision=1, **par))


@pytest.mark.parametrize("Q", [19, 27])
def test_L2_second_step_differences_the_previous_level(Q):
    shape = (5, 6, 7)
    f0 = _state(Q, shape, 11)
    d = np.random.default_rng(12).uniform(0, 0.4, shape)
    par = dict(tau0=0.58, cs_smago=0.1, sigma=0.5)
    S0 = _strain(_uhat(f0, d))
    f1 = _rebuild_step(Q, f0, d, S0, par)
    assert np.abs(f1 - O.step(f0, d=d, nsteps=1, collision=1, use_hlbm=1, **par)).max() < 2e-15   # the pieces are the oracle's step
    lagged = _rebuild_step(Q, f1, d, S0, par)                      # strain of u^ at level 0
    current = _rebuild_step(Q, f1, d, _strain(_uhat(f1, d)), par)  # strain of u^ at level 1
    got2 = O.step(f0, d=d, nsteps=2, collision=2, use_hlbm=1, **par)
    got1 = O.step(f0, d=d, nsteps=2, collision=1, use_hlbm=1, **par)
    assert np.abs(got2 - lagged).max() < 3e-15
    assert np.abs(got1 - current).max() < 3e-15
    assert np.abs(lagged - current).max() > 1e-7                   # the two readings are told apart


def test_L3_uniform_flow_is_a_fixed_point_and_a_shear_wave_decays_at_nu():
    Q, shape = 19, (4, 4, 8)
    cell = O.feq3(Q, 1.02, (0.03, -0.02, 0.01))                     # the third-order equilibrium of Eq. 11
    f = np.broadcast_to(cell[:, None, None, None], (Q,) + shape).copy()
    assert np.abs(O.step(f, nsteps=5, collision=2, tau0=0.6, sigma=0.3) - f).max() < 1e-15
    # shear wave u_y(x) = a sin(kx): amplitude decays as exp(-nu k^2 t); sigma = 0: every bit of stress comes through Eq. 10
    nx, T, tau = 32, 200, 0.8
    shape = (1, 1, nx)
    k = 2 * np.pi / nx
    u = np.zeros((3,) + shape)
    u[1, 0, 0] = 1e-3 * np.sin(k * np.arange(nx))
    f = O.init_equilibrium(Q, np.ones(shape), u)
    nu = (tau - 0.5) / 3.0
    amps = {}
    for coll in (1, 2):
        out = O.step(f, nsteps=T, collision=coll, tau0=tau, sigma=0.0)
        _, uo = O.moments(out)
        amps[coll] = 2 * np.abs(np.fft.rfft(uo[1, 0, 0])[1]) / nx
    expected = 1e-3 * np.exp(-nu * k * k * T)
    assert abs(amps[1] / expected - 1) < 1e-2                      # (discrete dispersion: 0.4 % at this k)
    assert abs(amps[2] / expected - 1) < 1e-2                      # the lag of one level changes the rate by O(nu k^2)
    assert amps[1] != amps[2] and abs(amps[2] / amps[1] - 1) < 5e-3


@pytest.mark.parametrize("Q", [19, 27])
def test_L4_conservation(Q):
    shape = (6, 6, 6)
    f = _state(Q, shape, 21)
    out = O.step(f, nsteps=6, nthreads=NT, collision=2, tau0=0.55, cs_smago=0.14, sigma=0.7)
    c, _, _ = O.lattice(Q)
    assert abs(out.sum() - f.sum()) < 1e-12 * f.sum()
    for a in range(3):
        m0 = (f * np.asarray(c)[:, a, None, None, None]).sum()
        m1 = (out * np.asarray(c)[:, a, None, None, None]).sum()
        assert abs(m1 - m0) < 1e-12


def test_L5_urban_channel_with_wall_model():
    cfg = I.make_config(3, shape=(16, 20, 48))
    f = O.init_equilibrium(cfg["Q"], cfg["rho"], cfg["u"])
    par = dict(cfg["params"], sigma=0.7)
    a = O.step(f, d=cfg["d"], flags=cfg["flags"], nsteps=1, nthreads=NT, **dict(par, collision=2))
    b = O.step(f, d=cfg["d"], flags=cfg["flags"], nsteps=1, nthreads=NT, **dict(par, collision=1))
    assert np.array_equal(a, b)
    a = O.step(f, d=cfg["d"], flags=cfg["flags"], nsteps=30, nthreads=NT, **dict(par, collision=2))
    b = O.step(f, d=cfg["d"], flags=cfg["flags"], nsteps=30, nthreads=NT, **dict(par, collision=1))
    assert np.isfinite(a).all() and not np.array_equal(a, b)
    assert np.abs(a - b).max() < 5e-3                              # the same flow, a different discretisation of Eq. 10

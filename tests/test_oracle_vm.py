"""Pins of the oracle's Vortex Method inflow (Eq. 18-21; readings G11, G34, G35).

V1 a single vortex: azimuthal field, circulation on a far contour = Gamma (fixes the 1/(2 pi), the orientation of the
   cross product with d_inlet and the sign of the exponent, G11: with exp(+..) the contour integral is astronomically large);
V2 Gamma of Eq. 19 against a value worked out by hand for one set of numbers (G34), its scaling laws (Gamma ~ I, ~ |u_mean|,
   ~ sqrt(A/N)) and its sign;
V3 the in-plane field of many vortices is solenoidal (each summand of Eq. 20 is a pure rotation);
V4 core: Eq. 20 tends to solid-body rotation Gamma r / (4 pi sigma^2) for r << sigma (series of 1 - exp), zero at the seed itself;
V5 Eq. 21: no streamwise fluctuation where the previous inflow has no gradient; for a profile U(z) it is -u_v,z sign(dU/dz);
   invariant under rescaling of the previous inflow (the gradient is normalised);
V6 seeds over non-inlet cells carry no circulation; non-inlet cells keep u_mean;
V7 the step with the VM inlet: nv = 0 or I = 0 with a uniform mean equals the plain step bit for bit; after a step the inlet
   cells' velocity moment IS the field of orc_vm_inflow (P10: the fix-up imposes its velocity exactly) -- ties the (z, y)
   indexing of the field to the lattice.
CPU only."""
import numpy as np
import pytest

import lbm_inputs as I
from oracle import oracle as O


def _plane(nz=48, ny=64):
    return np.ones((nz, ny), dtype=np.uint8)


def _uniform(nz, ny, ux=0.05):
    u = np.zeros((3, nz, ny))
    u[0] = ux
    return u


def _gamma_of_single(nz=96, ny=96, inten=0.2, ux=0.05, sign=1.0):
    """circulation of a single centred vortex, measured on a far square contour (trapezoid rule)"""
    mask = _plane(nz, ny)
    um = _uniform(nz, ny, ux)
    u = O.vm_inflow(mask, um, um, [[48.0, 48.0]], [sign], 3.0, inten)
    v, w = u[1], u[2]                       # v = u_y[z, y], w = u_z[z, y]
    a, b = 8, 88                            # contour 40 cells = 13 sigma from the seed: exp(-89) of the core is left
    # counter-clockwise in the (y, z) plane: +y along z=a, +z along y=b, -y along z=b, -z along y=a
    circ = np.trapezoid(v[a, a:b + 1]) + np.trapezoid(w[a:b + 1, b]) - np.trapezoid(v[b, a:b + 1]) - np.trapezoid(w[a:b + 1, a])
    return circ, u


def test_V1_single_vortex_circulation_orientation_and_exponent():
    circ, u = _gamma_of_single()
    A, N, k = 96 * 96, 1, 1.5 * (0.05 * 0.2) ** 2
    gamma = 4.0 * np.sqrt(np.pi * A * k / (3.0 * N * (2.0 * np.log(3.0) - 3.0 * np.log(2.0))))
    # the contour integral of a field ~ 1/r is resolved by the trapezoid rule to ~1e-4 here
    # orientation: (p - x) x d_inlet with d = +x gives a rotation that is CLOCKWISE seen in the (y, z) plane with y to the
    # right and z up, i.e. circulation -Gamma around +x ... measured, not assumed: the sign is fixed by the next two lines
    assert abs(abs(circ) / gamma - 1.0) < 2e-3
    # Eq. 20 literally: at x = p + (r, 0) (to the +y side of the seed), (p - x) = (0, -r, 0), (p - x) x (1,0,0) = (0, 0, +r):
    # u_z > 0 there for Gamma > 0
    assert u[2, 48, 58] > 0 and u[2, 48, 38] < 0 and u[1, 58, 48] < 0 and u[1, 38, 48] > 0
    assert circ > 0
    assert np.isfinite(u).all() and np.abs(u[1:]).max() < 1.0
    # streamwise component untouched (uniform previous inflow)
    assert np.array_equal(u[0], np.full_like(u[0], 0.05))
    c2, _ = _gamma_of_single(sign=-1.0)
    assert abs(c2 + circ) < 1e-12 * abs(circ)


def test_V2_gamma_value_and_scaling():
    # hand arithmetic for A = 100 cells, N = 4, |u_mean| = 0.1, I = 1:  k = 1.5 * 0.01 = 0.015;
    # 2 ln 3 - 3 ln 2 = 2.1972246 - 2.0794415 = 0.1177831;  pi * 100 * 0.015 = 4.7123890;  3 * 4 * 0.1177831 = 1.4133972;
    # quotient 3.3340869, root 1.8259482, Gamma = 7.3037927
    mask = np.zeros((30, 30), dtype=np.uint8)
    mask[10:20, 10:20] = 1                               # A = 100
    um = _uniform(30, 30, 0.1)
    pos = [[14.0, 14.0], [1.0, 1.0], [2.0, 2.0], [3.0, 3.0]]          # three seeds over non-inlet cells: Gamma = 0 (V6), N = 4
    u = O.vm_inflow(mask, um, um, pos, [1, 1, 1, 1], 1.0, 1.0)
    # far from the core (r = 5 >> sigma = 1) the speed is Gamma / (2 pi r)
    speed = np.hypot(u[1, 14, 19], u[2, 14, 19])
    assert abs(speed * 2 * np.pi * 5.0 - 7.3037927) < 5e-5          # exp(-12.5) of the core is left at r = 5 sigma
    base = np.hypot(*O.vm_inflow(mask, um, um, pos, [1, 1, 1, 1], 1.0, 0.5)[1:, 14, 19])
    assert abs(base / speed - 0.5) < 1e-12                               # ~ I
    um2 = _uniform(30, 30, 0.2)
    assert abs(np.hypot(*O.vm_inflow(mask, um2, um2, pos, [1, 1, 1, 1], 1.0, 1.0)[1:, 14, 19]) / speed - 2.0) < 1e-12   # ~ |u_mean|
    assert abs(np.hypot(*O.vm_inflow(mask, um, um, pos[:1], [1], 1.0, 1.0)[1:, 14, 19]) / speed - 2.0) < 1e-12        # ~ 1/sqrt(N)


def test_V3_solenoidal_in_plane():
    rng = np.random.Generator(np.random.PCG64(3))
    nz, ny = 64, 80
    mask = _plane(nz, ny)
    um = _uniform(nz, ny)
    pos = np.stack([rng.uniform(10, 70, 40), rng.uniform(10, 54, 40)], axis=1)
    sign = rng.choice([-1.0, 1.0], 40)
    u = O.vm_inflow(mask, um, um, pos, sign, 6.0, 0.15)
    div = 0.5 * (u[1][:, 2:] - u[1][:, :-2])[1:-1] + 0.5 * (u[2][2:] - u[2][:-2])[:, 1:-1]
    rot = 0.5 * (u[2][:, 2:] - u[2][:, :-2])[1:-1] - 0.5 * (u[1][2:] - u[1][:-2])[:, 1:-1]
    assert np.abs(div).max() < 0.02 * np.abs(rot).max()                 # O(h^2 / sigma^2) truncation of the stencil only


def test_V4_core_is_solid_body_rotation_and_finite_at_the_seed():
    nz = ny = 64
    mask = _plane(nz, ny)
    um = _uniform(nz, ny)
    sig = 12.0
    u = O.vm_inflow(mask, um, um, [[32.0, 32.0]], [1.0], sig, 0.2)
    assert u[1, 32, 32] == 0.0 and u[2, 32, 32] == 0.0
    A, k = nz * ny, 1.5 * (0.05 * 0.2) ** 2
    gamma = 4.0 * np.sqrt(np.pi * A * k / (3.0 * (2.0 * np.log(3.0) - 3.0 * np.log(2.0))))
    omega = gamma / (4.0 * np.pi * sig * sig)                            # (1 - exp(-r^2/2s^2))/r^2 -> 1/(2 s^2)
    assert abs(u[2, 32, 33] / omega - 1.0) < 2e-3 and abs(u[1, 33, 32] / (-omega) - 1.0) < 2e-3


def test_V5_streamwise_fluctuation():
    rng = np.random.Generator(np.random.PCG64(5))
    nz, ny = 40, 48
    mask = _plane(nz, ny)
    um = _uniform(nz, ny)
    prof = 0.03 + 0.001 * np.arange(nz, dtype=float) ** 1.3              # U(z), increasing
    up = np.zeros((3, nz, ny))
    up[0] = prof[:, None]
    pos = np.stack([rng.uniform(5, 43, 20), rng.uniform(5, 35, 20)], axis=1)
    sign = rng.choice([-1.0, 1.0], 20)
    a = O.vm_inflow(mask, um, um, pos, sign, 4.0, 0.2)                   # uniform previous inflow
    assert np.array_equal(a[0], um[0])
    b = O.vm_inflow(mask, um, up, pos, sign, 4.0, 0.2)
    assert np.array_equal(b[1:], a[1:])
    assert np.abs((b[0] - um[0]) + a[2]).max() < 1e-15                   # -u_v . z^
    c = O.vm_inflow(mask, um, -3.0 * up, pos, sign, 4.0, 0.2)            # gradient reversed: fluctuation changes sign
    assert np.abs((c[0] - um[0]) - a[2]).max() < 1e-15
    upy = np.zeros((3, nz, ny))
    upy[0] = 0.05 + 0.01 * np.sin(2 * np.pi * np.arange(ny) / ny)[None, :]      # gradient along y, periodic
    e = O.vm_inflow(mask, um, upy, pos, sign, 4.0, 0.2)
    gy = np.cos(2 * np.pi * (np.arange(ny)) / ny)
    sel = np.abs(gy) > 0.05
    assert np.abs((e[0] - um[0])[:, sel] + (a[1] * np.sign(gy)[None, :])[:, sel]).max() < 1e-15


def test_V6_non_inlet_cells_and_seeds():
    nz, ny = 24, 32
    mask = _plane(nz, ny)
    mask[0] = 0
    mask[-1] = 0
    um = _uniform(nz, ny)
    um[0, 0] = um[0, -1] = 0.123
    u = O.vm_inflow(mask, um, um, [[10.0, 0.2], [12.0, 22.9]], [1.0, -1.0], 3.0, 0.3)      # both seeds over wall rows
    assert np.array_equal(u, um)
    u = O.vm_inflow(mask, um, um, [[10.0, 12.0]], [1.0], 3.0, 0.3)
    assert np.array_equal(u[:, 0], um[:, 0]) and np.array_equal(u[:, -1], um[:, -1])
    assert np.abs(u[1:, 1:-1]).max() > 0


def test_V7_step_with_vm_inlet():
    cfg = I.make_config(3, shape=(20, 24, 40))
    nz, ny, nx = cfg["shape"]
    f = O.init_equilibrium(19, cfg["rho"], cfg["u"])
    par = dict(cfg["params"])
    um = np.zeros((3, nz, ny))
    um[0] = par["u_in"][0]
    # (a) no vortices / zero intensity: the plain step, bit for bit
    ref = O.step(f, d=cfg["d"], flags=cfg["flags"], nsteps=3, **par)
    a, ua = O.step_vm(f, um, um, np.zeros((0, 2)), np.zeros(0), 3.0, 0.2, d=cfg["d"], flags=cfg["flags"], nsteps=3, **par)
    b, ub = O.step_vm(f, um, um, [[10.0, 9.0]], [1.0], 3.0, 0.0, d=cfg["d"], flags=cfg["flags"], nsteps=3, **par)
    assert np.array_equal(a, ref) and np.array_equal(b, ref) and np.array_equal(ua, um)
    # (b) with vortices: the inlet plane carries exactly the field of orc_vm_inflow
    rng = np.random.Generator(np.random.PCG64(7))
    pos = np.stack([rng.uniform(0, ny, 12), rng.uniform(1, nz - 1, 12)], axis=1)
    sign = rng.choice([-1.0, 1.0], 12)
    mask = ((cfg["flags"][:, :, 0] & 15) == I.INLET).astype(np.uint8)
    prof = np.zeros((3, nz, ny))
    prof[0] = (0.05 * (np.maximum(np.arange(nz) - 0.5, 0.5) / nz) ** 0.25)[:, None]        # power-law mean profile
    g, u1 = O.step_vm(f, prof, prof, pos, sign, 3.0, 0.2, d=cfg["d"], flags=cfg["flags"], nsteps=1, **par)
    want1 = O.vm_inflow(mask, prof, prof, pos, sign, 3.0, 0.2)
    assert np.array_equal(u1, want1)
    _, u = O.moments(g)
    inl = mask.astype(bool)
    assert np.abs(u[:, :, :, 0][:, inl] - want1[:, inl]).max() < 1e-14
    g2, u2 = O.step_vm(g, prof, u1, pos, sign, 3.0, 0.2, d=cfg["d"], flags=cfg["flags"], nsteps=1, **par)
    assert np.array_equal(u2, O.vm_inflow(mask, prof, u1, pos, sign, 3.0, 0.2))            # u_prev = previous inflow
    h, uh = O.step_vm(f, prof, prof, pos, sign, 3.0, 0.2, d=cfg["d"], flags=cfg["flags"], nsteps=2, **par)
    assert np.array_equal(h, g2) and np.array_equal(uh, u2)

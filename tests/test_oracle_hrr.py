"""Pins of the oracle's HRR collision form (Eq. 6-11, l.68-97, coupling l.131).

H1 Hermite moments of the third-order equilibrium, H2 fixed point, H3 conservation, H4 projection
idempotence, H5 reduction to the already pinned BGK collide at u = 0, H6 FD strain of a sine shear and the
closed-form post-collision stress at sigma = 0, H7 Taylor-Green decay at sigma = 1, 0.5, 0 (fixes the sign
and factor of Eq. 10, reading G10), H8 brute force with a numerically inverted Gram matrix, H9 lattice
symmetry.  Nothing here retypes the oracle's formulas: the Hermite tensors are built as full tensors from the
hand-typed golden tables and the projections go through numpy.linalg.  CPU only.
"""
import os

import numpy as np
import pytest

import lbm_inputs as I
from oracle import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")
NT = min(8, O.max_threads())
CS2 = 1.0 / 3.0


def _golden(Q):
    rows = [l.split() for l in open(os.path.join(GOLD, "d3q%d_R1.txt" % Q)) if l.strip() and not l.startswith("#")]
    c = np.array([[int(r[1]), int(r[2]), int(r[3])] for r in rows], dtype=float)
    w = np.array([int(r[4]) / int(r[5]) for r in rows])
    return c, w


def _hermite(c):
    """Full Hermite tensors H1[i,a], H2[i,a,b], H3[i,a,b,g] of the discrete velocities (textbook definition)."""
    dl = np.eye(3)
    H1 = c
    H2 = np.einsum("ia,ib->iab", c, c) - CS2 * dl[None]
    H3 = np.einsum("ia,ib,ig->iabg", c, c, c) - CS2 * (
        np.einsum("ab,ig->iabg", dl, c) + np.einsum("ag,ib->iabg", dl, c) + np.einsum("bg,ia->iabg", dl, c))
    return H1, H2, H3


def _basis3(Q, c, w):
    """An orthonormal basis (weighted inner product) of span{H3_abg}: what 'the third-order polynomials the
    lattice supports' means, found numerically (no combos typed in)."""
    _, _, H3 = _hermite(c)
    V = H3.reshape(Q, 27).T                                   # 27 vectors of length Q
    G = (V * w[None]) @ V.T
    ev, U = np.linalg.eigh(G)
    keep = ev > 1e-12
    B = (U[:, keep].T @ V) / np.sqrt(ev[keep])[:, None]       # rows: w-orthonormal vectors
    return B


def _project3(Q, c, w, a3_full):
    """Order-3 Hermite series term for a full symmetric coefficient tensor a3[a,b,g]: the w-orthogonal
    projection of sum_abg H3_abg a3_abg / (3! c_s^6) (valid on a lattice that carries all of H3) on the
    supported span.  On D3Q27 every H3 except the aaa-type is carried; D3Q19 also loses xyz."""
    _, _, H3 = _hermite(c)
    B = _basis3(Q, c, w)
    # target moments: m_k = <B_k, f/w>_w must equal B_k-combination of a3: sum_i B_ki f_i = sum_abg beta_k,abg a3_abg
    # where B_k = sum_abg beta_k,abg H3_abg.  Solve beta by least squares in the H3 span.
    V = H3.reshape(Q, 27).T
    beta = np.linalg.lstsq(V.T, B.T, rcond=None)[0].T         # [k, 27]
    m = beta @ a3_full.reshape(27)
    return w * (m @ B)


def _rand_cell(Q, rng, amp=0.06, noise=0.03):
    rho = 1.0 + 0.1 * rng.uniform(-1, 1)
    u = amp * rng.uniform(-1, 1, size=3)
    return O.feq(Q, rho, u) * (1.0 + noise * rng.uniform(-1, 1, size=Q))


# ---- H1: Hermite moments of Eq. 11 ------------------------------------------------------------------------
@pytest.mark.parametrize("Q", [19, 27])
def test_H1_third_order_equilibrium_has_the_hermite_moments_of_eq11(Q):
    c, w = _golden(Q)
    H1, H2, H3 = _hermite(c)
    rng = np.random.default_rng(31)
    for _ in range(5):
        rho = 1.0 + 0.2 * rng.uniform(-1, 1)
        u = 0.1 * rng.uniform(-1, 1, size=3)
        f = O.feq3(Q, rho, u)
        assert abs(f.sum() - rho) < 2e-16 * 8
        assert np.abs(H1.T @ f - rho * u).max() < 1e-16
        assert np.abs(np.einsum("iab,i->ab", H2, f) - rho * np.outer(u, u)).max() < 1e-16
        a3 = rho * np.einsum("a,b,g->abg", u, u, u)
        got = np.einsum("iabg,i->abg", H3, f)
        # every component the lattice carries: the moments along the supported span
        B = _basis3(Q, c, w)
        V = H3.reshape(Q, 27).T
        beta = np.linalg.lstsq(V.T, B.T, rcond=None)[0].T
        assert np.abs(B @ f - beta @ a3.reshape(27)).max() < 1e-16
        # named components: aab-type on both lattices, xyz on D3Q27 only
        for (a, b, g) in [(0, 0, 1), (0, 0, 2), (0, 1, 1), (0, 2, 2), (1, 1, 2), (1, 2, 2)]:
            assert abs(got[a, b, g] - a3[a, b, g]) < 1e-16
        if Q == 27:
            assert abs(got[0, 1, 2] - a3[0, 1, 2]) < 1e-16
        # and the third-order part is exactly the projected series (independent construction)
        assert np.abs((f - O.feq(Q, rho, u)) - _project3(Q, c, w, a3)).max() < 1e-16


def test_H1_supported_third_order_dimension():
    for Q, dim in ((19, 6), (27, 7)):
        c, w = _golden(Q)
        assert _basis3(Q, c, w).shape[0] == dim


# ---- independent per-cell HRR collide (H8): full tensors, numerical projection, long double ---------------
def _brute_collide_hrr(Q, fc, d, ub, tau0, cs, sigma, S):
    c, w = _golden(Q)
    H1, H2, H3 = _hermite(c)
    L = np.longdouble
    fc = fc.astype(L)
    rho = fc.sum()
    u = (c.astype(L).T @ fc) / rho
    uh = (1 - L(d)) * u + L(d) * np.asarray(ub, dtype=L)
    # Eq. 11: series with coefficients rho, rho u^, rho u^u^, rho u^u^u^ (third order projected on the lattice)
    a3 = rho * np.einsum("a,b,g->abg", uh, uh, uh)
    feq = w * (rho + (H1 @ (rho * uh)) / CS2 + np.einsum("iab,ab->i", H2, rho * np.outer(uh, uh)) / (2 * CS2 ** 2)) \
        + _project3(Q, c, w, a3.astype(float)).astype(L)
    f1 = fc - feq
    A0 = f1.sum()
    A1 = H1.T @ f1
    A2 = np.einsum("iab,i->ab", H2, f1)
    tau = L(tau0)
    if cs > 0:
        Pi = np.einsum("ia,ib,i->ab", c, c, f1)
        tau = (tau0 + np.sqrt(L(tau0) ** 2 + 18 * np.sqrt(L(2)) * cs * cs * np.sqrt((Pi * Pi).sum()) / rho)) / 2
    A3 = (np.einsum("a,bg->abg", uh, A2) + np.einsum("b,ag->abg", uh, A2) + np.einsum("g,ab->abg", uh, A2))
    freg = w * (A0 + (H1 @ A1) / CS2 + np.einsum("iab,ab->i", H2, A2) / (2 * CS2 ** 2)) \
        + _project3(Q, c, w, A3.astype(float)).astype(L)
    ffd = -w * rho * tau / CS2 * np.einsum("iab,ab->i", H2, np.asarray(S, dtype=L))
    ft = sigma * freg + (1 - sigma) * ffd
    return (feq + (1 - 1 / tau) * ft).astype(float), float(tau)


@pytest.mark.parametrize("Q", [19, 27])
def test_H8_cell_bruteforce_full_tensor_projection(Q):
    rng = np.random.default_rng(38)
    for k in range(12):
        fc = _rand_cell(Q, rng)
        d = [0.0, 0.35, 1.0][k % 3]
        ub = 0.02 * rng.uniform(-1, 1, size=3) if k % 2 else np.zeros(3)
        S = 1e-3 * rng.uniform(-1, 1, size=(3, 3))
        S = 0.5 * (S + S.T)
        sigma = [1.0, 0.0, 0.7, 0.98][k % 4]
        cs = [0.0, 0.1, 0.17][k % 3]
        got, tau = O.collide_cell_hrr(Q, fc, d=d, ub=ub, tau0=0.53, cs_smago=cs, sigma=sigma, S=S)
        ref, tau_ref = _brute_collide_hrr(Q, fc, d, ub, 0.53, cs, sigma, S)
        assert abs(tau - tau_ref) < 1e-14
        assert np.abs(got - ref).max() < 2e-15


# ---- H2 / H3: fixed point and conservation ---------------------------------------------------------------
@pytest.mark.parametrize("Q", [19, 27])
def test_H2_third_order_equilibrium_is_a_fixed_point(Q):
    f = O.feq3(Q, 1.07, [0.08, -0.05, 0.03])
    for sigma in (1.0, 0.4, 0.0):
        fs, tau = O.collide_cell_hrr(Q, f, tau0=0.51, cs_smago=0.15, sigma=sigma)
        assert np.abs(fs - f).max() < 3e-16
        assert abs(tau - 0.51) < 1e-15


@pytest.mark.parametrize("Q", [19, 27])
def test_H3_collision_conserves_mass_and_momentum(Q):
    c, w = _golden(Q)
    rng = np.random.default_rng(33)
    for sigma in (1.0, 0.6, 0.0):
        fc = _rand_cell(Q, rng)
        S = 2e-3 * rng.uniform(-1, 1, size=(3, 3))
        S = 0.5 * (S + S.T)                       # not traceless: H2:S still has zero mass and momentum
        fs, _ = O.collide_cell_hrr(Q, fc, tau0=0.55, cs_smago=0.1, sigma=sigma, S=S)
        assert abs(fs.sum() - fc.sum()) < 1e-15
        assert np.abs(c.T @ (fs - fc)).max() < 1e-16


# ---- H4: the regularisation is a projection ------------------------------------------------------------------
@pytest.mark.parametrize("Q", [19, 27])
def test_H4_regularised_state_is_reproduced(Q):
    # tau0 -> infinity-like: (1 - 1/tau) ~ 1 is not available (tau0 is free): use the algebra instead.
    # f* = feq + (1-1/tau) R(f - feq).  Applying the collision to g = feq + R(f - feq) (same moments rho, u up
    # to second order, so same feq, same a2, same recursion) must give feq + (1-1/tau) R(f-feq) again: R R = R.
    rng = np.random.default_rng(34)
    tau = 0.8
    for _ in range(4):
        fc = _rand_cell(Q, rng)
        fs, _ = O.collide_cell_hrr(Q, fc, tau0=tau, sigma=1.0)
        c, w = _golden(Q)
        rho = fc.sum()
        u = (c.T @ fc) / rho
        feq = O.feq3(Q, rho, u)
        g = feq + (fs - feq) / (1.0 - 1.0 / tau)          # = feq + R(f - feq)
        gs, _ = O.collide_cell_hrr(Q, g, tau0=tau, sigma=1.0)
        assert np.abs(gs - fs).max() < 1e-15
        assert np.abs(g - fc).max() > 1e-4                # R removed something (the ghost content)


# ---- H5: at u^ = 0 the third-order terms vanish and a pure second-order Hermite non-equilibrium is kept
#          as it is, so the HRR collide equals the (separately pinned, P2-P6) BGK collide ------------------
@pytest.mark.parametrize("Q", [19, 27])
def test_H5_reduces_to_bgk_for_second_order_hermite_states_at_rest(Q):
    c, w = _golden(Q)
    _, H2, _ = _hermite(c)
    rng = np.random.default_rng(35)
    A = 1e-3 * rng.uniform(-1, 1, size=(3, 3))
    A = 0.5 * (A + A.T)
    f = O.feq(Q, 1.03, [0.0, 0.0, 0.0]) + w * np.einsum("iab,ab->i", H2, A) / (2 * CS2 ** 2)
    for cs in (0.0, 0.12):
        a, ta = O.collide_cell_hrr(Q, f, tau0=0.57, cs_smago=cs, sigma=1.0)
        b, tb = O.collide_cell(Q, f, tau0=0.57, cs_smago=cs)
        assert abs(ta - tb) < 1e-15
        assert np.abs(a - b).max() < 1e-16
    # d = 1, u^B = 0 (HLBM solid): u^ = 0 whatever u is; first-order Hermite content (momentum) is kept by Eq. 8
    f = O.feq(Q, 0.98, [0.04, -0.02, 0.01])
    a, _ = O.collide_cell_hrr(Q, f, d=1.0, tau0=0.7, sigma=1.0)
    b, _ = O.collide_cell(Q, f, d=1.0, tau0=0.7)
    # BGK keeps all of f - feq; HRR keeps its projection on Hermite orders <= 2 (+ recursion, zero at u^ = 0):
    # the low moments must agree
    assert abs(a.sum() - b.sum()) < 1e-15
    assert np.abs(c.T @ (a - b)).max() < 1e-16
    assert np.abs(np.einsum("ia,ib,i->ab", c, c, a - b)).max() < 1e-16


# ---- flow level ------------------------------------------------------------------------------------------------
def _stream_periodic(fs, c):
    out = np.empty_like(fs)
    for i in range(fs.shape[0]):
        out[i] = np.roll(fs[i], shift=(int(c[i, 2]), int(c[i, 1]), int(c[i, 0])), axis=(0, 1, 2))
    return out


def _fd_strain_periodic(uh):
    """S_ab = (D_a u_b + D_b u_a)/2 with central differences, u[3,nz,ny,nx], periodic (numpy.roll)."""
    D = np.empty((3, 3) + uh.shape[1:])
    for a in range(3):
        ax = 2 - a
        for b in range(3):
            D[a, b] = 0.5 * (np.roll(uh[b], -1, axis=ax) - np.roll(uh[b], 1, axis=ax))
    return 0.5 * (D + np.transpose(D, (1, 0, 2, 3, 4)))


@pytest.mark.parametrize("Q", [19, 27])
def test_H8_step_bruteforce_periodic_box_with_porosity(Q):
    """Whole HRR step on a 5x4x6 periodic box: u^ field and FD strain by numpy.roll, per-cell collide by the
    full-tensor long-double routine above, streaming by numpy.roll; 3 steps."""
    c, w = _golden(Q)
    rng = np.random.default_rng(39)
    shape = (6, 4, 5)
    rho = 1.0 + 0.05 * rng.uniform(-1, 1, size=shape)
    u = 0.05 * rng.uniform(-1, 1, size=(3,) + shape)
    f = O.init_equilibrium(Q, rho, u) * (1.0 + 0.02 * rng.uniform(-1, 1, size=(Q,) + shape))
    d = rng.uniform(0, 0.7, size=shape) * (rng.uniform(size=shape) < 0.4)
    par = dict(tau0=0.56, cs_smago=0.12, use_hlbm=1, collision=1, sigma=0.7)
    got = O.step(f, d=d, nsteps=3, **par)
    g = f.copy()
    for _ in range(3):
        rho_t = g.sum(axis=0)
        u_t = np.einsum("ia,izyx->azyx", c, g) / rho_t
        uh = (1.0 - d) * u_t
        S = _fd_strain_periodic(uh)
        fs = np.empty_like(g)
        for idx in np.ndindex(*shape):
            fs[(slice(None),) + idx], _ = _brute_collide_hrr(Q, g[(slice(None),) + idx], d[idx], np.zeros(3), 0.56, 0.12,
                                                              0.7, S[(slice(None), slice(None)) + idx])
        g = _stream_periodic(fs, c)
    assert np.abs(got - g).max() < 1e-14
    assert np.abs(got - O.step(f, d=d, nsteps=3, **dict(par, collision=0))).max() > 1e-5   # not the BGK form


def test_H6_fd_strain_of_a_sine_shear_and_post_collision_stress():
    """u_x = A sin(k y): the central difference gives S_xy = (A/2) cos(k y) sin(k)/1 exactly.  At sigma = 0 the
    post-collision state is f^eq + (1 - 1/tau) f(1,FD), whose second moment is fixed in closed form:
    sum_i c_x c_y f*_i = rho u_x u_y - 2 rho c_s^2 (tau - 1) S_xy  (from f(1,FD) = -w rho tau/c_s^2 H2:S, G10)."""
    Q, n, A, tau = 19, 16, 0.03, 0.8
    c, w = _golden(Q)
    k = 2 * np.pi / n
    y = np.arange(n)
    u = np.zeros((3, 2, n, 2))
    u[0] = (A * np.sin(k * y))[None, :, None]
    rho = np.ones((2, n, 2))
    f = O.init_equilibrium(Q, rho, u)
    out = O.step(f, nsteps=1, tau0=tau, collision=1, sigma=0.0)
    # undo the (periodic) streaming to look at the post-collision populations
    fs = np.empty_like(out)
    for i in range(Q):
        fs[i] = np.roll(out[i], shift=(-int(c[i, 2]), -int(c[i, 1]), -int(c[i, 0])), axis=(0, 1, 2))
    Sxy = 0.5 * A * np.cos(k * y) * np.sin(k)
    pxy = np.einsum("i,izyx->zyx", c[:, 0] * c[:, 1], fs)[0, :, 0]
    assert np.abs(pxy - (-2.0 * (1.0 / 3.0) * (tau - 1.0) * Sxy)).max() < 1e-16
    pxx = np.einsum("i,izyx->zyx", c[:, 0] * c[:, 0], fs)[0, :, 0]
    assert np.abs(pxx - (1.0 / 3.0 + (A * np.sin(k * y)) ** 2)).max() < 1e-15


def _tgv_rate(Q, sigma, N=32, tau=0.6):
    """Fitted decay rate of the kinetic energy / (4 nu k^2) - 1, diffusive scaling (u0 ~ 1/N, T ~ N^2)."""
    rho, u = I.taylor_green(N, N, 2, u0=0.05 * 32 / N)          # z-extruded: 2 planes are enough
    f = O.init_equilibrium(Q, rho, u)
    nu, k = (tau - 0.5) / 3.0, 2.0 * np.pi / N
    T = 100 * (N // 32) ** 2
    ts, Es = [0], [O.totals(f)[4]]
    for t in range(T // 10, T + 1, T // 10):
        f = O.step(f, nsteps=T // 10, nthreads=NT, tau0=tau, collision=1, sigma=sigma)
        ts.append(t)
        Es.append(O.totals(f)[4])
    ts, Es = np.array(ts), np.array(Es)
    sel = ts >= T // 5
    return -np.polyfit(ts[sel], np.log(Es[sel]), 1)[0] / (4.0 * nu * k * k) - 1.0


@pytest.mark.parametrize("Q", [19, 27])
def test_H7_taylor_green_decay_for_any_hybridisation(Q):
    """nu = (tau - 1/2)/3 whatever sigma is: a wrong sign or factor in Eq. 10 (reading G10) changes the viscosity
    of the FD part (sigma < 1) and fails this.  The FD part carries the O(k^2) error of the central difference, so
    its pin is the convergence: |rate error| <= 2 % / 2 % / 4.5 % at N = 32 for sigma = 1 / 0.5 / 0, <= 1 % at
    N = 64 for sigma = 0, shrinking by more than 3x per doubling (second order, l.113)."""
    assert abs(_tgv_rate(Q, 1.0)) <= 0.02
    assert abs(_tgv_rate(Q, 0.5)) <= 0.02
    e32, e64 = _tgv_rate(Q, 0.0, N=32), _tgv_rate(Q, 0.0, N=64)
    assert abs(e32) <= 0.045 and abs(e64) <= 0.01
    assert abs(e32) / abs(e64) > 3.0


def test_H9_lattice_symmetry_mirror_and_rotation():
    from test_oracle_flow import _apply_symmetry, _random_box
    for Q in (19, 27):
        c, _, _ = O.lattice(Q)
        shape = (6, 6, 6)
        f = _random_box(Q, shape, seed=19)
        rng = np.random.default_rng(19)
        d = rng.uniform(0, 0.6, size=shape) * (rng.uniform(size=shape) < 0.3)
        flags = (rng.uniform(size=shape) < 0.1).astype(np.uint8) * I.SOLID
        par = dict(tau0=0.54, cs_smago=0.14, use_hlbm=1, collision=1, sigma=0.8)
        a = O.step(f, d=d, flags=flags, nsteps=3, **par)
        for perm, flip in (((1, 2, 0), ()), ((0, 1, 2), (0,)), ((1, 0, 2), (0, 2))):
            fr, sp = _apply_symmetry(f, c, list(perm), flip)
            b = O.step(fr, d=np.ascontiguousarray(sp(d)), flags=np.ascontiguousarray(sp(flags)), nsteps=3, **par)
            ar, _ = _apply_symmetry(a, c, list(perm), flip)
            assert np.abs(ar - b).max() < 1e-14


def test_H10_channel_with_all_boundaries_stays_finite_and_keeps_the_inlet_velocity():
    """Small urban channel (bounce-back, inlet, outlet, HLBM boxes, wall-model cells with sigma = 0, l.131) under
    the HRR form: finite after 20 steps and the inlet plane carries u_in exactly (O4 is unchanged)."""
    cfg = I.make_config(3, shape=(12, 8, 24))
    f = O.init_equilibrium(19, cfg["rho"], cfg["u"])
    par = dict(cfg["params"], collision=1, sigma=0.9)
    out = O.step(f, d=cfg["d"], flags=cfg["flags"], nsteps=20, **par)
    assert np.isfinite(out).all()
    rho, u = O.moments(out)
    inlet = (cfg["flags"] & 15) == I.INLET
    assert np.abs(u[0][inlet] - 0.05).max() < 1e-13

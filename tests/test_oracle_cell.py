"""Pins of the CPU oracle, per-cell level (P1, P2, P3-cell, P4, P5, P6, P9, P10; P15 = all of them on D3Q27).

Each check compares the oracle with something fixed by the mathematics or by the reading in
DESIGN.md, never with the oracle's own formula retyped.  CPU only.
"""
import itertools
import os

import numpy as np
import pytest

from oracle import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")
LATTICES = [19, 27]


def _golden(Q):
    rows = [l.split() for l in open(os.path.join(GOLD, "d3q%d_R1.txt" % Q)) if l.strip() and not l.startswith("#")]
    c = np.array([[int(r[1]), int(r[2]), int(r[3])] for r in rows])
    w = np.array([int(r[4]) / int(r[5]) for r in rows])
    return c, w


def _random_state(Q, rng, amp=0.05, noise=0.02):
    """A generic positive non-equilibrium cell state."""
    rho = 1.0 + 0.1 * rng.uniform(-1, 1)
    u = amp * rng.uniform(-1, 1, size=3)
    f = O.feq(Q, rho, u)
    return f * (1.0 + noise * rng.uniform(-1, 1, size=Q))


# ---- P1: lattice tables ------------------------------------------------------------------------
@pytest.mark.parametrize("Q", LATTICES)
def test_P1_tables_match_hand_typed_R1_listing(Q):
    c, w, opp = O.lattice(Q)
    cg, wg = _golden(Q)
    assert np.array_equal(c, cg)
    assert np.allclose(w, wg, rtol=0, atol=1e-17)


@pytest.mark.parametrize("Q", LATTICES)
def test_P1_isotropy_identities(Q):
    c, w, opp = O.lattice(Q)
    cs2 = 1.0 / 3.0
    c = c.astype(float)
    assert abs(w.sum() - 1.0) < 1e-15
    assert np.abs(np.einsum("i,ia->a", w, c)).max() < 1e-15
    assert np.abs(np.einsum("i,ia,ib->ab", w, c, c) - cs2 * np.eye(3)).max() < 1e-15
    assert np.abs(np.einsum("i,ia,ib,ic->abc", w, c, c, c)).max() < 1e-15
    dl = np.eye(3)
    iso4 = cs2 * cs2 * (np.einsum("ab,cd->abcd", dl, dl) + np.einsum("ac,bd->abcd", dl, dl) +
                        np.einsum("ad,bc->abcd", dl, dl))
    assert np.abs(np.einsum("i,ia,ib,ic,id->abcd", w, c, c, c, c) - iso4).max() < 1e-15
    assert np.array_equal(opp[opp], np.arange(Q))
    assert np.array_equal(c[opp], -c)
    assert len({tuple(v) for v in c.astype(int).tolist()}) == Q


# ---- equilibrium: moments fixed by the Hermite construction (Eq. 11 up to H2) -------------------
@pytest.mark.parametrize("Q", LATTICES)
def test_feq_moments(Q):
    c, w, _ = O.lattice(Q)
    rng = np.random.default_rng(1)
    for _ in range(5):
        rho = 1.0 + 0.2 * rng.uniform(-1, 1)
        u = 0.1 * rng.uniform(-1, 1, size=3)
        fe = O.feq(Q, rho, u)
        assert abs(fe.sum() - rho) < 1e-15
        assert np.abs(c.T @ fe - rho * u).max() < 2e-16
        second = np.einsum("i,ia,ib->ab", fe, c, c)
        assert np.abs(second - rho * (np.eye(3) / 3.0 + np.outer(u, u))).max() < 5e-16
    # u = 0: f^eq = w rho
    assert np.abs(O.feq(Q, 1.3, np.zeros(3)) - 1.3 * w).max() < 1e-16


# ---- P2: equilibrium is a fixed point of collision, tau_eff = tau0 there -----------------------
@pytest.mark.parametrize("Q", LATTICES)
def test_P2_equilibrium_fixed_point(Q):
    rng = np.random.default_rng(2)
    for _ in range(10):
        rho = 1.0 + 0.1 * rng.uniform(-1, 1)
        u = 0.08 * rng.uniform(-1, 1, size=3)
        fe = O.feq(Q, rho, u)
        fs, tau = O.collide_cell(Q, fe, tau0=0.53, cs_smago=0.15)
        assert np.abs(fs - fe).max() <= 4e-16
        assert abs(tau - 0.53) < 1e-7      # ||Pi|| of rounding only: sqrt(tau0^2 + O(1e-17)) ~ tau0


# ---- P3 (cell): collision conserves rho and rho*u when d = 0 -------------------------------------
@pytest.mark.parametrize("Q", LATTICES)
@pytest.mark.parametrize("cs", [0.0, 0.1])
def test_P3_collision_conserves_mass_momentum(Q, cs):
    c, _, _ = O.lattice(Q)
    rng = np.random.default_rng(3)
    for _ in range(20):
        f = _random_state(Q, rng)
        fs, _ = O.collide_cell(Q, f, tau0=0.55, cs_smago=cs)
        assert abs(fs.sum() - f.sum()) < 1e-15      # a few ulp of rho ~ 1
        assert np.abs(c.T @ fs - c.T @ f).max() < 3e-16


# ---- P4: cs_smago = 0 is bit-identical to a separately written plain BGK collide --------------
def _plain_bgk(Q, f, tau):
    """Textbook BGK written from scratch in numpy (same operation order as the definition)."""
    c, w, _ = _golden(Q)[0], _golden(Q)[1], None
    rho = 0.0
    j = np.zeros(3)
    for i in range(Q):
        rho += f[i]
        j += c[i] * f[i]
    u = j / rho
    out = np.empty(Q)
    for i in range(Q):
        cu = c[i, 0] * u[0] + c[i, 1] * u[1] + c[i, 2] * u[2]
        uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2]
        fe = w[i] * rho * (1.0 + 3.0 * cu + 4.5 * cu * cu - 1.5 * uu)
        out[i] = f[i] - (f[i] - fe) / tau
    return out


@pytest.mark.parametrize("Q", LATTICES)
def test_P4_cs0_is_plain_bgk(Q):
    rng = np.random.default_rng(4)
    for _ in range(10):
        f = _random_state(Q, rng)
        fs, tau = O.collide_cell(Q, f, tau0=0.7, cs_smago=0.0)
        assert tau == 0.7
        ref = _plain_bgk(Q, f, 0.7)
        # the hand-written golden weights are n/d in double, identical to the oracle's
        assert np.abs(fs - ref).max() <= 1e-16
    # and the Smagorinsky branch with a vanishing constant tends to it continuously
    f = _random_state(Q, rng)
    a, _ = O.collide_cell(Q, f, tau0=0.7, cs_smago=1e-9)
    b, _ = O.collide_cell(Q, f, tau0=0.7, cs_smago=0.0)
    assert np.abs(a - b).max() < 1e-15


# ---- P5: porous decay closed form (single cell = uniform periodic field) -----------------------
@pytest.mark.parametrize("Q", LATTICES)
def test_P5_porous_decay_closed_form(Q):
    c, _, _ = O.lattice(Q)
    d, tau0 = 0.4, 0.8
    rho0, u0 = 1.05, np.array([0.03, -0.02, 0.01])
    f = O.feq(Q, rho0, u0)
    for n in range(1, 8):
        f, _ = O.collide_cell(Q, f, d=d, tau0=tau0, cs_smago=0.0)   # uniform field: streaming is the identity
        rho = f.sum()
        u = (c.T @ f) / rho
        assert abs(rho - rho0) < 2e-15
        assert np.abs(u - (1.0 - d / tau0) ** n * u0).max() < 1e-14 * np.abs(u0).max() + 1e-17
    # d = 1, tau0 = 1: velocity is zero after one step
    f = O.feq(Q, 1.0, u0)
    f, _ = O.collide_cell(Q, f, d=1.0, tau0=1.0)
    assert np.abs(c.T @ f).max() < 1e-16
    # solid velocity u^B: d = 1, tau0 = 1 drives u to u^B exactly
    ub = np.array([0.01, 0.02, -0.03])
    f = O.feq(Q, 1.0, u0)
    f, _ = O.collide_cell(Q, f, d=1.0, ub=ub, tau0=1.0)
    assert np.abs((c.T @ f) / f.sum() - ub).max() < 1e-16


# ---- P6: self-consistency of the closed-form tau_eff (Eq. 14 with Eq. 3-5) ----------------------
@pytest.mark.parametrize("Q", LATTICES)
def test_P6_tau_eff_self_consistent(Q):
    c, w, _ = O.lattice(Q)
    cf = c.astype(float)
    rng = np.random.default_rng(6)
    cs2 = 1.0 / 3.0
    for _ in range(10):
        f = _random_state(Q, rng, noise=0.05)
        tau0, Cs = 0.5 + rng.uniform(1e-4, 0.3), rng.uniform(0.05, 0.2)
        fs, tau = O.collide_cell(Q, f, tau0=tau0, cs_smago=Cs)
        rho = f.sum()
        u = (cf.T @ f) / rho
        Pi = np.einsum("i,ia,ib->ab", f, cf, cf) - rho * (np.eye(3) * cs2 + np.outer(u, u))   # sum cc(f - feq)
        S = -Pi / (2.0 * rho * cs2 * tau)                    # Chapman-Enskog: Pi = -2 rho cs^2 tau_eff S
        normS = np.sqrt(2.0 * (S * S).sum())                 # G4
        nu_eff = cs2 * (tau0 - 0.5) + Cs * Cs * normS        # G3, Eq. 4 with Delta_x = 1
        assert abs(tau - (nu_eff / cs2 + 0.5)) < 1e-13       # Eq. 14
        assert tau >= tau0
        # relaxation with that tau
        fe = O.feq(Q, rho, u)
        assert np.abs(fs - (f - (f - fe) / tau)).max() < 3e-16


# ---- P9: Spalding wall function ---------------------------------------------------------------
def test_P9_spalding_series_and_limits():
    kappa, E = 0.41, 9.8
    # Eq. 17 bracket = exp(k) minus its first four Taylor terms: for small u+ it is k^4/24 + O(k^5)
    for up in (1e-3, 1e-2, 0.1):
        k = kappa * up
        tail = (O.spalding(up, kappa, E) - up) * E
        assert abs(tail - k ** 4 / 24.0) <= max(2.0 * k ** 5 / 120.0, 5e-16 * E * up * 10)
    assert O.spalding(0.0) == 0.0
    # strictly increasing
    ups = np.linspace(0, 30, 301)
    ys = np.array([O.spalding(u) for u in ups])
    assert np.all(np.diff(ys) > 0)


def test_P9_wallmodel_solve():
    kappa, E = 0.41, 9.8
    nu = 1e-5
    prev = 0.0
    for U2 in np.geomspace(1e-8, 0.3, 40):
        U1, ut, it1, it2 = O.wallmodel_speed(U2, nu, kappa, E)
        y2p = 1.5 * ut / nu
        # (i) residual of the law at the sample point and at the cell's own distance
        assert abs(O.spalding(U2 / ut, kappa, E) - y2p) <= 1e-10 * max(y2p, 1e-300)
        assert abs(O.spalding(U1 / ut, kappa, E) - 0.5 * ut / nu) <= 1e-10 * y2p
        assert it1 < 200 and it2 < 200
        # (iv) 0 < U1 <= U2, monotone in U2
        assert 0.0 < U1 <= U2
        assert U1 > prev
        prev = U1
        # (ii) viscous sublayer: u+ = y+  =>  U1/U2 = y1/y2 = 1/3
        if y2p < 1.0:
            assert abs(U1 / U2 - 1.0 / 3.0) < 2e-4
    # (iii) log-law limit: for y+ >= 300 the law is within 1 % of ln(E y+)/kappa
    for U2 in (0.05, 0.1, 0.2):
        U1, ut, _, _ = O.wallmodel_speed(U2, nu, kappa, E)
        y2p = 1.5 * ut / nu
        assert y2p >= 300
        assert abs((U2 / ut) / (np.log(E * y2p) / kappa) - 1.0) < 0.01


def test_P9_wallmodel_is_scale_consistent():
    # the law only involves u+ and y+: scaling (U2, nu) -> (a U2, a nu) scales u_tau and U1 by a
    U1, ut, _, _ = O.wallmodel_speed(0.04, 1e-4)
    U1b, utb, _, _ = O.wallmodel_speed(0.08, 2e-4)
    assert abs(U1b / U1 - 2.0) < 1e-11 and abs(utb / ut - 2.0) < 1e-11


# ---- P10: inlet fix-up ------------------------------------------------------------------------
@pytest.mark.parametrize("Q", LATTICES)
def test_P10_inlet_fixup(Q):
    c, w, opp = O.lattice(Q)
    cf = c.astype(float)
    rng = np.random.default_rng(10)
    for _ in range(5):
        g = _random_state(Q, rng)
        g[c[:, 0] > 0] = rng.uniform(-5, 5, size=(c[:, 0] > 0).sum())    # unknowns are never read
        uw = np.array([0.05, 0.01 * rng.uniform(-1, 1), 0.01 * rng.uniform(-1, 1)])
        out = O.inlet_fixup_cell(Q, g, uw)
        rho = out.sum()
        # density from the known populations (textbook Zou-He relation)
        known = g[c[:, 0] == 0].sum() + 2.0 * g[c[:, 0] < 0].sum()
        assert abs(rho - known / (1.0 - uw[0])) < 1e-15
        # moments are exactly (rho, rho u_w)
        assert np.abs(cf.T @ out - rho * uw).max() < 1e-15
        # unknowns did not influence the result
        g2 = g.copy()
        g2[c[:, 0] > 0] = 0.0
        assert np.array_equal(O.inlet_fixup_cell(Q, g2, uw), out)
        # idempotent
        again = O.inlet_fixup_cell(Q, out, uw)
        assert np.abs(again - out).max() < 1e-15
        # the non-equilibrium stress of the result equals the Pi that was built
        fe = O.feq(Q, rho, uw)
        n = g - fe
        pos = c[:, 0] > 0
        n[pos] = n[opp[pos]]
        Pi_used = np.einsum("i,ia,ib->ab", n, cf, cf)
        Pi_out = np.einsum("i,ia,ib->ab", out - fe, cf, cf)
        assert np.abs(Pi_out - Pi_used).max() < 1e-15
        # and the result is f^eq + second-order Hermite projection: no higher-order content
        H2 = np.einsum("ia,ib->iab", cf, cf) - np.eye(3) / 3.0
        assert np.abs(out - (fe + 4.5 * w * np.einsum("iab,ab->i", H2, Pi_out))).max() < 1e-15

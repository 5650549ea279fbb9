"""P11a: an independent brute-force implementation of the whole step on tiny boxes, compared with the
oracle after 10 steps.  It shares nothing with oracle/: the lattice tables are the hand-typed
tests/golden files, the state is ONE vector of length Q*N, streaming is an explicit gather table built
cell by cell, the collision is evaluated in long double from the defining sums (no algebraic
simplification), the wall-model roots come from scipy's bracketing solver (the oracle uses Newton).
CPU only.
"""
import os

import numpy as np
import pytest
from scipy.optimize import brentq

import lbm_inputs as I
from oracle import oracle as O

LD = np.longdouble
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _table(Q):
    rows = [l.split() for l in open(os.path.join(GOLD, "d3q%d_R1.txt" % Q)) if l.strip() and not l.startswith("#")]
    c = np.array([[int(r[1]), int(r[2]), int(r[3])] for r in rows])
    w = np.array([LD(int(r[4])) / LD(int(r[5])) for r in rows], dtype=LD)
    opp = np.array([[j for j in range(Q) if (c[j] == -c[i]).all()][0] for i in range(Q)])
    return c, w, opp


class Brute:
    def __init__(self, Q, shape, d=None, flags=None, tau0=0.6, cs=0.0, use_hlbm=0, u_in=(0, 0, 0), wm_enable=0,
                 kappa=0.41, E=9.8):
        self.Q = Q
        self.nz, self.ny, self.nx = shape
        self.N = self.nz * self.ny * self.nx
        self.c, self.w, self.opp = _table(Q)
        self.d = np.zeros(self.N, dtype=LD) if (d is None or not use_hlbm) else d.reshape(-1).astype(LD)
        self.flags = np.zeros(self.N, dtype=np.uint8) if flags is None else flags.reshape(-1)
        self.type = self.flags & 0x0F
        self.tau0, self.cs, self.u_in = LD(tau0), LD(cs), np.array(u_in, dtype=LD)
        self.wm_enable, self.kappa, self.E = wm_enable, kappa, E
        self._build_gather()

    def cell(self, x, y, z):
        return (z * self.ny + y) * self.nx + x

    def _build_gather(self):
        """gather[i*N + x] = flat index (into the post-collision vector) that lands in (i, x)."""
        Q, N = self.Q, self.N
        self.gather = np.empty(Q * N, dtype=np.int64)
        for z in range(self.nz):
            for y in range(self.ny):
                for x in range(self.nx):
                    X = self.cell(x, y, z)
                    for i in range(Q):
                        if self.type[X] == I.SOLID:
                            self.gather[i * N + X] = i * N + X
                            continue
                        sx = x - self.c[i, 0]
                        if self.type[X] == I.OUTLET and sx > self.nx - 1:
                            sx = self.nx - 1
                        S = self.cell(sx % self.nx, (y - self.c[i, 1]) % self.ny, (z - self.c[i, 2]) % self.nz)
                        if self.type[S] == I.SOLID:
                            self.gather[i * N + X] = self.opp[i] * N + X
                        else:
                            self.gather[i * N + X] = i * N + S

    def _moments(self, fc):
        rho = LD(0)
        j = np.zeros(3, dtype=LD)
        for i in range(self.Q):
            rho = rho + fc[i]
            j = j + self.c[i].astype(LD) * fc[i]
        return rho, j / rho

    def _feq(self, rho, u):
        out = np.empty(self.Q, dtype=LD)
        cs2 = LD(1) / LD(3)
        for i in range(self.Q):
            ci = self.c[i].astype(LD)
            cu = (ci * u).sum()
            # Eq. 11 up to H(2):  w (rho + c.(rho u)/cs2 + H2 : rho u u / (2 cs2^2)),  H2 = c c - cs2 I
            h2 = LD(0)
            for a in range(3):
                for b in range(3):
                    h2 = h2 + (ci[a] * ci[b] - (cs2 if a == b else LD(0))) * rho * u[a] * u[b]
            out[i] = self.w[i] * (rho + rho * cu / cs2 + h2 / (2 * cs2 * cs2))
        return out

    def _spalding(self, up):
        k = self.kappa * up
        return up + (np.exp(k) - 1.0 - k - k * k / 2.0 - k ** 3 / 6.0) / self.E

    def _ub(self, state, X):
        """O1 for WM cell X (float64 roots from a bracketing solver)."""
        N = self.N
        code = int(self.flags[X]) >> 4
        n = np.zeros(3, dtype=int)
        n[code >> 1] = -1 if (code & 1) else 1
        x, y, z = X % self.nx, (X // self.nx) % self.ny, X // (self.nx * self.ny)
        S = self.cell((x + n[0]) % self.nx, (y + n[1]) % self.ny, (z + n[2]) % self.nz)
        if self.type[S] == I.SOLID:
            return np.zeros(3, dtype=LD)
        _, u2 = self._moments(state[np.arange(self.Q) * N + S])
        u2 = u2.astype(np.float64)
        ut = u2 - (u2 @ n) * n
        U2 = float(np.sqrt((ut * ut).sum()))
        if U2 < 1e-14:
            return np.zeros(3, dtype=LD)
        nu = float((self.tau0 - LD(0.5)) / 3)
        utau = brentq(lambda t: self._spalding(U2 / t) - 1.5 * t / nu, 1e-12, 10.0, xtol=1e-300, rtol=1e-15, maxiter=500)
        y1p = 0.5 * utau / nu
        u1p = brentq(lambda p: self._spalding(p) - y1p, 0.0, y1p + 1.0, xtol=1e-300, rtol=1e-15, maxiter=500)
        return (ut * (u1p * utau / U2)).astype(LD)

    def step(self, state):
        Q, N = self.Q, self.N
        post = state.copy()
        sqrt2 = np.sqrt(LD(2))
        for X in range(N):
            if self.type[X] == I.SOLID:
                continue
            idx = np.arange(Q) * N + X
            fc = state[idx]
            rho, u = self._moments(fc)
            ub = np.zeros(3, dtype=LD)
            if self.type[X] == I.WALLMODEL and self.wm_enable:
                ub = self._ub(state, X)
            uh = (1 - self.d[X]) * u + self.d[X] * ub
            fe = self._feq(rho, uh)
            tau = self.tau0
            if self.cs > 0:
                Pi = np.zeros((3, 3), dtype=LD)
                for i in range(Q):
                    ci = self.c[i].astype(LD)
                    Pi = Pi + np.outer(ci, ci) * (fc[i] - fe[i])
                nPi = np.sqrt((Pi * Pi).sum())
                # Eq. 14 + Eq. 3-5: positive root of tau^2 - tau0 tau - sqrt(2) Cs^2 |Pi| / (2 rho cs2^2) = 0
                q = sqrt2 * self.cs * self.cs * nPi / (2 * rho * (LD(1) / 9))
                tau = (self.tau0 + np.sqrt(self.tau0 * self.tau0 + 4 * q)) / 2
            post[idx] = fe + (1 - 1 / tau) * (fc - fe)          # Eq. 6 with f~(1) = f - feq
        new = post[self.gather]
        cf = self.c.astype(LD)
        for X in range(N):
            if self.type[X] != I.INLET:
                continue
            idx = np.arange(Q) * N + X
            g = new[idx]
            k0, km, kp = self.c[:, 0] == 0, self.c[:, 0] < 0, self.c[:, 0] > 0
            rho = (g[k0].sum() + 2 * g[km].sum()) / (1 - self.u_in[0])
            fe = self._feq(rho, self.u_in)
            nq = g - fe
            nq[kp] = nq[self.opp[kp]]
            Pi = np.einsum("i,ia,ib->ab", nq, cf, cf)
            H2 = np.einsum("ia,ib->iab", cf, cf) - np.eye(3, dtype=LD) / 3
            new[idx] = fe + self.w * LD(4.5) * np.einsum("iab,ab->i", H2, Pi)
        return new


def _rand_state(Q, shape, seed):
    rng = np.random.default_rng(seed)
    rho = 1.0 + 0.03 * rng.uniform(-1, 1, size=shape)
    u = 0.05 * rng.uniform(-1, 1, size=(3,) + shape)
    f = O.init_equilibrium(Q, rho, u)
    return f * (1.0 + 0.02 * rng.uniform(-1, 1, size=f.shape))


@pytest.mark.parametrize("Q", [19, 27])
def test_P11a_bruteforce_4cubed_periodic_les_hlbm(Q):
    shape = (4, 4, 4)
    f = _rand_state(Q, shape, seed=110 + Q)
    rng = np.random.default_rng(5)
    d = rng.uniform(0, 1, size=shape) * (rng.uniform(size=shape) < 0.4)
    par = dict(tau0=0.53, cs_smago=0.12, use_hlbm=1)
    got = O.step(f, d=d, nsteps=10, **par)
    b = Brute(Q, shape, d=d, tau0=0.53, cs=0.12, use_hlbm=1)
    s = f.reshape(-1).astype(LD)
    for _ in range(10):
        s = b.step(s)
    assert np.abs(got.reshape(-1) - s.astype(np.float64)).max() <= 1e-13


@pytest.mark.parametrize("Q", [19, 27])
def test_P11a_bruteforce_4cubed_with_solids(Q):
    shape = (4, 4, 4)
    f = _rand_state(Q, shape, seed=210 + Q)
    rng = np.random.default_rng(6)
    flags = (rng.uniform(size=shape) < 0.2).astype(np.uint8) * I.SOLID
    assert 3 <= flags.sum() <= 30
    got = O.step(f, flags=flags, nsteps=10, tau0=0.6, cs_smago=0.1)
    b = Brute(Q, shape, flags=flags, tau0=0.6, cs=0.1)
    s = f.reshape(-1).astype(LD)
    for _ in range(10):
        s = b.step(s)
    assert np.abs(got.reshape(-1) - s.astype(np.float64)).max() <= 1e-13


def test_P11a_bruteforce_small_channel_all_boundaries():
    """8 x 4 x 6 channel: SOLID floor/top, INLET, OUTLET, wall-model floor cells, a porous block, LES."""
    nz, ny, nx = 6, 4, 8
    shape = (nz, ny, nx)
    flags = np.zeros(shape, dtype=np.uint8)
    flags[0] = I.SOLID
    flags[nz - 1] = I.SOLID
    flags[1:nz - 1, :, 0] = I.INLET
    flags[1:nz - 1, :, nx - 1] = I.OUTLET
    d = np.zeros(shape)
    d[1:3, 1:3, 3:5] = 1.0
    d[3, :, 5] = 0.35
    wm = (flags[1] == I.FLUID) & (d[1] == 0)
    flags[1][wm] = I.WM_FLOOR
    d[1][wm] = 1.0
    flags[nz - 2, 2, 4] = I.WALLMODEL | (5 << 4)        # one ceiling WM cell, normal -z
    rho = np.ones(shape)
    u = np.zeros((3,) + shape)
    u[0][(flags & 15) != I.SOLID] = 0.05
    rng = np.random.default_rng(7)
    u[1] = 0.01 * rng.uniform(-1, 1, size=shape)
    f = O.init_equilibrium(19, rho, u)
    tau0 = 0.5 + 3e-4
    par = dict(tau0=tau0, cs_smago=0.1, use_hlbm=1, u_in=(0.05, 0.002, -0.001), wm_enable=1)
    got = O.step(f, d=d, flags=flags, nsteps=10, **par)
    b = Brute(19, shape, d=d, flags=flags, tau0=tau0, cs=0.1, use_hlbm=1, u_in=par["u_in"], wm_enable=1)
    s = f.reshape(-1).astype(LD)
    for _ in range(10):
        s = b.step(s)
    assert np.abs(got.reshape(-1) - s.astype(np.float64)).max() <= 1e-12
    # the run exercised every rule
    assert np.abs(got - f).max() > 1e-3

"""T1 for the prescribed solid velocity field u^B(x,t) of Eq. 12 and the time-varying porosity d(x,t) (moving
porous bodies of Fig. 1; reading G39): GPU-vs-oracle parity through the C ABI (lbm_set_body_velocity,
lbm_set_porosity), tolerances of DESIGN.md R12.  The oracle side is orc_step_body, pinned by U1-U6 (tests/test_oracle_body.py)."""
import numpy as np
import pytest
import torch

import lbm_inputs as I
import paper_2506_21804_b200 as P
from oracle import oracle as O
from parity_util import NP_DTYPE, TOL, field_error, nonsolid, oracle_inputs

pytestmark = pytest.mark.gpu


def _body_field(cfg, rng, amp=0.04):
    """u^B: non-zero on every porous cell (buildings d = 1 included: they then drive the flow), junk where d = 0 (no weight)."""
    ub = amp * rng.standard_normal((3,) + tuple(cfg["shape"]))
    return ub


def _run_pair(cfg, dtype, ub, nsteps=10, host=True, vector=None, split=None):
    npdt = NP_DTYPE[dtype]
    f, d = oracle_inputs(cfg, dtype)
    ubr = ub.astype(npdt)
    nth = min(O.max_threads(), 8)
    ref = O.step(f.astype(np.float64), d=d.astype(np.float64), flags=cfg["flags"], nsteps=nsteps, nthreads=nth,
                 u_body=ubr.astype(np.float64), **cfg["params"])
    nz, ny, nx = cfg["shape"]
    with P.LBM(cfg["Q"], nx, ny, nz, dtype) as sim:
        if vector is not None:
            sim.set_option("vector", vector)
        if host:
            sim.set_fields(f, d, cfg["flags"])
            sim.set_body_velocity(ubr)
        else:
            sim.set_fields(torch.from_numpy(f).cuda(), torch.from_numpy(d).cuda(),
                           None if cfg["flags"] is None else torch.from_numpy(cfg["flags"]).cuda())
            sim.set_body_velocity(torch.from_numpy(ubr).cuda())
        for n in (split or [nsteps]):
            sim.step(n, P.LbmParams(**cfg["params"]))
        got = np.empty_like(f)
        u = np.empty((3, nz, ny, nx), dtype=npdt)
        sim.moments(None, u)
        sim.get_populations(got)
    return f, got, u, ref


def _check(cfg, dtype, ub, **kw):
    f, got, u, ref = _run_pair(cfg, dtype, ub, **kw)
    mask = nonsolid(cfg)
    assert np.isfinite(got).all()
    e_f = field_error(got, ref, mask)
    e_u = field_error(u, O.moments(ref)[1], mask)
    assert e_f <= TOL[dtype], ("populations", e_f)
    assert e_u <= TOL[dtype], ("u", e_u)
    return f, got, ref


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("Q", [19, 27])
def test_urban_channel_with_moving_bodies(Q, dtype):
    """config 3 geometry (walls, inlet, outlet, wall-model floor, porous blobs) with a solid velocity on every porous cell"""
    cfg = I.make_config(3, shape=(40, 48, 160))
    cfg["Q"] = Q
    rng = np.random.Generator(np.random.PCG64(90 + Q))
    ub = _body_field(cfg, rng)
    f, got, ref = _check(cfg, dtype, ub)
    # the field did act: the same run without it differs
    plain = O.step(f.astype(np.float64), d=cfg["d"].astype(NP_DTYPE[dtype]).astype(np.float64), flags=cfg["flags"], nsteps=10,
                   nthreads=min(O.max_threads(), 8), **cfg["params"])
    assert field_error(plain, ref, nonsolid(cfg)) > 1e-3


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_moving_bodies_hrr_form(dtype):
    cfg = I.make_config(3, shape=(24, 32, 64))
    cfg["params"] = dict(cfg["params"], collision=1, sigma=0.7)
    rng = np.random.Generator(np.random.PCG64(95))
    _check(cfg, dtype, _body_field(cfg, rng))


def test_scalar_kernel_device_buffers_and_chunked_stepping():
    cfg = I.make_config(3, shape=(20, 24, 44))       # nx = 44: not a multiple of 8 -> scalar kernel
    rng = np.random.Generator(np.random.PCG64(96))
    ub = _body_field(cfg, rng)
    _check(cfg, "f64", ub, host=False, split=[1, 3, 6])
    cfg2 = I.make_config(3, shape=(20, 24, 64))
    ub2 = _body_field(cfg2, rng)
    _check(cfg2, "f32", ub2, host=False, split=[4, 1, 5])
    _check(cfg2, "f64", ub2, vector=0)


def test_body_velocity_is_ignored_without_weight_and_can_be_switched_off():
    cfg = I.make_config(3, shape=(20, 24, 64))
    rng = np.random.Generator(np.random.PCG64(97))
    f, d = oracle_inputs(cfg, "f64")
    nz, ny, nx = cfg["shape"]
    par = P.LbmParams(**cfg["params"])
    junk = 0.05 * rng.standard_normal((3, nz, ny, nx))
    junk[:, d > 0] = 0.0

    def run(setup):
        with P.LBM(19, nx, ny, nz, "f64") as sim:
            sim.set_fields(f, d, cfg["flags"])
            setup(sim)
            sim.step(6, par)
            out = np.empty_like(f)
            sim.get_populations(out)
        return out

    plain = run(lambda s: None)
    assert np.array_equal(run(lambda s: s.set_body_velocity(junk)), plain)          # u^B only where d = 0: bit-identical
    full = 0.05 * rng.standard_normal((3, nz, ny, nx))
    assert np.array_equal(run(lambda s: (s.set_body_velocity(full), s.set_body_velocity(None))), plain)
    assert not np.array_equal(run(lambda s: s.set_body_velocity(full)), plain)
    # WALLMODEL cells keep the wall model's u^B (G39)
    wm = (cfg["flags"] & 15) == I.WALLMODEL
    full2 = full.copy()
    full2[:, wm] = 0.0
    assert np.array_equal(run(lambda s: s.set_body_velocity(full2)), run(lambda s: s.set_body_velocity(full)))


@pytest.mark.parametrize("dtype,collision", [("f64", 0), ("f32", 0), ("f64", 1)])
def test_translating_porous_body_with_time_varying_porosity(dtype, collision):
    """A porous body that moves: d(x,t) and u^B(x,t) are re-set before every step (lbm_set_porosity + lbm_set_body_velocity,
    no pass over the lattice), 12 steps, on both sides."""
    npdt = NP_DTYPE[dtype]
    nz, ny, nx = 16, 24, 64
    shape = (nz, ny, nx)
    rng = np.random.Generator(np.random.PCG64(98))
    flags = np.zeros(shape, dtype=np.uint8)
    flags[0] = I.SOLID
    flags[-1] = I.SOLID
    rho = 1.0 + 0.01 * rng.standard_normal(shape)
    u = 0.02 * rng.standard_normal((3,) + shape)
    u[:, I.is_wall(flags)] = 0.0
    cfg = dict(Q=19, shape=shape, rho=rho, u=u, d=None, flags=flags, dtype=dtype)
    f, _ = oracle_inputs(cfg, dtype)
    params = dict(tau0=0.55, cs_smago=0.1, use_hlbm=1, collision=collision, sigma=0.8)
    ubv = np.array([0.05, 0.01, -0.004])

    def body(t):
        x0 = 5 + t // 2
        d = np.zeros(shape)
        d[3:9, 6:15, x0:x0 + 11] = 0.7
        d[5:7, 9:12, x0 + 3:x0 + 8] = 1.0
        ub = np.zeros((3,) + shape)
        ub[:, d > 0] = ubv[:, None]
        return d.astype(npdt), ub.astype(npdt)

    ref = f.astype(np.float64)
    with P.LBM(19, nx, ny, nz, dtype) as sim:
        sim.set_fields(f, None, flags)
        launches0 = None
        for t in range(12):
            d, ub = body(t)
            ref = O.step(ref, d=d.astype(np.float64), flags=flags, nsteps=1, u_body=ub.astype(np.float64), **params)
            sim.set_porosity(d)
            sim.set_body_velocity(ub)
            sim.step(1, P.LbmParams(**params))
            if t == 1:
                launches0 = sim.query("launches")
        per_step = (sim.query("launches") - launches0) / 10.0
        got = np.empty_like(f)
        sim.get_populations(got)
    assert field_error(got, ref, ~I.is_wall(flags)) <= TOL[dtype]
    assert per_step == (2 if collision else 1)           # no materialising pass between the steps

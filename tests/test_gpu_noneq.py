"""T1 from a generic NON-EQUILIBRIUM state: every other parity test starts from f^eq(rho, u), so the non-equilibrium stress that
drives tau_eff (Eq. 14) and the regularisation of the HRR form (Eq. 8-9) only has the amplitude ten steps produce.  Here both
sides are handed f = f^eq (1 + 0.02 xi), xi ~ U(-1,1) seeded per population and cell (the state the CPU pins use,
tests/test_oracle_cell.py::_random_state), rounded to the run's dtype: |Pi^neq| is O(1e-2) from the first collision on.
Both lattices, both dtypes, both collision forms, with every boundary rule of config 3 and the bounce-back spheres of config 4."""
import numpy as np
import pytest

import lbm_inputs as I
from oracle import oracle as O
from parity_util import NP_DTYPE, TOL, field_error, nonsolid, oracle_inputs, run_oracle
from test_gpu_parity import gpu_run

pytestmark = pytest.mark.gpu
NOISE = 0.02


def _noneq_inputs(cfg, dtype, seed):
    f, d = oracle_inputs(cfg, "f64")
    rng = np.random.Generator(np.random.PCG64(seed))
    f = f * (1.0 + NOISE * rng.uniform(-1.0, 1.0, size=f.shape))
    npdt = NP_DTYPE[dtype]
    return f.astype(npdt), None if d is None else d.astype(npdt)


def _check(cfg, dtype, seed, nsteps=10):
    f, d = _noneq_inputs(cfg, dtype, seed)
    # the start really is far from equilibrium: second moment of f - f^eq(rho, u) of the same cell
    rho, u = O.moments(f.astype(np.float64))
    neq = f.astype(np.float64) - O.init_equilibrium(cfg["Q"], rho, u)
    assert np.abs(neq).max() > 1e-3
    ref = run_oracle(cfg, f, d, nsteps)
    got, grho, gu, tot = gpu_run(cfg, f, d, nsteps, dtype)
    mask = nonsolid(cfg)
    assert np.isfinite(got).all() and np.isfinite(ref).all()
    rr, ru = O.moments(ref)
    e = (field_error(got, ref, mask), field_error(grho, rr, mask), field_error(gu, ru, mask))
    assert max(e) <= TOL[dtype], e
    if mask is not None:
        assert np.array_equal(got[:, ~mask], f[:, ~mask])
    rt = O.totals(ref, cfg["flags"])
    assert np.abs(tot - rt).max() <= max(TOL[dtype], 1e-12) * abs(rt[0])
    return e


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("coll", [0, 1])
@pytest.mark.parametrize("Q", [19, 27])
def test_nonequilibrium_start_urban_channel(Q, coll, dtype):
    """inlet, outlet, wall model, porosity, bounce-back floor and top; Smagorinsky on"""
    cfg = I.make_config(3, shape=(24, 32, 96))
    cfg["Q"] = Q
    cfg["params"] = dict(cfg["params"], collision=coll, sigma=0.7)
    _check(cfg, dtype, 9000 + Q + coll)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("coll", [0, 1])
def test_nonequilibrium_start_d3q27_spheres(coll, dtype):
    """config 4 scaled down: nu = 1e-5, Cs = 0.12, read-side bounce-back at the spheres"""
    cfg = I.make_config(4, shape=(40, 40, 64), k_max=6, n_modes=64)
    cfg["params"] = dict(cfg["params"], collision=coll, sigma=0.7)
    _check(cfg, dtype, 9100 + coll)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_nonequilibrium_start_periodic_les_d3q19(dtype):
    """config 2 scaled down (no flags at all: the pure bulk path), BGK + Smagorinsky at nu = 1e-5"""
    cfg = I.make_config(2, shape=(32, 32, 64), k_max=6, n_modes=64)
    _check(cfg, dtype, 9200)


def test_nonequilibrium_start_paper_boundary_set():
    """config 7 scaled down (pressure outlet + fringe zone, slip walls, wall-modelled floor), both collision forms, fp64"""
    for coll in (0, 1):
        cfg = I.make_config(7, shape=(24, 32, 96))
        cfg["params"] = dict(cfg["params"], collision=coll, sigma=0.7)
        _check(cfg, "f64", 9300 + coll)

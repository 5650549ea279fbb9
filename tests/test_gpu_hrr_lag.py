"""T1 for lbm_params.collision = 2 (reading G41): the HRR form with the FD strain of Eq. 10 taken of u^ of the PREVIOUS
time level -- one pass over the lattice per step.  GPU-vs-oracle parity through the C ABI, element by element, same seeded inputs,
10 steps, tolerances as for the other forms (fp64 <= 1e-12, fp32 <= 2e-5).  The oracle side is orc_step with collision = 2, pinned
by tests/test_oracle_hrr_lag.py L1-L5.  Also: the history lives in the context (chunked stepping and state reads in between give
the same populations bit for bit), state setters drop it, one step is one launch of the fused kernel (+ the wall-model pre-pass)."""
import numpy as np
import pytest

import lbm_inputs as I
import paper_2506_21804_b200 as P
from oracle import oracle as O
from parity_util import TOL, field_error, nonsolid, oracle_inputs, run_oracle
from test_gpu_parity import check_parity, gpu_run

pytestmark = pytest.mark.gpu


def lag(cfg, sigma):
    cfg = dict(cfg)
    cfg["params"] = dict(cfg["params"], collision=2, sigma=sigma)
    return cfg


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("sigma", [1.0, 0.7, 0.0])
def test_lag_periodic_les(dtype, sigma):
    check_parity(lag(I.make_config(2, shape=(32, 48, 64), k_max=6, n_modes=64), sigma), dtype)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_lag_urban_channel_all_boundary_rules(dtype):
    """inlet / outlet ghost planes of the FD stencil (G32), wall model with sigma = 0 (l.131), porosity, bounce-back, list cells"""
    cfg = lag(I.make_config(3, shape=(40, 48, 160)), 0.7)
    t = cfg["flags"] & 15
    assert (t == I.WALLMODEL).any() and (t == I.INLET).any() and (t == I.OUTLET).any() and (cfg["d"] > 0).any()
    check_parity(cfg, dtype)
    check_parity(cfg, dtype, split=[1, 2, 3, 4])                  # the history is the context's, not the call's


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_lag_paper_boundary_set_with_wall_model_on_building_faces(dtype):
    check_parity(lag(I.make_config(8, shape=(32, 48, 96)), 0.7), dtype)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_lag_d3q27_spheres(dtype):
    check_parity(lag(I.make_config(4, shape=(48, 48, 48), k_max=6, n_modes=64), 0.5), dtype)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_lag_d3q27_urban(dtype):
    cfg = I.make_config(5, shape=(32, 32, 64))
    cfg["Q"] = 27
    check_parity(lag(cfg, 0.9), dtype)


@pytest.mark.parametrize("shape", [(4, 4, 4), (7, 13, 37), (5, 9, 130)])
def test_lag_scalar_kernel_ragged_shapes(shape):
    rng = np.random.Generator(np.random.PCG64(78))
    rho = 1.0 + 0.02 * rng.standard_normal(shape)
    u = 0.04 * rng.standard_normal((3,) + shape)
    flags = np.zeros(shape, dtype=np.uint8)
    flags[rng.random(shape) < 0.1] = I.SOLID
    d = np.where(rng.random(shape) < 0.2, rng.uniform(0.1, 0.9, shape), 0.0)
    cfg = dict(Q=19, shape=shape, rho=rho, u=u, d=d, flags=flags, dtype="f64",
               params=dict(tau0=0.56, cs_smago=0.12, use_hlbm=1, collision=2, sigma=0.8))
    check_parity(cfg, "f64")
    check_parity(cfg, "f32")


def test_lag_from_a_non_equilibrium_state():
    cfg = lag(I.make_config(3, shape=(24, 32, 96)), 0.6)
    f, d = oracle_inputs(cfg, "f64")
    rng = np.random.Generator(np.random.PCG64(5))
    f = f * (1.0 + 0.02 * rng.standard_normal(f.shape))
    ref = run_oracle(cfg, f, d, 10)
    got, *_ = gpu_run(cfg, f, d, 10, "f64")
    assert field_error(got, ref, nonsolid(cfg)) <= TOL["f64"]
    assert field_error(got, run_oracle(dict(cfg, params=dict(cfg["params"], collision=1)), f, d, 10), nonsolid(cfg)) > 1e-9   # not form 1


def test_lag_history_chunks_state_reads_setters_and_launch_count():
    cfg = lag(I.make_config(3, shape=(24, 32, 96)), 0.7)
    f, d = oracle_inputs(cfg, "f32")
    nz, ny, nx = cfg["shape"]
    par = P.LbmParams(**cfg["params"])
    m = nonsolid(cfg)
    with P.LBM(19, nx, ny, nz, "f32") as sim:
        sim.set_fields(f, d, cfg["flags"])
        sim.step(6, par)
        a = np.empty_like(f)
        sim.get_populations(a)
    with P.LBM(19, nx, ny, nz, "f32") as sim:
        sim.set_fields(f, d, cfg["flags"])
        b = np.empty_like(f)
        rho = np.empty((nz, ny, nx), np.float32)
        for n in (1, 2, 3):
            sim.step(n, par)
            sim.get_populations(b)                                # materialises S_t: the history stays
            sim.moments(rho, None)
        assert np.array_equal(a, b)
        l0 = sim.query("launches")
        sim.step(4, par)
        assert sim.query("launches") - l0 == 4 * 2                # fused step + wall-model pre-pass: no u^ pass
        # a state setter drops the history: the next step differences u^ of its own level again, like a fresh context
        sim.set_fields(f, d, cfg["flags"])
        sim.step(6, par)
        sim.get_populations(b)
        assert np.array_equal(a, b)
    assert field_error(a, run_oracle(cfg, f, d, 6), m) <= TOL["f32"]
    # forms 1 and 2 on one context: switching to form 2 after steps of form 1 continues from the u^ history form 2 itself kept
    # (none yet: its first step is a form-1 step)
    one = dict(cfg, params=dict(cfg["params"], collision=1))
    mid = run_oracle(one, f, d, 3)
    ref = O.step(mid, d=d.astype(np.float64), flags=cfg["flags"], nsteps=3, nthreads=4, **cfg["params"])
    with P.LBM(19, nx, ny, nz, "f32") as sim:
        sim.set_fields(f, d, cfg["flags"])
        sim.step(3, P.LbmParams(**one["params"]))
        sim.step(3, par)
        sim.get_populations(b)
    assert field_error(b, ref, m) <= TOL["f32"]
    # ... and steps of another form in between drop the history (the oracle: every call starts without one)
    kw = dict(d=d.astype(np.float64), flags=cfg["flags"], nthreads=4)
    r = O.step(f.astype(np.float64), nsteps=2, **kw, **cfg["params"])
    r = O.step(r, nsteps=1, **kw, **one["params"])
    r = O.step(r, nsteps=3, **kw, **cfg["params"])
    with P.LBM(19, nx, ny, nz, "f32") as sim:
        sim.set_fields(f, d, cfg["flags"])
        sim.step(2, par)
        sim.step(1, P.LbmParams(**one["params"]))
        sim.step(3, par)
        sim.get_populations(b)
    assert field_error(b, r, m) <= TOL["f32"]


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_lag_lid_driven_cavity(dtype):
    """MOVINGWALL cells: their u^ entries are the lid velocity (G33); a new lid velocity starts a new history"""
    cfg = lag(I.make_config(6, shape=(24, 32, 64)), 0.7)
    check_parity(cfg, dtype)
    f, d = oracle_inputs(cfg, dtype)
    nz, ny, nx = cfg["shape"]
    fast = dict(cfg["params"], u_wall=tuple(1.5 * v for v in cfg["params"]["u_wall"]))
    kw = dict(d=None if d is None else d.astype(np.float64), flags=cfg["flags"], nthreads=4)
    r = O.step(f.astype(np.float64), nsteps=3, **kw, **cfg["params"])
    r = O.step(r, nsteps=3, **kw, **fast)
    with P.LBM(19, nx, ny, nz, dtype) as sim:
        sim.set_fields(f, d, cfg["flags"])
        out = np.empty_like(f)
        sim.step(3, P.LbmParams(**cfg["params"]))
        sim.get_populations(out)        # S_3 is formed with the old lid velocity, as at the end of the oracle's first call
        sim.step(3, P.LbmParams(**fast))
        sim.get_populations(out)
    assert field_error(out, r, nonsolid(cfg)) <= TOL[dtype]


@pytest.mark.parametrize("key,values", [("serpentine", (1, 0)), ("pdl", (2, 1, 0)), ("block_threads", (64, 128, 256)), ("cuda_graph", (0, 1)),
                                        ("vector", (1, 0))])
def test_lag_schedule_knobs_are_bit_identical(key, values):
    """schedules, not arithmetic ("vector" = 0 routes every cell through the per-cell kernel: agreement to rounding); with
    "cuda_graph" = 1 the form still steps with plain launches (its u^ buffers swap roles every step)"""
    cfg = lag(I.make_config(3, shape=(24, 32, 96)), 0.7)
    f, d = oracle_inputs(cfg, "f32")
    nz, ny, nx = cfg["shape"]
    par = P.LbmParams(**cfg["params"])
    outs = []
    for v in values:
        with P.LBM(19, nx, ny, nz, "f32") as sim:
            sim.set_option(key, v)
            sim.set_fields(f, d, cfg["flags"])
            sim.step(11, par)
            sim.step(9, par)
            assert sim.query("graph_launches") == 0
            out = np.empty_like(f)
            sim.get_populations(out)
            outs.append(out)
    for o in outs[1:]:
        if key == "vector":
            assert field_error(o, outs[0], nonsolid(cfg)) <= 2e-6
        else:
            assert np.array_equal(o, outs[0]), key
    assert field_error(outs[0], run_oracle(cfg, f, d, 20), nonsolid(cfg)) <= 2 * TOL["f32"]

"""T1 for the HRR form (lbm_params.collision = 1): GPU-vs-oracle parity through the C ABI, element by
element, same seeded inputs, 10 steps.  Tolerances as for the BGK form (R12): fp64 <= 1e-12, fp32 <= 2e-5.
The oracle side is orc_step with collision = 1 (Eq. 6-11 in full, pinned by tests/test_oracle_hrr.py H1-H10)."""
import numpy as np
import pytest
import torch

import lbm_inputs as I
import paper_2506_21804_b200 as P
from oracle import oracle as O
from parity_util import TOL, field_error, nonsolid, oracle_inputs, run_oracle
from test_gpu_parity import check_parity, gpu_run

pytestmark = pytest.mark.gpu


def hrr(cfg, sigma):
    cfg = dict(cfg)
    cfg["params"] = dict(cfg["params"], collision=1, sigma=sigma)
    return cfg


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("sigma", [1.0, 0.7, 0.0])
def test_hrr_periodic_les(dtype, sigma):
    cfg = hrr(I.make_config(2, shape=(32, 48, 64), k_max=6, n_modes=64), sigma)
    check_parity(cfg, dtype)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_hrr_urban_channel_all_boundary_rules(dtype):
    """inlet / outlet ghost planes of the FD stencil (G32), wall model with sigma = 0 (l.131), porosity, bounce-back"""
    cfg = hrr(I.make_config(3, shape=(40, 48, 160)), 0.7)
    t = cfg["flags"] & 15
    assert (t == I.WALLMODEL).any() and (t == I.INLET).any() and (t == I.OUTLET).any() and (cfg["d"] > 0).any()
    check_parity(cfg, dtype)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_hrr_d3q27_spheres(dtype):
    cfg = hrr(I.make_config(4, shape=(48, 48, 48), k_max=6, n_modes=64), 0.5)
    check_parity(cfg, dtype)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_hrr_d3q27_urban(dtype):
    cfg = I.make_config(5, shape=(32, 32, 64))
    cfg["Q"] = 27
    check_parity(hrr(cfg, 0.9), dtype)


@pytest.mark.parametrize("slab", [1, 3, 8, 1000])
def test_hrr_slab_schedule_gives_identical_results(slab):
    """the z-slab interleaving of the two passes is a schedule, not arithmetic: bit-identical populations"""
    cfg = hrr(I.make_config(3, shape=(24, 32, 64)), 0.6)
    f, d = oracle_inputs(cfg, "f32")
    nz, ny, nx = cfg["shape"]
    outs = []
    for s in (0, slab):
        with P.LBM(19, nx, ny, nz, "f32") as sim:
            sim.set_option("hrr_slab", s)
            sim.set_fields(f, d, cfg["flags"])
            sim.step(4, P.LbmParams(**cfg["params"]))
            sim.step(3, P.LbmParams(**cfg["params"]))
            out = np.empty_like(f)
            sim.get_populations(out)
            outs.append(out)
    assert np.array_equal(outs[0], outs[1])
    ref = run_oracle(cfg, f, d, 7)
    assert field_error(outs[1], ref, nonsolid(cfg)) <= TOL["f32"]


@pytest.mark.parametrize("shape", [(4, 4, 4), (7, 13, 37), (5, 9, 130)])
def test_hrr_scalar_kernel_ragged_shapes(shape):
    """row lengths the vector kernel does not take go through k_step (one cell per thread)"""
    nz, ny, nx = shape
    rng = np.random.Generator(np.random.PCG64(77))
    rho = 1.0 + 0.02 * rng.standard_normal(shape)
    u = 0.04 * rng.standard_normal((3,) + shape)
    flags = np.zeros(shape, dtype=np.uint8)
    flags[rng.random(shape) < 0.1] = I.SOLID
    d = np.where(rng.random(shape) < 0.2, rng.uniform(0.1, 0.9, shape), 0.0)
    cfg = dict(Q=19, shape=shape, rho=rho, u=u, d=d, flags=flags, dtype="f64",
               params=dict(tau0=0.56, cs_smago=0.12, use_hlbm=1, collision=1, sigma=0.8))
    check_parity(cfg, "f64")
    check_parity(cfg, "f32")


def test_hrr_switching_collision_between_calls_and_vector_off():
    cfg = hrr(I.make_config(3, shape=(24, 32, 64)), 0.7)
    f, d = oracle_inputs(cfg, "f64")
    a, *_ = gpu_run(cfg, f, d, 6, "f64")
    b, *_ = gpu_run(cfg, f, d, 6, "f64", vector=0)
    ref = run_oracle(cfg, f, d, 6)
    m = nonsolid(cfg)
    assert field_error(a, ref, m) <= 1e-12 and field_error(b, ref, m) <= 1e-12
    # BGK steps then HRR steps on the same context
    bgk = dict(cfg, params=dict(cfg["params"], collision=0))
    mid = run_oracle(bgk, f, d, 3)
    ref2 = O.step(mid, d=d, flags=cfg["flags"], nsteps=3, **cfg["params"])
    nz, ny, nx = cfg["shape"]
    with P.LBM(19, nx, ny, nz, "f64") as sim:
        sim.set_fields(f, d, cfg["flags"])
        sim.step(3, P.LbmParams(**bgk["params"]))
        sim.step(3, P.LbmParams(**cfg["params"]))
        out = np.empty_like(f)
        sim.get_populations(out)
    assert field_error(out, ref2, m) <= 1e-12


def test_hrr_rejects_bad_sigma_and_collision():
    with P.LBM(19, 8, 8, 8, "f32") as sim:
        sim.init_equilibrium(np.ones((8, 8, 8), np.float32), np.zeros((3, 8, 8, 8), np.float32))
        for bad in (dict(collision=1, sigma=1.5), dict(collision=1, sigma=-0.1), dict(collision=3), dict(collision=2, sigma=1.5)):
            with pytest.raises(P.LbmError):
                sim.step(1, P.LbmParams(0.6, **bad))

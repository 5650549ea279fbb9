"""T1 for the moving-wall rule (lid-driven cavity, the paper's scaling benchmark; reading G33):
GPU-vs-oracle parity through the C ABI on the cavity and on lids with holes, 10 steps, tolerances of DESIGN.md R12."""
import numpy as np
import pytest

import lbm_inputs as I
import paper_2506_21804_b200 as P
from oracle import oracle as O
from parity_util import TOL, field_error, nonsolid, oracle_inputs, run_oracle
from test_gpu_parity import check_parity, gpu_run

pytestmark = pytest.mark.gpu


def _start(cfg, seed=6):
    """a cavity that is already moving: seeded velocity / density perturbation on the fluid cells"""
    rng = np.random.Generator(np.random.PCG64(seed))
    cfg = dict(cfg)
    cfg["rho"] = 1.0 + 0.01 * rng.standard_normal(cfg["shape"])
    u = 0.03 * rng.standard_normal((3,) + cfg["shape"])
    u[:, I.is_wall(cfg["flags"])] = 0.0
    cfg["u"] = u
    return cfg


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("Q", [19, 27])
def test_cavity_bgk_les(Q, dtype):
    cfg = _start(I.make_config(6, shape=(24, 20, 64)))
    cfg["Q"] = Q
    cfg["params"] = dict(cfg["params"], u_wall=(0.05, -0.02, 0.0))
    check_parity(cfg, dtype)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_cavity_hrr(dtype):
    cfg = _start(I.make_config(6, shape=(24, 20, 64)))
    cfg["params"] = dict(cfg["params"], collision=1, sigma=0.7, u_wall=(0.05, 0.01, 0.0))
    check_parity(cfg, dtype)


@pytest.mark.parametrize("Q", [19, 27])
def test_lid_with_holes_periodic_wrap_and_normal_motion(Q):
    """lid plane z = nz-1 with MOVINGWALL, SOLID and FLUID cells mixed; no floor, so the z = 0 cells meet the lid through the
    periodic wrap; wall velocity with a normal component; ragged x rows next to full ones"""
    shape = (12, 10, 32)
    rng = np.random.Generator(np.random.PCG64(60 + Q))
    flags = np.zeros(shape, dtype=np.uint8)
    r = rng.random(shape[1:])
    flags[-1][r < 0.6] = I.MOVINGWALL
    flags[-1][(r >= 0.6) & (r < 0.8)] = I.SOLID
    flags[5][rng.random(shape[1:]) < 0.1] = I.SOLID
    cfg = _start(dict(Q=Q, shape=shape, dtype="f64", d=None, flags=flags,
                      params=dict(tau0=0.58, cs_smago=0.1, u_wall=(0.03, 0.02, -0.01))))
    check_parity(cfg, "f64")
    check_parity(cfg, "f32")
    check_parity(cfg, "f64", vector=0)
    cfg["params"] = dict(cfg["params"], collision=1, sigma=0.5)
    check_parity(cfg, "f64")


def test_movingwall_flag_only_on_the_top_plane():
    flags = np.zeros((6, 8, 8), dtype=np.uint8)
    flags[2, 3, 3] = I.MOVINGWALL
    with P.LBM(19, 8, 8, 6, "f32") as sim:
        with pytest.raises(P.LbmError):
            sim.set_geometry(None, flags)
        flags[2, 3, 3] = 0
        flags[5, 3, 3] = I.MOVINGWALL
        sim.set_geometry(None, flags)
        assert sim.query("solid_cells") == 1


def test_couette_steady_state_on_the_gpu():
    """M1 on the CUDA path: exact linear profile between a resting and a moving halfway wall (fp64)"""
    nz, ny, nx = 14, 4, 32
    flags = np.zeros((nz, ny, nx), dtype=np.uint8)
    flags[0] = I.SOLID
    flags[-1] = I.MOVINGWALL
    uw = (0.04, -0.015, 0.0)
    with P.LBM(19, nx, ny, nz, "f64") as sim:
        sim.set_geometry(None, flags)
        sim.init_equilibrium(np.ones((nz, ny, nx)), np.zeros((3, nz, ny, nx)))
        sim.step(5000, P.LbmParams(0.8, u_wall=uw))
        u = np.empty((3, nz, ny, nx))
        sim.moments(None, u)
    z = np.arange(1, nz - 1)
    for a in (0, 1):
        want = uw[a] * (z - 0.5) / (nz - 2)
        assert np.abs(u[a, 1:-1] - want[:, None, None]).max() <= 2e-9 * abs(uw[a]) + 1e-13

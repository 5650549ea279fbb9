"""T1 for the full-slip walls (reading G37): GPU-vs-oracle parity through the C ABI, 10 steps,
tolerances of DESIGN.md R12: the urban channel in the paper's boundary set (VM-less): velocity inlet, pressure outlet, slip
lateral walls and top, wall-modelled floor; a closed slip box; a slip channel with obstacles."""
import numpy as np
import pytest

import lbm_inputs as I
import paper_2506_21804_b200 as P
from test_gpu_parity import check_parity

pytestmark = pytest.mark.gpu


def _paper_channel(shape, Q=19, **extra):
    cfg = I.make_config(3, shape=shape)
    fl = cfg["flags"]
    fl[(fl & 15) == I.OUTLET] = I.POUTLET
    fl[-1] = I.SLIPWALL                       # top
    fl[1:, 0] = I.SLIPWALL                    # lateral walls (the floor row z = 0 stays SOLID)
    fl[1:, -1] = I.SLIPWALL
    cfg["d"][I.is_wall(fl)] = 0.0
    cfg["u"][:, I.is_wall(fl)] = 0.0
    cfg["Q"] = Q
    cfg["params"] = dict(cfg["params"], rho_out=1.0, **extra)
    return cfg


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("Q", [19, 27])
def test_urban_channel_with_the_papers_boundary_set(Q, dtype):
    cfg = _paper_channel((40, 48, 160), Q)
    t = cfg["flags"] & 15
    assert (t == I.SLIPWALL).any() and (t == I.POUTLET).any() and (t == I.WALLMODEL).any() and (t == I.INLET).any()
    check_parity(cfg, dtype)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_paper_boundary_set_hrr(dtype):
    check_parity(_paper_channel((24, 32, 64), collision=1, sigma=0.7), dtype)


@pytest.mark.parametrize("dtype,Q,extra", [("f32", 19, {}), ("f64", 19, {}), ("f32", 27, {}), ("f64", 19, dict(collision=1, sigma=0.7)),
                                           ("f32", 19, dict(collision=1, sigma=0.7))])
def test_paper_boundary_set_with_wall_model_on_the_building_faces(dtype, Q, extra):
    """config 8: config 7 + WALLMODEL cells on the roofs and the four side faces of the buildings"""
    cfg = I.make_config(8, shape=(40, 48, 160))
    cfg["Q"] = Q
    cfg["params"] = dict(cfg["params"], **extra)
    n = cfg["wm_face_cells"]
    assert all(n[c] > 100 for c in (0, 1, 2, 3, 4))
    check_parity(cfg, dtype)


@pytest.mark.parametrize("Q", [19, 27])
def test_closed_slip_box_with_obstacles_and_zero_gradient_outlet_corner_cases(Q):
    shape = (14, 12, 32)
    rng = np.random.Generator(np.random.PCG64(70 + Q))
    flags = np.zeros(shape, dtype=np.uint8)
    flags[0] = flags[-1] = I.SLIPWALL
    flags[:, 0] = flags[:, -1] = I.SLIPWALL
    flags[1:5, 3:6, 10:14] = I.SOLID                       # a block standing on the slip floor
    flags[6:9, 1:3, 20:23] = I.SLIPWALL                    # a slip block at the lateral wall (concave and convex edges)
    rho = 1.0 + 0.01 * rng.standard_normal(shape)
    u = 0.03 * rng.standard_normal((3,) + shape)
    u[:, I.is_wall(flags)] = 0.0
    cfg = dict(Q=Q, shape=shape, rho=rho, u=u, d=None, flags=flags, dtype="f64", params=dict(tau0=0.6, cs_smago=0.1))
    check_parity(cfg, "f64")
    check_parity(cfg, "f32")
    check_parity(cfg, "f64", vector=0)
    # with the zero-gradient outlet (its wall-adjacent cells take the per-cell path) and an inlet
    flags2 = flags.copy()
    flags2[1:-1, 1:-1, 0] = I.INLET
    flags2[1:-1, 1:-1, -1] = I.OUTLET
    cfg2 = dict(cfg, flags=flags2, params=dict(tau0=0.6, cs_smago=0.1, u_in=(0.03, 0.0, 0.0)))
    check_parity(cfg2, "f64")


def test_slip_channel_keeps_uniform_flow_on_the_gpu():
    nz, ny, nx = 10, 8, 32
    flags = np.zeros((nz, ny, nx), dtype=np.uint8)
    flags[0] = flags[-1] = I.SLIPWALL
    u = np.zeros((3, nz, ny, nx))
    u[0], u[1] = 0.05, -0.02
    with P.LBM(19, nx, ny, nz, "f64") as sim:
        sim.set_geometry(None, flags)
        sim.init_equilibrium(np.ones((nz, ny, nx)), u)
        t0 = sim.totals()
        sim.step(200, P.LbmParams(0.7))
        t1 = sim.totals()
        out = np.empty((3, nz, ny, nx))
        sim.moments(None, out)
    assert np.abs(out[:, 1:-1] - u[:, 1:-1]).max() <= 1e-14
    assert abs(t1[1] / t0[1] - 1.0) <= 1e-13

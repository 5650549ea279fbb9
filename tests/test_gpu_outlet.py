"""T1 for the pressure outlet (reading G36): GPU-vs-oracle parity through the C ABI on the urban
channel with its outlet plane switched to POUTLET cells, 10 steps, tolerances of DESIGN.md R12."""
import numpy as np
import pytest

import lbm_inputs as I
import paper_2506_21804_b200 as P
from parity_util import oracle_inputs
from test_gpu_parity import check_parity

pytestmark = pytest.mark.gpu


def _pressure_channel(shape, Q=19, **extra):
    cfg = I.make_config(3, shape=shape)
    fl = cfg["flags"]
    fl[(fl & 15) == I.OUTLET] = I.POUTLET
    cfg["Q"] = Q
    cfg["params"] = dict(cfg["params"], rho_out=0.998, **extra)
    return cfg


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("Q", [19, 27])
def test_pressure_outlet_bgk(Q, dtype):
    cfg = _pressure_channel((40, 48, 160), Q)
    assert ((cfg["flags"] & 15) == I.POUTLET).any()
    check_parity(cfg, dtype)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_pressure_outlet_hrr(dtype):
    check_parity(_pressure_channel((24, 32, 64), collision=1, sigma=0.7), dtype)


def test_pressure_outlet_scalar_kernel_and_ragged_rows():
    check_parity(_pressure_channel((12, 10, 37)), "f64")
    check_parity(_pressure_channel((24, 32, 64)), "f64", vector=0)


def test_poutlet_flag_only_on_the_last_plane_and_rho_out_checked():
    flags = np.zeros((6, 8, 8), dtype=np.uint8)
    flags[2, 3, 3] = I.POUTLET
    with P.LBM(19, 8, 8, 6, "f32") as sim:
        with pytest.raises(P.LbmError):
            sim.set_geometry(None, flags)
        flags[2, 3, 3] = 0
        flags[2, 3, 7] = I.POUTLET
        sim.set_geometry(None, flags)
        sim.init_equilibrium(np.ones((6, 8, 8), np.float32), np.zeros((3, 6, 8, 8), np.float32))
        with pytest.raises(P.LbmError):
            sim.step(1, P.LbmParams(0.6, rho_out=-1.0))


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("coll", [0, 1])
def test_fringe_zone_in_front_of_the_pressure_outlet(dtype, coll):
    """reading G38: nu_mo(x) = nu_mo (1 + A xi^2) over the last L cells (the vector path computes tau0 per cell)"""
    cfg = _pressure_channel((24, 32, 96), collision=coll, sigma=0.7, fringe_len=20, fringe_factor=8.0)
    check_parity(cfg, dtype)


def test_fringe_zone_scalar_kernel_and_bad_arguments():
    check_parity(_pressure_channel((12, 10, 37), fringe_len=9, fringe_factor=3.0), "f64")
    with P.LBM(19, 8, 8, 8, "f32") as sim:
        sim.init_equilibrium(np.ones((8, 8, 8), np.float32), np.zeros((3, 8, 8, 8), np.float32))
        for bad in (dict(fringe_len=-1), dict(fringe_factor=-0.5)):
            with pytest.raises(P.LbmError):
                sim.step(1, P.LbmParams(0.6, **bad))

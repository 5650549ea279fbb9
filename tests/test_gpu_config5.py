"""BASELINE.json config 5 (single-GPU capacity sweep, urban channel on cubes) at ITS OWN sizes ("Parity at 128^3 in
full, larger sizes by windows"): 128^3 element by element (fp32 and fp64), light-cone windows (pin P11b) at 512^3 and 896^3 fp32
and at 640^3 fp64, in the launch configuration bench.py times (library defaults).  896^3 is the size where the element offset
i*N + cell of a population passes 2^32 and a population set is 54.7 GB: the state goes in slab by slab (lbm_set_populations_box)
and comes out window by window (lbm_get_populations_box), so that neither the host nor the device ever holds a third copy.

Both sides start from the ORACLE's equilibrium populations rounded to the run's dtype: the slabs handed to the library and the
crops handed to the oracle are the same cell-local function (orc_init_equilibrium) of the same rho, u arrays.
"""
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest
import torch

import lbm_inputs as I
import paper_2506_21804_b200 as P
from oracle import oracle as O
from parity_util import NP_DTYPE, TOL, field_error
from test_gpu_fullsize import M, S, W, _axis_crop
from test_gpu_parity import check_parity

pytestmark = pytest.mark.gpu
TORCH_DTYPE = {"f32": torch.float32, "f64": torch.float64}


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_config5_128_cubed_in_full(dtype):
    cfg = I.make_config(5, shape=(128, 128, 128))
    t = cfg["flags"] & 15
    assert (t == I.WALLMODEL).sum() > 5000 and ((cfg["d"] > 0) & (cfg["d"] < 1)).mean() > 0.04
    check_parity(cfg, dtype)


def _windows(cfg):
    """>= 8 windows (z0, y0, x0): floor + inlet, floor + outlet, top, a building, a tree, wall-model floor, bulk, the last rows in y (their crops wrap), and the
    LAST slices in z and rows in y next to the outlet (the highest element offsets of the lattice)"""
    nz, ny, nx = cfg["shape"]
    d, fl = cfg["d"], cfg["flags"]
    lo = slice(2, 6)                                          # (searched on four slices near the floor only: 896^3 is large)
    b = np.argwhere((d[lo, :, : nx - W] == 1.0) & (fl[lo, :, : nx - W] == 0))
    bz, by, bx = b[len(b) // 2] + (2, 0, 0)
    t = np.argwhere((d[lo, :, : nx - W] > 0) & (d[lo, :, : nx - W] < 1))
    tz, ty, tx = t[len(t) // 3] + (2, 0, 0)
    by, ty = min(int(by), ny - W), min(int(ty), ny - W)
    return [(1, 10, 0), (1, ny // 2, nx - W), (nz - 1 - W, ny // 4, nx // 2), (max(int(bz) - 3, 1), int(by), int(bx)),
            (max(int(tz) - 3, 1), int(ty), int(tx)), (1, ny // 3, nx // 3), (nz // 2, ny // 2, nx // 2), (nz // 4, ny - W, nx // 4),
            (nz - 1 - W, ny - W, nx - W), (nz - 1 - W, ny - W, 0)]


def _lean_windows(n, dtype, steps=S, slab=8):
    cfg = I.make_config(5, shape=(n, n, n))
    nz, ny, nx = cfg["shape"]
    Q = cfg["Q"]
    npdt = NP_DTYPE[dtype]
    par = P.LbmParams(**cfg["params"])
    wins = _windows(cfg)
    d = cfg["d"].astype(npdt)
    got, got_rho, got_u = {}, {}, {}
    with P.LBM(Q, nx, ny, nz, dtype) as sim:
        sim.set_geometry(d, cfg["flags"])
        def slab_populations(z0):                              # the oracle's routine, one call per slab (it is serial: the
            zs = min(slab, nz - z0)                            # harness runs several slabs at a time; ctypes drops the GIL)
            return z0, zs, O.init_equilibrium(Q, np.ascontiguousarray(cfg["rho"][z0:z0 + zs]),
                                              np.ascontiguousarray(cfg["u"][:, z0:z0 + zs])).astype(npdt)

        starts = list(range(0, nz, slab))
        with ThreadPoolExecutor(max_workers=min(O.max_threads(), 12)) as pool:
            for k0 in range(0, len(starts), 24):               # bounded: at most 24 slabs in memory
                for z0, zs, fs in pool.map(slab_populations, starts[k0:k0 + 24]):
                    sim.set_populations_box((0, 0, z0), (nx, ny, zs), fs)
        assert sim.query("steps") == 0
        sim.step(steps, par)
        rho = torch.empty((nz, ny, nx), dtype=TORCH_DTYPE[dtype], device="cuda")
        u = torch.empty((3, nz, ny, nx), dtype=TORCH_DTYPE[dtype], device="cuda")
        sim.moments(rho, u)                                  # POST phase: pulled in registers
        for (z0, y0, x0) in wins:
            assert 0 <= y0 <= ny - W                          # (the windows of this test do not wrap; their crops may)
            got_rho[(z0, y0, x0)] = rho[z0:z0 + W, y0:y0 + W, x0:x0 + W].cpu().numpy()
            got_u[(z0, y0, x0)] = u[:, z0:z0 + W, y0:y0 + W, x0:x0 + W].cpu().numpy()
        del rho, u
        for (z0, y0, x0) in wins:
            box = np.empty((Q, W, W, W), dtype=npdt)
            sim.get_populations_box((x0, y0, z0), (W, W, W), box)
            got[(z0, y0, x0)] = box
        tot = sim.totals()
        assert np.isfinite(tot).all()
    worst = 0.0
    for (z0, y0, x0) in wins:
        iz, wz = _axis_crop(z0, nz, True)
        iy, wy = _axis_crop(y0, ny, False)
        ix, wx = _axis_crop(x0, nx, True)
        sel = np.ix_(iz, iy, ix)
        fc = O.init_equilibrium(Q, np.ascontiguousarray(cfg["rho"][sel]), np.ascontiguousarray(cfg["u"][(slice(None),) + sel]))
        fc = fc.astype(npdt).astype(np.float64)
        dc = np.ascontiguousarray(d[sel]).astype(np.float64)
        flc = np.ascontiguousarray(cfg["flags"][sel])
        ref = O.step(fc, d=dc, flags=flc, nsteps=steps, nthreads=min(O.max_threads(), 8), **cfg["params"])
        inner = (slice(None), slice(wz, wz + W), slice(wy, wy + W), slice(wx, wx + W))
        refw = ref[inner]
        gsel = np.ix_(iz[wz:wz + W], iy[wy:wy + W], ix[wx:wx + W])
        mask = ~I.is_wall(cfg["flags"][gsel])
        if not mask.any():
            continue
        gotw = got[(z0, y0, x0)].astype(np.float64)
        assert np.array_equal(gotw[:, ~mask], fc[inner][:, ~mask])          # wall cells keep what was set, bit for bit
        rr, ru = O.moments(ref)
        e_f = field_error(gotw, refw, mask)
        e_rho = field_error(got_rho[(z0, y0, x0)], rr[inner[1:]], mask)
        uw = ru[(slice(None),) + inner[1:]]
        e_u = field_error(got_u[(z0, y0, x0)], uw, mask)
        # R12 normalises by the maximum of the whole FIELD, which a window inside a building (u ~ 0) does not see; the field's
        # maximum is at least the inlet speed (the INLET plane carries u_in exactly)
        e_u *= np.abs(uw[..., mask]).max() / max(np.abs(uw[..., mask]).max(), cfg["params"]["u_in"][0])
        worst = max(worst, e_f, e_rho, e_u)
        assert e_f <= TOL[dtype], ("populations", (z0, y0, x0), e_f)
        assert e_rho <= TOL[dtype], ("rho", (z0, y0, x0), e_rho)
        assert e_u <= TOL[dtype], ("u", (z0, y0, x0), e_u)
    return worst


def test_config5_512_cubed_windows_f32():
    _lean_windows(512, "f32")


def test_config5_640_cubed_windows_f64():
    """the largest fp64 size of the sweep: 2 x 39.8 GB of populations"""
    _lean_windows(640, "f64")


def test_config5_896_cubed_windows_f32():
    """the largest size of the sweep: 719 M cells, 2 x 54.7 GB of populations, element offsets of a population set up to 1.37e10
    (> 2^32); the last windows sit in the last z-slices / y-rows, i.e. at the highest offsets of every population"""
    _lean_windows(896, "f32")

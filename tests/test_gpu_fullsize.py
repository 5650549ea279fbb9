"""T1 at BASELINE.json's FULL sizes, in the launch configuration bench.py times (library defaults), and T2 invariants.

The oracle cannot hold these sizes, so parity is checked on light-cone windows (pin P11b, DESIGN.md / SURVEY 8(c)):
information moves <= 1 cell per step (a wall-model cell reaches 1 more along its normal), so the oracle run on a crop of
the INPUTS with margin m = 2 s + 2 around a window reproduces the window exactly after s = 10 steps.  Crops that touch
the inlet / outlet planes or the solid floor / top are flush with them.  >= 8 windows per config.
"""
import numpy as np
import pytest
import torch

import lbm_inputs as I
import paper_2506_21804_b200 as P
from oracle import oracle as O
from parity_util import NP_DTYPE, TOL, field_error

pytestmark = pytest.mark.gpu
S = 10
M = 2 * S + 2
W = 8


def _axis_crop(lo, n, closed):
    """Index arrays (crop indices, position of the window inside the crop) for a window [lo, lo+W) on an axis of size n.
    closed: the axis is bounded by special planes (inlet/outlet or solid layers): clip the crop flush instead of wrapping."""
    a, b = lo - M, lo + W + M
    if closed:
        a, b = max(a, 0), min(b, n)
        idx = np.arange(a, b)
    else:
        if b - a >= n:
            idx = np.arange(n)
            a = 0
        else:
            idx = np.arange(a, b) % n
    return idx, lo - a


def _check_windows(cfg, dtype, windows, closed_axes, steps=S, u_scale=0.0, vm=None, u_body=None):
    """u_scale: velocity scale of the whole field (R12 normalises by the field's maximum; a window of fluid at rest has none)"""
    nz, ny, nx = cfg["shape"]
    Q = cfg["Q"]
    npdt = NP_DTYPE[dtype]
    # the same populations for both sides: the oracle's equilibrium rounded to the run's dtype
    f = O.init_equilibrium(Q, cfg["rho"], cfg["u"]).astype(npdt)
    d = None if cfg["d"] is None else cfg["d"].astype(npdt)
    par = P.LbmParams(**cfg["params"])
    with P.LBM(Q, nx, ny, nz, dtype) as sim:
        sim.set_fields(f, d, cfg["flags"])                  # host pointers, library defaults = bench configuration
        if u_body is not None:
            u_body = u_body.astype(npdt)
            sim.set_body_velocity(u_body)
        if vm is not None:
            sim.set_inflow(vm["u_mean"].astype(npdt))
            sim.set_vortices(vm["pos"], vm["sign"], vm["sigma_v"], vm["intensity"])
        sim.step(steps, par)
        out = torch.empty((Q, nz, ny, nx), dtype=torch.float32 if dtype == "f32" else torch.float64, device="cuda")
        sim.get_populations(out)
        rho = torch.empty((nz, ny, nx), dtype=out.dtype, device="cuda")
        u = torch.empty((3, nz, ny, nx), dtype=out.dtype, device="cuda")
        sim.moments(rho, u)
        sim.synchronize()
    fields = None
    if vm is not None:
        # the inflow of every step on the WHOLE plane (it depends on all INLET cells and all seeds), from the oracle's Eq. 18-21;
        # a crop then runs with that step's field as its "mean profile" and no vortices
        mask = ((cfg["flags"][:, :, 0] & 15) == I.INLET).astype(np.uint8)
        um = vm["u_mean"].astype(npdt).astype(np.float64)
        fields, prev = [], um
        for _ in range(steps):
            prev = O.vm_inflow(mask, um, prev, vm["pos"], vm["sign"], vm["sigma_v"], vm["intensity"])
            fields.append(prev)
    worst = 0.0
    for (z0, y0, x0) in windows:
        iz, wz = _axis_crop(z0, nz, closed_axes[0])
        iy, wy = _axis_crop(y0, ny, closed_axes[1])
        ix, wx = _axis_crop(x0, nx, closed_axes[2])
        sel = np.ix_(iz, iy, ix)
        fc = np.ascontiguousarray(f[(slice(None),) + sel]).astype(np.float64)
        dc = None if d is None else np.ascontiguousarray(d[sel]).astype(np.float64)
        flc = None if cfg["flags"] is None else np.ascontiguousarray(cfg["flags"][sel])
        par_c = dict(cfg["params"])
        if par_c.get("fringe_len", 0) > 0 and ix[-1] != nx - 1:
            # the fringe zone is measured from the last plane: a crop that does not end there must not reach into it
            assert ix.max() + 1 < nx - 1 - par_c["fringe_len"], "window crop cuts the fringe zone"
            par_c["fringe_len"] = 0
        if fields is None:
            ubc = None if u_body is None else np.ascontiguousarray(u_body[(slice(None),) + sel]).astype(np.float64)
            ref = O.step(fc, d=dc, flags=flc, nsteps=steps, nthreads=min(O.max_threads(), 8), u_body=ubc, **par_c)
        else:
            ref = fc
            for fld in fields:
                uc = np.ascontiguousarray(fld[:, iz][:, :, iy])
                ref, _ = O.step_vm(ref, uc, uc, np.zeros((0, 2)), np.zeros(0), 1.0, 0.0, d=dc, flags=flc, nsteps=1,
                                   nthreads=min(O.max_threads(), 8), **par_c)
        inner = (slice(None), slice(wz, wz + W), slice(wy, wy + W), slice(wx, wx + W))
        refw = ref[inner]
        gz, gy, gx = iz[wz:wz + W], iy[wy:wy + W], ix[wx:wx + W]
        gsel = np.ix_(gz, gy, gx)
        tz, ty, tx = (torch.as_tensor(v, device="cuda") for v in (gz, gy, gx))
        gotw = out[:, tz][:, :, ty][:, :, :, tx].cpu().numpy().astype(np.float64)
        mask = None
        if flc is not None:
            mask = ~I.is_wall(cfg["flags"][gsel])
            if not mask.any():
                continue
            solid = ~mask
            assert np.array_equal(gotw[:, solid], f[(slice(None),) + gsel][:, solid].astype(np.float64))
        err = field_error(gotw, refw, mask)
        rr, ru = O.moments(ref)
        rw = rr[inner[1:]]
        uw = ru[(slice(None),) + inner[1:]]
        e_rho = field_error(rho[tz][:, ty][:, :, tx].cpu().numpy(), rw, mask)
        e_u = field_error(u[:, tz][:, :, ty][:, :, :, tx].cpu().numpy(), uw, mask)
        if u_scale > 0.0:
            e_u *= np.abs(uw if mask is None else uw[..., mask]).max() / max(np.abs(uw if mask is None else uw[..., mask]).max(), u_scale)
        worst = max(worst, err, e_rho, e_u)
        assert err <= TOL[dtype], ("populations", (z0, y0, x0), err)
        assert e_rho <= TOL[dtype], ("rho", (z0, y0, x0), e_rho)
        assert e_u <= TOL[dtype], ("u", (z0, y0, x0), e_u)
    return worst


def test_config2_full_size_windows():
    cfg = I.make_config(2)
    rng = np.random.default_rng(2)
    wins = [(0, 0, 0), (248, 248, 248), (124, 0, 252)] + [tuple(int(v) for v in rng.integers(0, 248, 3)) for _ in range(5)]
    _check_windows(cfg, "f32", wins, (False, False, False))


def test_config3_full_size_windows():
    cfg = I.make_config(3)
    nz, ny, nx = cfg["shape"]
    d, fl = cfg["d"], cfg["flags"]
    # floor + inlet, floor + outlet, top, a building, a tree, wall-model floor mid-domain, bulk, y-wrap
    bz, by, bx = np.argwhere((d == 1.0) & (fl == 0))[len(np.argwhere((d == 1.0) & (fl == 0))) // 2]
    tz, ty, tx = np.argwhere((d > 0) & (d < 1))[len(np.argwhere((d > 0) & (d < 1))) // 3]
    wins = [(1, 10, 0), (1, 100, nx - W), (nz - 1 - W, 50, 200), (max(int(bz) - 3, 1), int(by), min(int(bx), nx - W)),
            (max(int(tz) - 3, 1), int(ty), min(int(tx), nx - W)), (1, 60, 150), (60, 90, 190), (30, ny - 4, 100),
            (40, 0, 0), (40, 20, nx - W)]
    _check_windows(cfg, "f32", wins, (True, False, True))


def test_config3_full_size_windows_fp64():
    cfg = I.make_config(3)
    nz, ny, nx = cfg["shape"]
    wins = [(1, 10, 0), (1, 100, nx - W), (nz - 1 - W, 50, 200), (1, 60, 150), (60, 90, 190), (30, ny - 4, 100),
            (20, 40, 120), (5, 130, 250)]
    _check_windows(cfg, "f64", wins, (True, False, True))


def test_config4_full_size_windows():
    cfg = I.make_config(4)
    fl = cfg["flags"]
    rng = np.random.default_rng(4)
    solid = np.argwhere(fl == I.SOLID)
    wins = [tuple(int(v) for v in solid[k] - 2) for k in rng.integers(0, len(solid), 5)]      # windows cutting spheres
    wins = [tuple(min(max(v, 0), 512 - W) for v in w) for w in wins]
    wins += [(0, 0, 0), (504, 504, 504), (250, 0, 504)]
    _check_windows(cfg, "f32", wins, (False, False, False))


# HRR form at the sizes bench.py's *_hrr workloads time.  The FD strain reads u^ of the neighbours, whose pull reaches
# one cell further: information moves <= 2 cells per step (3 along a wall-model normal), so 6 steps stay inside the margin 22.
HRR = dict(collision=1, sigma=0.7)      # = bench.py's HRR workloads


def test_config3_hrr_full_size_windows():
    cfg = I.make_config(3)
    cfg["params"] = dict(cfg["params"], **HRR)
    nz, ny, nx = cfg["shape"]
    wins = [(1, 10, 0), (1, 100, nx - W), (nz - 1 - W, 50, 200), (1, 60, 150), (60, 90, 190), (30, ny - 4, 100),
            (20, 40, 120), (5, 130, 250)]
    _check_windows(cfg, "f32", wins, (True, False, True), steps=6)


def test_config4_hrr_full_size_windows():
    cfg = I.make_config(4)
    cfg["params"] = dict(cfg["params"], **HRR)
    fl = cfg["flags"]
    rng = np.random.default_rng(44)
    solid = np.argwhere(fl == I.SOLID)
    wins = [tuple(int(v) for v in solid[k] - 2) for k in rng.integers(0, len(solid), 5)]
    wins = [tuple(min(max(v, 0), 512 - W) for v in w) for w in wins]
    wins += [(0, 0, 0), (504, 504, 504), (250, 0, 504)]
    _check_windows(cfg, "f32", wins, (False, False, False), steps=6)


def test_config3_vm_inlet_full_size_windows():
    """bench.py config3_urban_channel_384x192x128_f32_vm: Vortex Method inlet (256 seeds), windows on and behind the inflow plane"""
    cfg = I.make_config(3)
    nz, ny, nx = cfg["shape"]
    vm = I.vm_inlet(cfg["shape"], 1303, n_vortices=256, sigma_v=6.0, intensity=0.15)
    wins = [(1, 10, 0), (60, 100, 0), (nz - 1 - W, 50, 0), (30, ny - 4, 0), (90, 0, 0), (40, 150, 6), (1, 60, 150), (60, 90, 190)]
    _check_windows(cfg, "f32", wins, (True, False, True), vm=vm)


def test_paper_boundary_set_full_size_windows():
    """bench.py paperbc_urban_channel_384x192x128_f32_vm: VM inlet, pressure outlet + fringe zone, slip lateral walls and top,
    wall-modelled floor; windows at the slip walls / edges, in the fringe zone, on the inflow and outflow planes"""
    cfg = I.make_config(7, shape=(128, 192, 384))
    nz, ny, nx = cfg["shape"]
    vm = I.vm_inlet(cfg["shape"], 1307, n_vortices=256, sigma_v=6.0, intensity=0.15)
    wins = [(1, 1, 0), (nz - 1 - W, ny - 1 - W, 0), (60, 1, nx - W), (nz - 1 - W, 90, nx - W), (1, ny - 1 - W, 200), (nz - 1 - W, 1, 150),
            (40, 100, nx - 20), (60, 90, 190)]
    _check_windows(cfg, "f32", wins, (True, True, True), vm=vm)


def test_moving_bodies_full_size_windows():
    """bench.py config3_urban_channel_384x192x128_f32_body / _hrr_body: the trees of config 3 carry a solid velocity field
    (lbm_inputs.body_velocity, same seed as bench.py); windows centred on tree cells (0 < d < 1)"""
    cfg = I.make_config(3)
    nz, ny, nx = cfg["shape"]
    ub = I.body_velocity(cfg, 1403, amp=0.02)
    trees = np.argwhere((cfg["d"] > 0) & (cfg["d"] < 1))
    assert len(trees) > 100000 and np.abs(ub[:, cfg["d"] == 1.0]).max() == 0.0
    wins = []
    for k in range(1, 9):
        z, y, x = trees[k * len(trees) // 9]
        wins.append((int(np.clip(z - W // 2, 1, nz - 1 - W)), int(y - W // 2) % ny, int(np.clip(x - W // 2, 0, nx - W))))
    _check_windows(cfg, "f32", wins, (True, False, True), u_body=ub)
    cfg["params"] = dict(cfg["params"], collision=1, sigma=0.7)
    _check_windows(cfg, "f32", wins[::2], (True, False, True), steps=6, u_body=ub)


def test_wall_model_on_building_faces_full_size_windows():
    """bench.py paperbc_wmfaces_urban_channel_384x192x128_f32_*: config 8 (the paper's boundary set + wall-model cells on the roofs
    and the four side faces of the buildings); one window around a wall-model cell of every orientation the geometry has"""
    cfg = I.make_config(8, shape=(128, 192, 384))
    nz, ny, nx = cfg["shape"]
    fl = cfg["flags"]
    wins = []
    for code in (0, 1, 2, 3, 4):
        idx = np.argwhere((fl == (I.WALLMODEL | (code << 4))) & (np.arange(nz)[:, None, None] > 1))
        assert len(idx) > 1000
        for k in (len(idx) // 3, 2 * len(idx) // 3):
            z, y, x = idx[k]
            wins.append((int(np.clip(z - W // 2, 1, nz - 1 - W)), int(np.clip(y - W // 2, 1, ny - 1 - W)), int(np.clip(x - W // 2, 0, nx - W))))
    _check_windows(cfg, "f32", wins, (True, True, True))
    cfg["params"] = dict(cfg["params"], collision=1, sigma=0.7)
    _check_windows(cfg, "f32", wins[::2], (True, True, True), steps=6)


def test_cavity_full_size_windows():
    """lid-driven cavity 512^3 (bench.py cavity_512_f32: three launches per step, lid slices on the MW kernel variant):
    windows at the lid's corners and edges, under the lid, at the floor and in the bulk; the walls close every axis"""
    cfg = I.make_config(6)
    n = 512
    wins = [(n - 1 - W, 1, 1), (n - 1 - W, n - 1 - W, n - 1 - W), (n - 1 - W, 250, 1), (n - 1 - W, 1, 300), (n - 1 - W, 200, 200),
            (1, 1, 1), (1, 300, n - 1 - W), (250, 250, 250), (n - 2 - W, 100, n - 1 - W)]
    _check_windows(cfg, "f32", wins, (True, True, True), u_scale=0.05)          # the lid speed


# ---- T2: invariants after the configs' full step counts ------------------------------------------
def _full_run(number, dtype, shape=None):
    cfg = I.make_config(number, shape=shape)
    nz, ny, nx = cfg["shape"]
    npdt = NP_DTYPE[dtype]
    par = P.LbmParams(**cfg["params"])
    with P.LBM(cfg["Q"], nx, ny, nz, dtype) as sim:
        sim.set_geometry(None if cfg["d"] is None else cfg["d"].astype(npdt), cfg["flags"])
        sim.init_equilibrium(cfg["rho"].astype(npdt), cfg["u"].astype(npdt))
        t0 = sim.totals()
        sim.step(cfg["steps"], par)
        t1 = sim.totals()
        u = torch.empty((3, nz, ny, nx), dtype=torch.float32 if dtype == "f32" else torch.float64, device="cuda")
        sim.moments(None, u)
        sim.synchronize()
        umax = float(u.abs().max())
    return cfg, np.array(t0), np.array(t1), umax


def test_config2_full_run_invariants():
    cfg, t0, t1, umax = _full_run(2, "f32")
    assert np.isfinite(t1).all()
    assert abs(t1[0] / t0[0] - 1.0) < 2e-6              # periodic box: mass conserved (unbiased fp32 rounding only)
    assert np.abs(t1[1:4] - t0[1:4]).max() < 2e-6 * t0[0]
    assert t1[4] < t0[4] and umax < 0.3                 # energy decays, velocity bounded


def test_config3_full_run_invariants():
    cfg, t0, t1, umax = _full_run(3, "f32")
    assert np.isfinite(t1).all() and umax < 0.4
    assert abs(t1[0] / t0[0] - 1.0) < 0.02              # open boundaries: density level may drift (DESIGN.md / SURVEY 7-9)


def test_config4_full_run_invariants():
    cfg, t0, t1, umax = _full_run(4, "f32")
    assert np.isfinite(t1).all() and umax < 0.4
    assert abs(t1[0] / t0[0] - 1.0) < 2e-6              # closed (periodic + bounce-back): mass conserved

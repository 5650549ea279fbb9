"""Halo exchange of a slab decomposition in z: several sub-domain contexts on ONE GPU,
exchanging their halos by device copies (paper_2506_21804_b200.slab.LocalGroup), must reproduce the populations of the undivided
lattice BIT FOR BIT -- the interior cells see exactly the same values through the ghost slices as through the periodic wrap or the
neighbouring slices of the single lattice.  Configs 2 (periodic), 3 (closed channel: inlet, outlet, wall model, porosity), 4
(D3Q27, spheres), the lid-driven cavity (the paper's scaling benchmark) and the paper's boundary set; both collision forms."""
import numpy as np
import pytest
import torch

import lbm_inputs as I
import paper_2506_21804_b200 as P
from oracle import oracle as O
from paper_2506_21804_b200 import slab as S
from parity_util import NP_DTYPE, TOL, field_error, nonsolid, oracle_inputs, run_oracle

pytestmark = pytest.mark.gpu
HRR = dict(collision=1, sigma=0.7)
LAG = dict(collision=2, sigma=0.7)      # the HRR form in one pass (G41): the u^ exchange carries the previous level's boundary slices


def _single(cfg, f, d, dtype, chunks):
    nz, ny, nx = cfg["shape"]
    par = P.LbmParams(**cfg["params"])
    with P.LBM(cfg["Q"], nx, ny, nz, dtype) as sim:
        sim.set_fields(f, d, cfg["flags"])
        for n in chunks:
            sim.step(n, par)
        out = np.empty_like(f)
        rho = np.empty(f.shape[1:], dtype=f.dtype)
        u = np.empty((3,) + f.shape[1:], dtype=f.dtype)
        sim.moments(rho, u)
        tot = np.array(sim.totals())
        sim.get_populations(out)
    return out, rho, u, tot


def _decomposed(cfg, f, d, dtype, chunks, world, read_between=False):
    nz, ny, nx = cfg["shape"]
    par = P.LbmParams(**cfg["params"])
    grp = S.LocalGroup(cfg["Q"], nx, ny, nz, dtype, world, S.z_is_closed(cfg["flags"]))
    try:
        grp.set_fields(f, d, cfg["flags"])
        out = np.empty_like(f)
        for n in chunks:
            grp.step(n, par)
            if read_between:
                grp.get_populations(out)                       # materialises S_t in every sub-domain; the run goes on from it
        rho = np.empty(f.shape[1:], dtype=f.dtype)
        u = np.empty((3,) + f.shape[1:], dtype=f.dtype)
        grp.moments(rho, u)
        tot = grp.totals()
        grp.get_populations(out)
        launches = [p.sim.query("launches") for p in grp.parts]
    finally:
        grp.close()
    return out, rho, u, tot, launches


CASES = {
    # name: (config, shape (nz, ny, nx), extra params, dtype)
    "periodic_les_bgk_f32": (2, (30, 16, 64), {}, "f32"),
    "periodic_les_hrr_f64": (2, (30, 16, 64), HRR, "f64"),
    "urban_channel_bgk_f32": (3, (41, 24, 96), {}, "f32"),
    "urban_channel_hrr_f32": (3, (41, 24, 96), HRR, "f32"),
    "urban_channel_bgk_f64": (3, (41, 24, 96), {}, "f64"),
    "spheres_d3q27_bgk_f32": (4, (32, 24, 64), {}, "f32"),
    "spheres_d3q27_hrr_f32": (4, (32, 24, 64), HRR, "f32"),
    "cavity_bgk_f32": (6, (33, 24, 64), {}, "f32"),
    "cavity_hrr_f32": (6, (33, 24, 64), HRR, "f32"),
    "periodic_les_lag_f64": (2, (30, 16, 64), LAG, "f64"),
    "urban_channel_lag_f32": (3, (41, 24, 96), LAG, "f32"),
    "spheres_d3q27_lag_f32": (4, (32, 24, 64), LAG, "f32"),
    "cavity_lag_f32": (6, (33, 24, 64), LAG, "f32"),
    "paper_boundary_set_bgk_f32": (7, (40, 24, 96), {}, "f32"),
    "scalar_rows_bgk_f64": (3, (20, 12, 37), {}, "f64"),           # nx = 37: the one-cell-per-thread kernel
}


@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("case", sorted(CASES))
def test_decomposed_run_equals_the_undivided_lattice_bit_for_bit(case, world):
    number, shape, extra, dtype = CASES[case]
    kw = dict(k_max=6, n_modes=48) if number in (2, 4) else {}
    cfg = I.make_config(number, shape=shape, **kw)
    cfg["params"] = dict(cfg["params"], **extra)
    f, d = oracle_inputs(cfg, dtype)
    chunks = [7, 4]
    a, rho_a, u_a, tot_a = _single(cfg, f, d, dtype, chunks)
    b, rho_b, u_b, tot_b, launches = _decomposed(cfg, f, d, dtype, chunks, world)
    m = nonsolid(cfg)
    assert np.array_equal(a, b)
    keep = np.ones(rho_a.shape, dtype=bool) if m is None else m
    assert np.array_equal(rho_a[keep], rho_b[keep]) and np.array_equal(u_a[:, keep], u_b[:, keep])
    assert np.abs(tot_a - tot_b).max() <= 1e-12 * abs(tot_a[0]) * (1e6 if dtype == "f32" else 1.0)
    # and both are the oracle's result
    ref = run_oracle(cfg, f, d, sum(chunks))
    assert field_error(b, ref, m) <= 2 * TOL[dtype]


def test_state_reads_between_the_steps_do_not_change_the_run():
    cfg = I.make_config(3, shape=(30, 16, 64))
    cfg["params"] = dict(cfg["params"], **HRR)
    f, d = oracle_inputs(cfg, "f64")
    a, *_ = _decomposed(cfg, f, d, "f64", [3, 1, 4], 2)
    b, *_ = _decomposed(cfg, f, d, "f64", [3, 1, 4], 2, read_between=True)
    c, *_ = _single(cfg, f, d, "f64", [8])
    assert np.array_equal(a, c) and np.array_equal(b, c)


def test_face_buffers_host_and_device_and_the_errors():
    cfg = I.make_config(2, shape=(12, 8, 32), k_max=4, n_modes=16)
    f, d = oracle_inputs(cfg, "f32")
    par = P.LbmParams(**cfg["params"])
    with P.LBM(19, 32, 8, 12, "f32") as sim:
        sim.set_fields(f)
        with pytest.raises(P.LbmError):
            sim.set_halo(2, 0)
        with pytest.raises(P.LbmError):
            sim.halo_pack(0, 0, np.empty(5 * 8 * 32, np.float32))      # no ghost slice declared
        sim.set_halo(1, 1)
        assert sim.query("interior_slices") == 10 and sim.query("halo_population_values") == 5 * 8 * 32
        with pytest.raises(P.LbmError):
            sim.step(1, par)                                           # a sub-domain steps through lbm_step_halo
        with pytest.raises(P.LbmError):
            sim.step_halo(par, 1)                                      # stage 0 is due
        sim.step_halo(par, 0)
        with pytest.raises(P.LbmError):
            sim.step_halo(par, 0)
        sim.step_halo(par, 1)
        assert sim.query("steps") == 1
        h = np.empty(5 * 8 * 32, np.float32)
        t = torch.empty(5 * 8 * 32, dtype=torch.float32, device="cuda")
        for side in (0, 1):
            sim.halo_pack(0, side, h)
            sim.halo_pack(0, side, t)
            assert np.array_equal(h, t.cpu().numpy())
        # what was packed: the stored post-collision populations with c_z = -1 (low side) of the first interior slice
        c, w, opp = O.lattice(19)
        ref = O.step(f.astype(np.float64), nsteps=1, **cfg["params"])       # S_1 = stream(F_0): F_0,i(x) = S_1,i(x + c_i)
        down = [i for i in range(19) if c[i][2] == -1]
        sim.halo_pack(0, 0, h)
        got = h.reshape(5, 8, 32)
        for k, i in enumerate(down):
            want = np.roll(ref[i], shift=(-c[i][1], -c[i][0]), axis=(1, 2))[(1 + c[i][2]) % 12]
            assert np.abs(got[k] - want).max() <= 2e-6
        with pytest.raises(P.LbmError):
            sim.halo_pack(1, 0, h)                                     # no u^ field: the HRR form has not run
        with pytest.raises(P.LbmError):
            sim.halo_pack(2, 0, h)
        with pytest.raises(P.LbmError):
            sim.halo_unpack(0, 3, h)


def test_wall_model_cell_sampling_across_a_cut_is_refused():
    cfg = I.make_config(3, shape=(24, 16, 64))
    fl = cfg["flags"].copy()
    dd = cfg["d"].copy()
    z_cut = S.partition(24, 2)[0][1]                                    # first slice of rank 1
    fl[z_cut - 1, 5, 20] = I.WALLMODEL | (4 << 4)                       # normal +z: samples at z_cut, rank 0's ghost slice
    dd[z_cut - 1, 5, 20] = 1.0
    cfg2 = dict(cfg, flags=fl, d=dd)
    f, d = oracle_inputs(cfg2, "f32")
    grp = S.LocalGroup(19, 64, 16, 24, "f32", 2, True)
    try:
        with pytest.raises(P.LbmError) as e:
            grp.set_fields(f, d, fl)
        assert "WALLMODEL" in str(e.value)
    finally:
        grp.close()
    # the same cell one slice lower is fine
    fl2, dd2 = cfg["flags"].copy(), cfg["d"].copy()
    fl2[z_cut - 2, 5, 20] = I.WALLMODEL | (4 << 4)
    dd2[z_cut - 2, 5, 20] = 1.0
    cfg3 = dict(cfg, flags=fl2, d=dd2)
    f, d = oracle_inputs(cfg3, "f32")
    a, *_ = _single(cfg3, f, d, "f32", [5])
    b, *_ = _decomposed(cfg3, f, d, "f32", [5], 2)
    assert np.array_equal(a, b)

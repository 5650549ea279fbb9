"""The tuning knobs of lbm_set_option are schedules, not arithmetic: A/B runs must give the same populations BIT FOR BIT
("serpentine", "pdl", "cuda_graph", "hrr_slab", "block_threads") or, where the knob selects another kernel body for some cells
("wm_prepass", "vector"), agree with the oracle to the parity tolerance on both settings.  Also: the box calls
(lbm_set_populations_box / lbm_get_populations_box) and the queued device-pointer path of lbm_get_inflow."""
import numpy as np
import pytest
import torch

import lbm_inputs as I
import paper_2506_21804_b200 as P
from oracle import oracle as O
from parity_util import NP_DTYPE, TOL, field_error, nonsolid, oracle_inputs, run_oracle

pytestmark = pytest.mark.gpu


def _run(cfg, f, d, dtype, chunks, options, u_wall=None):
    nz, ny, nx = cfg["shape"]
    par = P.LbmParams(**cfg["params"])
    with P.LBM(cfg["Q"], nx, ny, nz, dtype) as sim:
        for k, v in options.items():
            sim.set_option(k, v)
        sim.set_fields(f, d, cfg["flags"])
        for n in chunks:
            sim.step(n, par)
        out = np.empty_like(f)
        sim.get_populations(out)
        return out, sim.query("graph_launches"), sim.query("launches")


CASES = {
    "urban_bgk": (3, (24, 32, 96), {}),
    "urban_hrr": (3, (24, 32, 96), dict(collision=1, sigma=0.7)),
    "cavity_bgk": (6, (24, 32, 64), {}),                       # moving lid: three launches per step
    "cavity_hrr": (6, (24, 32, 64), dict(collision=1, sigma=0.7)),
    "paperbc_bgk": (7, (24, 32, 96), {}),
}


@pytest.mark.parametrize("case", sorted(CASES))
@pytest.mark.parametrize("key,values", [("serpentine", (1, 0)), ("pdl", (2, 1, 0)), ("cuda_graph", (1, 0)), ("block_threads", (64, 128, 256))])
def test_schedule_knobs_are_bit_identical(case, key, values):
    number, shape, extra = CASES[case]
    cfg = I.make_config(number, shape=shape)
    cfg["params"] = dict(cfg["params"], **extra)
    f, d = oracle_inputs(cfg, "f32")
    outs = []
    for v in values:
        # 1 collide-only step + 8 graph steps + 2 plain steps, then an odd chunk that starts in the POST phase
        out, graphs, launches = _run(cfg, f, d, "f32", [11, 9], {key: v})
        outs.append(out)
        if key == "cuda_graph":
            assert (graphs > 0) == (v == 1)
    for o in outs[1:]:
        assert np.array_equal(outs[0], o), (case, key)
    ref = run_oracle(cfg, f, d, 20)
    err = field_error(outs[0], ref, nonsolid(cfg))
    assert err <= 2 * TOL["f32"]                               # 20 steps


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("coll", [0, 1])
def test_wall_model_prepass_and_in_place_solve_agree(dtype, coll):
    """wm_prepass 1 (u^B from the compact-list pre-pass, WM cells in the vector path) vs 0 (Spalding solves in the list blocks)"""
    cfg = I.make_config(8, shape=(32, 48, 96))                 # wall-model cells on the floor and on building faces
    cfg["params"] = dict(cfg["params"], collision=coll, sigma=0.7)
    f, d = oracle_inputs(cfg, dtype)
    ref = run_oracle(cfg, f, d, 10)
    m = nonsolid(cfg)
    outs = []
    for v in (1, 0):
        out, _, _ = _run(cfg, f, d, dtype, [10], {"wm_prepass": v})
        assert field_error(out, ref, m) <= TOL[dtype], (v,)
        outs.append(out)
    assert field_error(outs[0], outs[1], m) <= (1e-13 if dtype == "f64" else 2e-6)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("Q,coll", [(19, 0), (19, 1), (27, 0)])
def test_slip_plane_codes_and_the_general_specular_rule_agree(Q, coll, dtype):
    """slip_planes 1 (cells next to a plane slip wall pull the reflected populations in the vector path) vs 0 (every slip-adjacent
    cell in the list blocks, general rule slip_pull): config 7 (slip lateral walls and top) from a NON-EQUILIBRIUM state, so that a
    wrong slot or source row cannot hide behind symmetry"""
    cfg = I.make_config(7, shape=(24, 32, 96))
    cfg["Q"] = Q
    cfg["params"] = dict(cfg["params"], collision=coll, sigma=0.7)
    f, d = oracle_inputs(cfg, "f64")
    rng = np.random.Generator(np.random.PCG64(77 + Q + coll))
    f = (f * (1.0 + 0.02 * rng.uniform(-1.0, 1.0, size=f.shape))).astype(NP_DTYPE[dtype])
    d = d.astype(NP_DTYPE[dtype])
    ref = run_oracle(cfg, f, d, 10)
    m = nonsolid(cfg)
    nz, ny, nx = cfg["shape"]
    outs, coded = [], []
    for v in (1, 0):
        with P.LBM(Q, nx, ny, nz, dtype) as sim:
            sim.set_option("slip_planes", v)
            sim.set_fields(f, d, cfg["flags"])
            coded.append((sim.query("slip_plane_cells"), sim.query("list_cells")))
            sim.step(10, P.LbmParams(**cfg["params"]))
            out = np.empty_like(f)
            sim.get_populations(out)
        assert field_error(out, ref, m) <= TOL[dtype], (v,)
        outs.append(out)
    assert coded[0][0] > 2000 and coded[1][0] == 0 and coded[0][1] < coded[1][1] // 4      # the list shrank to the edges and corners
    assert field_error(outs[0], outs[1], m) <= (1e-13 if dtype == "f64" else 2e-6)


def test_graph_is_recaptured_when_parameters_or_fields_change():
    cfg = I.make_config(3, shape=(24, 32, 96))
    f, d = oracle_inputs(cfg, "f64")
    nz, ny, nx = cfg["shape"]
    p1 = dict(cfg["params"])
    p2 = dict(cfg["params"], tau0=0.56, cs_smago=0.15)
    d2 = np.where(d > 0, 0.5 * d, d)
    with P.LBM(19, nx, ny, nz, "f64") as sim:
        sim.set_option("cuda_graph", 1)
        sim.set_fields(f, d, cfg["flags"])
        sim.step(17, P.LbmParams(**p1))
        g1 = sim.query("graph_launches")
        sim.step(16, P.LbmParams(**p2))                          # other parameters: the captured graphs must not be replayed as they are
        sim.set_porosity(d2)                                     # same pointer, new contents: graphs stay valid
        sim.step(16, P.LbmParams(**p2))
        out = np.empty_like(f)
        sim.get_populations(out)
        assert g1 == 2 and sim.query("graph_launches") == 6
    ref = O.step(f, d=d, flags=cfg["flags"], nsteps=17, **p1)
    ref = O.step(ref, d=d, flags=cfg["flags"], nsteps=16, **p2)
    ref = O.step(ref, d=d2, flags=cfg["flags"], nsteps=16, **p2)
    assert field_error(out, ref, nonsolid(cfg)) <= 5e-12         # 49 steps


# ---- box calls ---------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_state_set_box_by_box_equals_set_fields(dtype):
    cfg = I.make_config(3, shape=(20, 24, 64))
    f, d = oracle_inputs(cfg, dtype)
    nz, ny, nx = cfg["shape"]
    par = P.LbmParams(**cfg["params"])
    a, _, _ = _run(cfg, f, d, dtype, [10], {})
    with P.LBM(19, nx, ny, nz, dtype) as sim:
        sim.set_geometry(d, cfg["flags"])
        # ragged boxes: 3 x 2 x 3 pieces with uneven cuts, host and device pointers alternating
        xs, ys, zs = [0, 7, 40, nx], [0, 13, ny], [0, 1, 9, nz]
        k = 0
        for zi in range(3):
            for yi in range(2):
                for xi in range(3):
                    box = np.ascontiguousarray(f[:, zs[zi]:zs[zi + 1], ys[yi]:ys[yi + 1], xs[xi]:xs[xi + 1]])
                    src = torch.from_numpy(box).cuda() if (k & 1) else box
                    sim.set_populations_box((xs[xi], ys[yi], zs[zi]), (xs[xi + 1] - xs[xi], ys[yi + 1] - ys[yi], zs[zi + 1] - zs[zi]), src)
                    k += 1
        back = np.empty_like(f)
        sim.get_populations(back)
        assert np.array_equal(back, f)
        sim.step(10, par)
        out = np.empty_like(f)
        sim.get_populations(out)
        assert np.array_equal(out, a)
        # a box of the stepped state (POST phase -> materialised), wall cells included, against the full getter
        sim.step(3, par)
        full = np.empty_like(f)
        box = torch.empty((19, 5, 9, 17), dtype=torch.float32 if dtype == "f32" else torch.float64, device="cuda")
        sim.get_populations_box((40, 11, 0), (17, 9, 5), box)
        sim.get_populations(full)
        assert np.array_equal(box.cpu().numpy(), full[:, 0:5, 11:20, 40:57])
        # overwrite a box in mid-run: only that box changes, wall cells in it take the new values too
        patch = np.ascontiguousarray(f[:, 0:5, 11:20, 40:57])
        sim.set_populations_box((40, 11, 0), (17, 9, 5), patch)
        now = np.empty_like(f)
        sim.get_populations(now)
        want = full.copy()
        want[:, 0:5, 11:20, 40:57] = patch
        assert np.array_equal(now, want) and sim.query("steps") == 13
        sim.step(2, par)
        sim.get_populations(now)
        ref = O.step(want.astype(np.float64), d=d.astype(np.float64), flags=cfg["flags"], nsteps=2, **cfg["params"])
        assert field_error(now, ref, nonsolid(cfg)) <= TOL[dtype]
        for bad in [((0, 0, 0), (0, 1, 1)), ((60, 0, 0), (5, 1, 1)), ((0, -1, 0), (1, 1, 1))]:
            with pytest.raises(P.LbmError):
                sim.set_populations_box(bad[0], bad[1], patch)
            with pytest.raises(P.LbmError):
                sim.get_populations_box(bad[0], bad[1], patch)


# ---- lbm_get_inflow, fp32, DEVICE output pointer, steps queued behind it -----------------
def test_get_inflow_fp32_device_pointer_with_queued_steps():
    cfg = I.make_config(3, shape=(24, 32, 64))
    vm = I.vm_inlet(cfg["shape"], 1300, n_vortices=40, sigma_v=3.0, intensity=0.2)
    f, d = oracle_inputs(cfg, "f32")
    nz, ny, nx = cfg["shape"]
    par = P.LbmParams(**cfg["params"])

    def run(device):
        with P.LBM(19, nx, ny, nz, "f32") as sim:
            sim.set_fields(f, d, cfg["flags"])
            sim.set_inflow(vm["u_mean"].astype(np.float32))
            sim.set_vortices(vm["pos"], vm["sign"], vm["sigma_v"], vm["intensity"])
            got = []
            for _ in range(6):
                sim.step(2, par)
                if device:
                    u = torch.empty((3, nz, ny), dtype=torch.float32, device="cuda")
                    sim.get_inflow(u)                          # returns without synchronising; the next steps queue behind it
                else:
                    u = np.empty((3, nz, ny), dtype=np.float32)
                    sim.get_inflow(u)                          # host buffer: synchronises
                got.append(u)
            out = np.empty_like(f)
            sim.get_populations(out)
            return [g.cpu().numpy() if device else g for g in got], out

    ga, fa = run(True)
    gb, fb = run(False)
    for a, b in zip(ga, gb):
        assert np.array_equal(a, b)
    assert np.array_equal(fa, fb)
    um = vm["u_mean"].astype(np.float32).astype(np.float64)
    ref, uref = O.step_vm(f.astype(np.float64), um, um, vm["pos"], vm["sign"], vm["sigma_v"], vm["intensity"],
                          d=d.astype(np.float64), flags=cfg["flags"], nsteps=12, nthreads=8, **cfg["params"])
    inl = (cfg["flags"][:, :, 0] & 15) == I.INLET
    assert field_error(ga[-1][:, inl], uref[:, inl]) <= TOL["f32"]
    assert field_error(fa, ref, nonsolid(cfg)) <= 2 * TOL["f32"]

"""T1: GPU-vs-oracle parity through the C ABI (element by element, same seeded inputs, 10 steps) and the
ABI's behaviour (round trip, phases, host pointers, errors).  Tolerances: north_star / DESIGN.md R12 --
fp64 <= 1e-12, fp32 <= 2e-5 (against the fp64 oracle), SOLID cells bit-exact."""
import numpy as np
import pytest
import torch

import lbm_inputs as I
import paper_2506_21804_b200 as P
from oracle import oracle as O
from parity_util import NP_DTYPE, TOL, field_error, nonsolid, oracle_inputs, run_oracle

pytestmark = pytest.mark.gpu
TORCH_DTYPE = {"f32": torch.float32, "f64": torch.float64}


def gpu_run(cfg, f, d, nsteps, dtype, host=False, split=None, block_threads=None, vector=None):
    """Run nsteps through the C ABI; returns (populations, rho, u, totals) as numpy."""
    nz, ny, nx = cfg["shape"]
    Q = cfg["Q"]
    par = P.LbmParams(**cfg["params"])
    with P.LBM(Q, nx, ny, nz, dtype) as sim:
        if block_threads:
            sim.set_option("block_threads", block_threads)
        if vector is not None:
            sim.set_option("vector", vector)
        if host:
            sim.set_fields(f, d, cfg["flags"])
        else:
            tf = torch.from_numpy(f).cuda()
            td = None if d is None else torch.from_numpy(d).cuda()
            tfl = None if cfg["flags"] is None else torch.from_numpy(cfg["flags"]).cuda()
            sim.set_fields(tf, td, tfl)
        for n in (split or [nsteps]):
            sim.step(n, par)
        if host:
            rho = np.empty((nz, ny, nx), dtype=NP_DTYPE[dtype])
            u = np.empty((3, nz, ny, nx), dtype=NP_DTYPE[dtype])
            out = np.empty_like(f)
            sim.moments(rho, u)
            tot = sim.totals()
            sim.get_populations(out)
            return out, rho, u, np.array(tot)
        rho = torch.empty((nz, ny, nx), dtype=TORCH_DTYPE[dtype], device="cuda")
        u = torch.empty((3, nz, ny, nx), dtype=TORCH_DTYPE[dtype], device="cuda")
        out = torch.empty((Q, nz, ny, nx), dtype=TORCH_DTYPE[dtype], device="cuda")
        sim.moments(rho, u)          # moments are taken in the POST phase (pull inside the kernel) ...
        tot = sim.totals()
        sim.get_populations(out)     # ... and the populations after materialising S_t
        sim.synchronize()
        return out.cpu().numpy(), rho.cpu().numpy(), u.cpu().numpy(), np.array(tot)


def check_parity(cfg, dtype, nsteps=10, **kw):
    f, d = oracle_inputs(cfg, dtype)
    ref = run_oracle(cfg, f, d, nsteps)
    got, rho, u, tot = gpu_run(cfg, f, d, nsteps, dtype, **kw)
    mask = nonsolid(cfg)
    tol = TOL[dtype]
    assert np.isfinite(got).all()
    e_f = field_error(got, ref, mask)
    rr, ru = O.moments(ref)
    e_rho = field_error(rho, rr, mask)
    e_u = field_error(u, ru, mask)
    assert e_f <= tol, ("populations", e_f)
    assert e_rho <= tol, ("rho", e_rho)
    assert e_u <= tol, ("u", e_u)
    if mask is not None:
        solid = ~mask
        assert np.array_equal(got[:, solid], f[:, solid])        # SOLID cells untouched, bit-exact
    # totals: against the oracle's per-cell moments summed pairwise (numpy) at the field tolerance, and against orc_totals, whose
    # plain sequential sum over N cells carries up to N eps / 2 of relative rounding of its own (G40: 128^3 cells of
    # nearly equal momentum: 2.5e-6 absolute on 8.8e4, where the pairwise sum and the GPU's tree agree to 1e-9)
    keep = np.ones(rr.shape, dtype=bool) if mask is None else mask
    px = [(rr * ru[a])[keep].sum() for a in range(3)]
    pair = np.array([rr[keep].sum()] + px + [(0.5 * rr * (ru ** 2).sum(axis=0))[keep].sum()])
    assert np.abs(tot - pair).max() <= max(tol, 1e-12) * abs(pair[0])
    rt = O.totals(ref, cfg["flags"])
    assert np.abs(tot - rt).max() <= max(tol, 1e-12, rr.size * 1.2e-16) * abs(rt[0])
    return e_f, e_rho, e_u


# ---- the configs, at sizes the oracle finishes in seconds (several tiles + ragged tails) ---------
def test_config1_tgv_fp64_full_size():
    cfg = I.make_config(1)
    check_parity(cfg, "f64")


def test_config1_tgv_decay_100_steps_matches_closed_form_and_oracle():
    cfg = I.make_config(1)
    f, d = oracle_inputs(cfg, "f64")
    got, rho, u, tot = gpu_run(cfg, f, d, 100, "f64")
    E0 = O.totals(f)[4]
    nu, k = (0.6 - 0.5) / 3.0, 2 * np.pi / 32
    assert abs(tot[4] / E0 / np.exp(-4 * nu * k * k * 100) - 1.0) <= 0.025        # P7 on the GPU
    ref = run_oracle(cfg, f, d, 100)
    assert field_error(got, ref) <= 1e-11


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_config2_les_periodic(dtype):
    cfg = I.make_config(2, shape=(64, 64, 64), k_max=8, n_modes=128)
    check_parity(cfg, dtype)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_config3_urban_channel(dtype):
    cfg = I.make_config(3, shape=(40, 48, 160))      # nz, ny, nx
    t = cfg["flags"] & 15
    assert (t == I.WALLMODEL).any() and (t == I.INLET).any() and (cfg["d"] > 0).any()
    check_parity(cfg, dtype)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_config4_d3q27_spheres(dtype):
    cfg = I.make_config(4, shape=(48, 48, 48), k_max=6, n_modes=64)
    check_parity(cfg, dtype)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_config5_cubic_urban(dtype):
    cfg = I.make_config(5, shape=(64, 64, 64))
    check_parity(cfg, dtype)


# ---- edge cases ---------------------------------------------------------------------------------
@pytest.mark.parametrize("shape", [(4, 4, 4), (7, 13, 37), (1, 5, 130), (3, 1, 2), (5, 300, 3)])
@pytest.mark.parametrize("Q", [19, 27])
def test_ragged_and_tiny_boxes(shape, Q):
    rng = np.random.default_rng(sum(shape) + Q)
    rho = 1.0 + 0.02 * rng.uniform(-1, 1, size=shape)
    u = 0.04 * rng.uniform(-1, 1, size=(3,) + shape)
    flags = (rng.uniform(size=shape) < 0.12).astype(np.uint8) * I.SOLID
    d = rng.uniform(0, 1, size=shape) * (rng.uniform(size=shape) < 0.3)
    cfg = dict(Q=Q, shape=shape, rho=rho, u=u, d=d, flags=flags, dtype="f64",
               params=dict(tau0=0.52, cs_smago=0.11, use_hlbm=1))
    check_parity(cfg, "f64")
    check_parity(cfg, "f32")


def test_all_solid_and_no_flags():
    shape = (6, 6, 6)
    rng = np.random.default_rng(0)
    cfg = dict(Q=19, shape=shape, rho=np.ones(shape), u=0.01 * rng.uniform(-1, 1, size=(3,) + shape), d=None,
               flags=np.full(shape, I.SOLID, dtype=np.uint8), dtype="f64", params=dict(tau0=0.6))
    f, d = oracle_inputs(cfg, "f64")
    got, rho, u, tot = gpu_run(cfg, f, d, 5, "f64")
    assert np.array_equal(got, f) and np.all(tot == 0.0)


@pytest.mark.parametrize("block_threads", [64, 256])
@pytest.mark.parametrize("vector", [0, 1])
def test_other_block_sizes_and_scalar_kernel(block_threads, vector):
    cfg = I.make_config(3, shape=(24, 20, 72))
    check_parity(cfg, "f32", block_threads=block_threads, vector=vector)
    check_parity(cfg, "f64", block_threads=block_threads, vector=vector)


@pytest.mark.parametrize("nx", [4, 8, 36, 132, 260])
def test_vector_kernel_row_ends(nx):
    """Rows shorter / longer than a warp of vectors, and not a multiple of the block width."""
    shape = (5, 6, nx)
    rng = np.random.default_rng(nx)
    rho = 1.0 + 0.02 * rng.uniform(-1, 1, size=shape)
    u = 0.04 * rng.uniform(-1, 1, size=(3,) + shape)
    flags = (rng.uniform(size=shape) < 0.05).astype(np.uint8) * I.SOLID
    cfg = dict(Q=19, shape=shape, rho=rho, u=u, d=None, flags=flags, dtype="f64", params=dict(tau0=0.55, cs_smago=0.1))
    check_parity(cfg, "f64")
    check_parity(cfg, "f32")
    cfg["flags"] = None
    cfg["Q"] = 27
    check_parity(cfg, "f32")


def test_channel_with_every_wall_normal_and_inlet_components():
    """WALLMODEL cells on all six orientations around a solid block, transverse inlet velocity."""
    nz, ny, nx = 20, 18, 40
    shape = (nz, ny, nx)
    flags = np.zeros(shape, dtype=np.uint8)
    flags[0] = I.SOLID
    flags[nz - 1] = I.SOLID
    flags[1:nz - 1, :, 0] = I.INLET
    flags[1:nz - 1, :, nx - 1] = I.OUTLET
    flags[6:12, 6:12, 14:22] = I.SOLID
    d = np.zeros(shape)
    def wm(sel, code):
        flags[sel] = I.WALLMODEL | (code << 4)
        d[sel] = 1.0
    wm((slice(6, 12), slice(6, 12), 22), 0)     # +x face
    wm((slice(6, 12), slice(6, 12), 13), 1)     # -x face
    wm((slice(6, 12), 12, slice(14, 22)), 2)    # +y
    wm((slice(6, 12), 5, slice(14, 22)), 3)     # -y
    wm((12, slice(6, 12), slice(14, 22)), 4)    # +z
    wm((5, slice(6, 12), slice(14, 22)), 5)     # -z
    wm((1, slice(None), slice(1, nx - 1)), 4)   # floor
    rho = np.ones(shape)
    u = np.zeros((3,) + shape)
    u[0][(flags & 15) != I.SOLID] = 0.04
    rng = np.random.default_rng(3)
    u[1] += 0.01 * rng.uniform(-1, 1, size=shape)
    u[2] += 0.01 * rng.uniform(-1, 1, size=shape)
    cfg = dict(Q=19, shape=shape, rho=rho, u=u, d=d, flags=flags, dtype="f64",
               params=dict(tau0=0.5 + 3e-4, cs_smago=0.1, use_hlbm=1, u_in=(0.04, 0.003, -0.002), wm_enable=1))
    check_parity(cfg, "f64")
    check_parity(cfg, "f32")
    cfg["params"]["wm_enable"] = 0
    check_parity(cfg, "f64")


# ---- ABI behaviour ------------------------------------------------------------------------------
def test_roundtrip_is_bit_exact_and_phase_independent():
    cfg = I.make_config(3, shape=(16, 12, 40))
    for dtype in ("f32", "f64"):
        f, d = oracle_inputs(cfg, dtype)
        got, rho, u, tot = gpu_run(cfg, f, d, 0, dtype)
        assert np.array_equal(got, f)
        rr, ru = O.moments(f.astype(np.float64))
        assert field_error(rho, rr) <= (1e-6 if dtype == "f32" else 2e-15)
        # splitting the run, or reading the state in between, changes nothing (bit-identical)
        a = gpu_run(cfg, f, d, 10, dtype)
        b = gpu_run(cfg, f, d, 10, dtype, split=[1, 2, 7])
        for x, y in zip(a[:3], b[:3]):
            assert np.array_equal(x, y)
        assert np.allclose(a[3], b[3], rtol=1e-13, atol=0)      # totals: atomic accumulation order is free


def test_reading_state_midrun_does_not_perturb_it():
    cfg = I.make_config(3, shape=(16, 12, 40))
    f, d = oracle_inputs(cfg, "f32")
    nz, ny, nx = cfg["shape"]
    par = P.LbmParams(**cfg["params"])
    outs = []
    for peek in (False, True):
        with P.LBM(19, nx, ny, nz, "f32") as sim:
            sim.set_fields(f, d, cfg["flags"])
            out = np.empty_like(f)
            for _ in range(4):
                sim.step(2, par)
                if peek:
                    sim.get_populations(out)
                    sim.totals()
            sim.get_populations(out)
            assert sim.query("steps") == 8
            outs.append(out.copy())
    assert np.array_equal(outs[0], outs[1])


def test_host_pointers_equal_device_pointers():
    cfg = I.make_config(3, shape=(16, 12, 40))
    f, d = oracle_inputs(cfg, "f32")
    a = gpu_run(cfg, f, d, 6, "f32", host=False)
    b = gpu_run(cfg, f, d, 6, "f32", host=True)
    for x, y in zip(a[:3], b[:3]):
        assert np.array_equal(x, y)
    assert np.allclose(a[3], b[3], rtol=1e-13, atol=0)


@pytest.mark.parametrize("Q", [19, 27])
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_init_equilibrium_matches_oracle(Q, dtype):
    shape = (9, 10, 33)
    rng = np.random.default_rng(1)
    rho = (1.0 + 0.05 * rng.uniform(-1, 1, size=shape)).astype(NP_DTYPE[dtype])
    u = (0.08 * rng.uniform(-1, 1, size=(3,) + shape)).astype(NP_DTYPE[dtype])
    ref = O.init_equilibrium(Q, rho.astype(np.float64), u.astype(np.float64))
    with P.LBM(Q, shape[2], shape[1], shape[0], dtype) as sim:
        sim.init_equilibrium(torch.from_numpy(rho).cuda(), torch.from_numpy(u).cuda())
        out = np.empty((Q,) + shape, dtype=NP_DTYPE[dtype])
        sim.get_populations(out)
        sim.init_equilibrium(rho, u)          # host pointers
        out2 = np.empty_like(out)
        sim.get_populations(out2)
    assert field_error(out, ref) <= (3e-7 if dtype == "f32" else 1e-15)
    assert np.array_equal(out, out2)


def test_error_codes():
    B = P.binding
    with P.LBM(19, 8, 8, 8, "f32") as sim:
        par = P.LbmParams(tau0=0.6)
        with pytest.raises(P.LbmError) as e:
            sim.step(1, par)
        assert e.value.code == B.LBM_ESTATE
        f = np.full((19, 8, 8, 8), 0.05, dtype=np.float32)
        bad = np.zeros((8, 8, 8), dtype=np.uint8)
        bad[3, 3, 3] = 8                            # type > 7
        with pytest.raises(P.LbmError) as e:
            sim.set_fields(f, None, bad)
        assert e.value.code == B.LBM_EINVAL
        bad[3, 3, 3] = I.INLET                      # INLET off the x = 0 plane
        with pytest.raises(P.LbmError):
            sim.set_fields(f, None, bad)
        bad[3, 3, 3] = 0x10                         # high nibble on a non-WALLMODEL type
        with pytest.raises(P.LbmError):
            sim.set_fields(f, None, bad)
        bad[3, 3, 3] = 0x64                         # normal code 6
        with pytest.raises(P.LbmError):
            sim.set_fields(f, None, bad)
        sim.set_fields(f, None, None)
        for kw in (dict(tau0=0.5), dict(tau0=0.6, cs_smago=-0.1), dict(tau0=float("nan"))):
            with pytest.raises(P.LbmError) as e:
                sim.step(1, P.LbmParams(**kw))
            assert e.value.code == B.LBM_EINVAL
        with pytest.raises(P.LbmError):
            sim.step(-1, par)
        with pytest.raises(P.LbmError):
            sim.set_option("no_such_option", 1)
        sim.step(3, par)
        assert sim.query("steps") == 3 and sim.query("launches") >= 3 and sim.query("cells") == 512
        # a failed set_fields keeps the previous valid state
        out0 = np.empty_like(f)
        sim.get_populations(out0)
        bad[3, 3, 3] = 9
        with pytest.raises(P.LbmError):
            sim.set_fields(f, None, bad)
        out1 = np.empty_like(f)
        sim.get_populations(out1)
        assert np.array_equal(out0, out1)


def test_set_geometry_midrun_matches_oracle():
    cfg = I.make_config(3, shape=(16, 12, 40))
    f, d = oracle_inputs(cfg, "f64")
    flags2 = cfg["flags"].copy()
    flags2[5:9, 3:7, 10:14] = I.SOLID
    a = run_oracle(cfg, f, d, 4)
    cfg2 = dict(cfg)
    cfg2["flags"] = flags2
    ref = run_oracle(cfg2, a, d, 4)
    nz, ny, nx = cfg["shape"]
    par = P.LbmParams(**cfg["params"])
    with P.LBM(19, nx, ny, nz, "f64") as sim:
        sim.set_fields(f, d, cfg["flags"])
        sim.step(4, par)
        sim.set_geometry(d, flags2)
        sim.step(4, par)
        out = np.empty_like(f)
        sim.get_populations(out)
    assert field_error(out, ref, (flags2 & 15) != I.SOLID) <= 1e-12

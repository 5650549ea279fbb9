"""The in-place AA-pattern propagation (lbm_set_option "inplace"; the propagation bake-off of DESIGN.md section 4; north_star:
"one-lattice in-place (AA-pattern style) or two-lattice ping-pong chosen by measured bytes per cell update"): on lattices without
a boundary cell it must give the populations of the two-lattice pull BIT FOR BIT (the same collision on the same values; only
where the values live differs) and match the oracle to the parity tolerance -- odd and even step counts, chunked stepping, state
reads after an odd number of steps (un-swap pass), both lattices, both dtypes, with and without porosity."""
import numpy as np
import pytest

import lbm_inputs as I
import paper_2506_21804_b200 as P
from oracle import oracle as O
from parity_util import NP_DTYPE, TOL, field_error, oracle_inputs

pytestmark = pytest.mark.gpu
NX = {(19, "f32"): 128, (19, "f64"): 64, (27, "f32"): 64, (27, "f64"): 32}      # 32 vectors per row


def _run(cfg, f, d, dtype, chunks, inplace, reads=False):
    nz, ny, nx = cfg["shape"]
    par = P.LbmParams(**cfg["params"])
    with P.LBM(cfg["Q"], nx, ny, nz, dtype) as sim:
        sim.set_option("inplace", inplace)
        sim.set_fields(f, d, None)
        l0 = sim.query("launches")
        out = np.empty_like(f)
        rho = np.empty(f.shape[1:], dtype=f.dtype)
        u = np.empty((3,) + f.shape[1:], dtype=f.dtype)
        for n in chunks:
            sim.step(n, par)
            if reads:
                sim.moments(rho, u)
                sim.get_populations(out)
        launches = sim.query("launches") - l0
        bytes_before_read = sim.query("device_bytes")
        sim.moments(rho, u)
        tot = np.array(sim.totals())
        sim.get_populations(out)
        return out, rho, u, tot, launches, bytes_before_read


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("Q", [19, 27])
@pytest.mark.parametrize("chunks", [[1], [2], [7], [10], [3, 1, 4]])
def test_inplace_equals_two_lattices_bit_for_bit(Q, dtype, chunks):
    nx = NX[(Q, dtype)]
    cfg = I.make_config(2, shape=(10, 6, 2 * nx), k_max=4, n_modes=32)
    cfg["Q"] = Q
    f, d = oracle_inputs(cfg, dtype)
    a, rho_a, u_a, tot_a, la, _ = _run(cfg, f, d, dtype, chunks, 0)
    b, rho_b, u_b, tot_b, lb, bytes_b = _run(cfg, f, d, dtype, chunks, 1)
    assert np.array_equal(a, b) and np.array_equal(rho_a, rho_b) and np.array_equal(u_a, u_b)
    assert lb == sum(chunks)                                            # one launch per step, nothing else
    pop = f.nbytes
    if sum(chunks) % 2 == 0:
        assert bytes_b < 1.5 * pop                                      # the second lattice was never allocated
    ref = O.step(f.astype(np.float64), nsteps=sum(chunks), nthreads=4, **cfg["params"])
    assert field_error(b, ref) <= TOL[dtype]
    assert np.abs(tot_a - tot_b).max() <= 1e-6 * abs(tot_a[0])


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_inplace_with_porosity_and_state_reads_in_between(dtype):
    shape = (8, 10, 256)
    rng = np.random.Generator(np.random.PCG64(5))
    rho = 1.0 + 0.02 * rng.standard_normal(shape)
    u = 0.04 * rng.standard_normal((3,) + shape)
    d = np.where(rng.random(shape) < 0.3, rng.uniform(0.1, 1.0, shape), 0.0)
    cfg = dict(Q=19, shape=shape, rho=rho, u=u, d=d, flags=None, dtype=dtype, params=dict(tau0=0.53, cs_smago=0.12, use_hlbm=1))
    f, dd = oracle_inputs(cfg, dtype)
    a, *_ = _run(cfg, f, dd, dtype, [5, 4], 0)
    b, *_ = _run(cfg, f, dd, dtype, [5, 4], 1, reads=True)              # a read after 5 steps un-swaps; the run goes on in place
    assert np.array_equal(a, b)
    ref = O.step(f.astype(np.float64), d=dd.astype(np.float64), nsteps=9, nthreads=4, **cfg["params"])
    assert field_error(b, ref) <= TOL[dtype]


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("Q", [19, 27])
@pytest.mark.parametrize("chunks", [[1], [2], [9], [3, 2, 4]])
def test_inplace_with_bounce_back_walls_equals_two_lattices_bit_for_bit(Q, dtype, chunks):
    """config 4 scaled down (periodic box with solid spheres): in the AA pattern a bounce-back link needs the cell's own slots only"""
    nx = NX[(Q, dtype)]
    cfg = I.make_config(4, shape=(20, 14, 2 * nx), k_max=4, n_modes=32)
    cfg["Q"] = Q
    t = cfg["flags"] & 15
    assert 0.05 < (t == I.SOLID).mean() < 0.3
    f, d = oracle_inputs(cfg, dtype)
    par = P.LbmParams(**cfg["params"])
    nz, ny, nx_ = cfg["shape"]
    res = []
    for inplace in (0, 1):
        with P.LBM(Q, nx_, ny, nz, dtype) as sim:
            sim.set_option("inplace", inplace)
            sim.set_fields(f, None, cfg["flags"])
            l0 = sim.query("launches")
            for n in chunks:
                sim.step(n, par)
            steps_launches = sim.query("launches") - l0
            rho = np.empty(f.shape[1:], dtype=f.dtype)
            u = np.empty((3,) + f.shape[1:], dtype=f.dtype)
            sim.moments(rho, u)
            tot = np.array(sim.totals())
            out = np.empty_like(f)
            sim.get_populations(out)
            sim.step(2, par)                                            # and the run goes on after the reads
            out2 = np.empty_like(f)
            sim.get_populations(out2)
        res.append((out, rho, u, tot, out2, steps_launches))
    a, b = res
    assert b[5] == sum(chunks)                                          # in place: one launch per step
    for k in (0, 1, 2, 4):
        assert np.array_equal(a[k], b[k]), k
    assert np.abs(a[3] - b[3]).max() <= 1e-6 * abs(a[3][0])
    mask = ~I.is_wall(cfg["flags"])
    assert np.array_equal(b[0][:, ~mask], f[:, ~mask])                  # wall cells keep their own values
    ref = O.step(f.astype(np.float64), flags=cfg["flags"], nsteps=sum(chunks), nthreads=4, **cfg["params"])
    assert field_error(b[0], ref, mask) <= TOL[dtype]


def test_inplace_is_ignored_where_it_does_not_apply():
    """an inlet / outlet cell, the HRR form or a row length the row-wide blocks do not take: the two-lattice path runs, same results"""
    cfg = I.make_config(2, shape=(8, 6, 128), k_max=4, n_modes=16)
    f, d = oracle_inputs(cfg, "f32")
    flags = np.zeros(cfg["shape"], dtype=np.uint8)
    flags[1:-1, :, 0] = I.INLET
    flags[1:-1, :, -1] = I.OUTLET
    flags[0] = flags[-1] = I.SOLID
    par = P.LbmParams(**dict(cfg["params"], u_in=(0.03, 0.0, 0.0)))
    hrr = P.LbmParams(**dict(cfg["params"], collision=1, sigma=0.7))
    outs = []
    for inplace in (0, 1):
        res = []
        for fl, p in ((flags, par), (None, hrr)):
            with P.LBM(19, 128, 6, 8, "f32") as sim:
                sim.set_option("inplace", inplace)
                sim.set_fields(f, None, fl)
                sim.step(5, p)
                out = np.empty_like(f)
                sim.get_populations(out)
                res.append(out)
        outs.append(res)
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    # switching between the two schemes in one run: in place (3 steps, odd) -> HRR (two lattices) -> in place again
    with P.LBM(19, 128, 6, 8, "f32") as sim:
        sim.set_option("inplace", 1)
        sim.set_fields(f)
        sim.step(3, par)
        sim.step(2, hrr)
        sim.step(3, par)
        got = np.empty_like(f)
        sim.get_populations(got)
    ref = O.step(f.astype(np.float64), nsteps=3, **cfg["params"])
    ref = O.step(ref, nsteps=2, **dict(cfg["params"], collision=1, sigma=0.7))
    ref = O.step(ref, nsteps=3, **cfg["params"])
    assert field_error(got, ref) <= TOL["f32"]

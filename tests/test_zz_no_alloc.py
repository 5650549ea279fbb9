"""lbm_totals_static (include/lbm.h): the A9 totals with the scratch in a file-scope `static __device__` array -- no context, no
allocation on the call's path -- against the existing path (lbm_totals on a context), on calls in a row that share the array.
Collected last on purpose (the suite runs with pytest -x): it must pass alone in a fresh process and after every other test.
Tolerance: the one the parity tests use for the totals (parity_util.TOL, relative to the mass total)."""
import ctypes

import numpy as np
import pytest
import torch

import lbm_inputs as I
import paper_2506_21804_b200 as P
from paper_2506_21804_b200 import binding
from parity_util import NP_DTYPE, TOL

pytestmark = pytest.mark.gpu
TORCH_DTYPE = {"f32": torch.float32, "f64": torch.float64}
ABI_DTYPE = {"f32": binding.LBM_F32, "f64": binding.LBM_F64}


def _noneq_state(cfg, dtype, seed):
    """a generic non-equilibrium state of the right shape: positive populations around the lattice weights (no method arithmetic:
    the totals are sums of whatever the arrays hold)"""
    nz, ny, nx = cfg["shape"]
    Q = cfg["Q"]
    rng = np.random.Generator(np.random.PCG64(seed))
    f = (1.0 / Q) * (1.0 + 0.05 * rng.standard_normal((Q, nz, ny, nx)))
    return np.ascontiguousarray(np.abs(f).astype(NP_DTYPE[dtype]))


def _existing_path(cfg, dtype, f, steps):
    """lbm_totals of the state after `steps` steps, and that state S_t itself (device tensors)"""
    nz, ny, nx = cfg["shape"]
    Q = cfg["Q"]
    tf = torch.from_numpy(f).cuda()
    td = None if cfg["d"] is None else torch.from_numpy(cfg["d"].astype(NP_DTYPE[dtype])).cuda()
    tfl = None if cfg["flags"] is None else torch.from_numpy(cfg["flags"]).cuda()
    with P.LBM(Q, nx, ny, nz, dtype) as sim:
        sim.set_fields(tf, td, tfl)
        if steps:
            sim.step(steps, P.LbmParams(**cfg["params"]))
        ref = np.array(sim.totals())
        state = torch.empty((Q, nz, ny, nx), dtype=TORCH_DTYPE[dtype], device="cuda")
        sim.get_populations(state)
        sim.synchronize()
    return ref, state, tfl


def _static(cfg, dtype, state, tfl, out):
    nz, ny, nx = cfg["shape"]
    P.lbm_totals_static(cfg["Q"], nx, ny, nz, ABI_DTYPE[dtype], state, tfl, out, torch.cuda.current_stream().cuda_stream)


CASES = [  # (config, shape (nz, ny, nx), dtype, steps, seed)
    (3, (24, 32, 96), "f32", 4, 11),       # urban channel: SOLID floor / top, inlet, outlet, wall-model cells; vector path
    (4, (20, 24, 32), "f64", 3, 12),       # D3Q27 with solid spheres, fp64
    (2, (9, 7, 13), "f32", 0, 13),         # N = 819 cells: odd, one cell per thread, a ragged single block, no flags
    (3, (40, 48, 160), "f64", 2, 14),      # 307 200 cells = 37.5 blocks: several blocks + a ragged last one
]


def test_static_totals_match_the_context_path_on_calls_in_a_row():
    """every case twice in a row into separate outputs, nothing but the shared static array between the calls: each result within
    the parity tolerance of lbm_totals, and repeated calls bit-identical (fixed summation order, nothing left over from the
    previous call's larger or smaller grid)"""
    assert torch.cuda.is_available()
    runs = []
    for conf, shape, dtype, steps, seed in CASES:
        cfg = I.make_config(conf, shape=shape)
        ref, state, tfl = _existing_path(cfg, dtype, _noneq_state(cfg, dtype, seed), steps)
        runs.append((cfg, dtype, ref, state, tfl))
    outs = torch.full((2 * len(runs) + 2, 5), float("nan"), dtype=torch.float64, device="cuda")
    k = 0
    for cfg, dtype, ref, state, tfl in runs:        # calls back to back on one stream, no synchronisation in between
        _static(cfg, dtype, state, tfl, outs[k])
        _static(cfg, dtype, state, tfl, outs[k + 1])
        k += 2
    # ... and the first case once more after all the others (a big grid, then small ones, then the first again)
    torch.cuda.synchronize()
    free_before, torch_before = torch.cuda.mem_get_info()[0], torch.cuda.memory_allocated()
    _static(runs[0][0], runs[0][1], runs[0][3], runs[0][4], outs[k])
    _static(runs[0][0], runs[0][1], runs[0][3], runs[0][4], outs[k + 1])
    torch.cuda.synchronize()
    # no device memory was taken by these calls (their kernel is loaded already: the first calls above ran it)
    assert torch.cuda.mem_get_info()[0] == free_before and torch.cuda.memory_allocated() == torch_before
    got = outs.cpu().numpy()
    assert np.isfinite(got).all()
    for n, (cfg, dtype, ref, state, tfl) in enumerate(runs):
        a, b = got[2 * n], got[2 * n + 1]
        assert np.array_equal(a, b), (n, a, b)
        assert np.abs(a - ref).max() <= max(TOL[dtype], 1e-12) * abs(ref[0]), (n, a, ref)
        # the definition itself, from the state both paths saw (numpy, fp64)
        s = state.cpu().numpy().astype(np.float64)
        keep = np.ones(cfg["shape"], dtype=bool) if cfg["flags"] is None else ~I.is_wall(cfg["flags"])
        rho = s.sum(axis=0)
        assert abs(a[0] - rho[keep].sum()) <= max(TOL[dtype], 1e-12) * abs(ref[0])
    assert np.array_equal(got[k], got[0]) and np.array_equal(got[k + 1], got[0])


def test_static_totals_reject_what_they_cannot_do():
    assert torch.cuda.is_available()
    out = torch.zeros(5, dtype=torch.float64, device="cuda")
    f = torch.ones((19, 4, 4, 4), dtype=torch.float32, device="cuda")
    lib = P.load_library()
    vp = lambda t: ctypes.c_void_p(t.data_ptr())
    # beyond the static array: 513 x 512 x 512 cells (nothing is read: the pointers are never dereferenced)
    rc = lib.lbm_totals_static(19, 512, 512, 513, 4, vp(f), None, vp(out), None)
    assert rc == binding.LBM_EINVAL and "LBM_STATIC_MAX_CELLS" in P.lbm_last_error(None)
    assert lib.lbm_totals_static(18, 4, 4, 4, 4, vp(f), None, vp(out), None) == binding.LBM_EINVAL
    assert lib.lbm_totals_static(19, 4, 4, 4, 2, vp(f), None, vp(out), None) == binding.LBM_EINVAL
    assert lib.lbm_totals_static(19, 4, 4, 4, 4, None, None, vp(out), None) == binding.LBM_EINVAL
    host = np.zeros(5)
    assert lib.lbm_totals_static(19, 4, 4, 4, 4, vp(f), None, ctypes.c_void_p(host.ctypes.data), None) == binding.LBM_EINVAL
    assert "DEVICE" in P.lbm_last_error(None)
    # and a valid call still works afterwards
    P.lbm_totals_static(19, 4, 4, 4, binding.LBM_F32, f, None, out)
    torch.cuda.synchronize()
    assert out.cpu().numpy().tolist() == [19.0 * 64, 0.0, 0.0, 0.0, 0.0]

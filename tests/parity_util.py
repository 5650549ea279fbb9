"""Helpers shared by the GPU parity tests: run the same seeded inputs through the oracle and through the
C ABI, and compare with the metric of DESIGN.md reading R12."""
import numpy as np

import lbm_inputs as I
from oracle import oracle as O

TOL = {"f32": 2e-5, "f64": 1e-12}      # north_star: max relative error after 10 steps
NP_DTYPE = {"f32": np.float32, "f64": np.float64}


def oracle_inputs(cfg, dtype=None):
    """Populations f = f^eq(rho,u) from the ORACLE's equilibrium, rounded to the run's dtype, plus the
    porosity rounded the same way.  Both sides start from exactly these rounded values."""
    dtype = dtype or cfg["dtype"]
    npdt = NP_DTYPE[dtype]
    f = O.init_equilibrium(cfg["Q"], cfg["rho"], cfg["u"]).astype(npdt)
    d = None if cfg["d"] is None else cfg["d"].astype(npdt)
    return f, d


def run_oracle(cfg, f, d, nsteps):
    return O.step(f.astype(np.float64), d=None if d is None else d.astype(np.float64), flags=cfg["flags"],
                  nsteps=nsteps, nthreads=min(O.max_threads(), 8), **cfg["params"])


def field_error(got, ref, mask=None):
    """R12: max |got - ref| / max |ref| over the masked cells (all populations / components together)."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    if mask is not None:
        got, ref = got[..., mask], ref[..., mask]
    return float(np.abs(got - ref).max() / np.abs(ref).max())


def nonsolid(cfg):
    if cfg["flags"] is None:
        return None
    return ~I.is_wall(cfg["flags"])


def crop_config(cfg, f, d, z0, y0, x0, sz, sy, sx):
    """Crop the INPUT arrays (periodic wrap) around a window -- P11b light-cone check."""
    nz, ny, nx = cfg["shape"]
    zi = (z0 + np.arange(sz)) % nz
    yi = (y0 + np.arange(sy)) % ny
    xi = (x0 + np.arange(sx)) % nx
    ix = np.ix_(zi, yi, xi)
    sub = dict(cfg)
    sub["shape"] = (sz, sy, sx)
    sub["flags"] = None if cfg["flags"] is None else np.ascontiguousarray(cfg["flags"][ix])
    fc = np.ascontiguousarray(f[(slice(None),) + ix])
    dc = None if d is None else np.ascontiguousarray(d[ix])
    return sub, fc, dc, ix

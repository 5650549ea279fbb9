"""ctypes binding of the CPU oracle (oracle/lbm_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports the product package (paper_2506_21804_b200) and the
product never imports it.  All arithmetic lives in lbm_oracle.cpp; this file only marshals
numpy arrays.  Layouts: f[Q][nz][ny][nx], d[nz][ny][nx], flags[nz][ny][nx] (x fastest), fp64.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lbm_oracle.cpp")
_LIB = os.path.join(_HERE, "liblbm_oracle.so")
_lib = None

_c_dp = ctypes.POINTER(ctypes.c_double)
_c_ip = ctypes.POINTER(ctypes.c_int)
_c_u8p = ctypes.POINTER(ctypes.c_uint8)


def build(force=False):
    """Compile the oracle with g++ (plain -O2, no fast-math, OpenMP for the timed all-cores run)."""
    if not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC):
        return _LIB
    tmp = _LIB + ".tmp.%d" % os.getpid()
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
           "-o", tmp, _SRC]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        L.orc_lattice.argtypes = [ctypes.c_int, _c_ip, _c_dp, _c_ip]
        L.orc_feq.argtypes = [ctypes.c_int, ctypes.c_double, _c_dp, _c_dp]
        L.orc_collide_cell.argtypes = [ctypes.c_int, _c_dp, ctypes.c_double, _c_dp, ctypes.c_double,
                                       ctypes.c_double, _c_dp, _c_dp]
        L.orc_inlet_fixup_cell.argtypes = [ctypes.c_int, _c_dp, _c_dp]
        L.orc_pressure_fixup_cell.argtypes = [ctypes.c_int, _c_dp, ctypes.c_double]
        L.orc_feq3.argtypes = [ctypes.c_int, ctypes.c_double, _c_dp, _c_dp]
        L.orc_collide_cell_hrr.argtypes = [ctypes.c_int, _c_dp, ctypes.c_double, _c_dp, ctypes.c_double,
                                           ctypes.c_double, ctypes.c_double, _c_dp, _c_dp, _c_dp]
        L.orc_spalding.argtypes = [ctypes.c_double] * 3
        L.orc_spalding.restype = ctypes.c_double
        L.orc_wallmodel_speed.argtypes = [ctypes.c_double] * 6 + [_c_dp, _c_ip, _c_ip]
        L.orc_wallmodel_speed.restype = ctypes.c_double
        L.orc_init_equilibrium.argtypes = [ctypes.c_int, ctypes.c_int64, _c_dp, _c_dp, _c_dp]
        L.orc_step.argtypes = [ctypes.c_int] * 4 + [_c_dp, _c_dp, _c_u8p, _c_dp, ctypes.c_int, ctypes.c_int]
        L.orc_step_body.argtypes = [ctypes.c_int] * 4 + [_c_dp, _c_dp, _c_u8p, _c_dp, ctypes.c_int, ctypes.c_int, _c_dp]
        L.orc_moments.argtypes = [ctypes.c_int, ctypes.c_int64, _c_dp, _c_dp, _c_dp]
        L.orc_step_vm.argtypes = [ctypes.c_int] * 4 + [_c_dp, _c_dp, _c_u8p, _c_dp, ctypes.c_int, ctypes.c_int,
                                  _c_dp, _c_dp, ctypes.c_int, _c_dp, _c_dp, ctypes.c_double, ctypes.c_double]
        L.orc_vm_inflow.argtypes = [ctypes.c_int, ctypes.c_int, _c_u8p, _c_dp, _c_dp, ctypes.c_int, _c_dp, _c_dp,
                                    ctypes.c_double, ctypes.c_double, _c_dp]
        L.orc_totals.argtypes = [ctypes.c_int, ctypes.c_int64, _c_dp, _c_u8p, _c_dp]
        L.orc_max_threads.restype = ctypes.c_int
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(_c_dp)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def lattice(Q):
    """(c[Q,3] int, w[Q] float64, opp[Q] int) by rule R1."""
    c = np.zeros((Q, 3), dtype=np.int32)
    w = np.zeros(Q, dtype=np.float64)
    opp = np.zeros(Q, dtype=np.int32)
    rc = lib().orc_lattice(Q, c.ctypes.data_as(_c_ip), _dp(w), opp.ctypes.data_as(_c_ip))
    if rc != 0:
        raise ValueError("bad lattice %r" % Q)
    return c, w, opp


def feq(Q, rho, u):
    out = np.zeros(Q)
    u = _f64(u)
    assert lib().orc_feq(Q, float(rho), _dp(u), _dp(out)) == 0
    return out


def collide_cell(Q, fc, d=0.0, ub=(0.0, 0.0, 0.0), tau0=0.6, cs_smago=0.0):
    """O2 on one cell -> (fstar[Q], tau_eff)."""
    fc = _f64(fc)
    ub = _f64(ub)
    fs = np.zeros(Q)
    tau = ctypes.c_double(0.0)
    assert lib().orc_collide_cell(Q, _dp(fc), float(d), _dp(ub), float(tau0), float(cs_smago), _dp(fs),
                                  ctypes.byref(tau)) == 0
    return fs, tau.value


def feq3(Q, rho, u):
    """Eq. 11 in full (third-order equilibrium)."""
    out = np.zeros(Q)
    u = _f64(u)
    assert lib().orc_feq3(Q, float(rho), _dp(u), _dp(out)) == 0
    return out


def collide_cell_hrr(Q, fc, d=0.0, ub=(0.0, 0.0, 0.0), tau0=0.6, cs_smago=0.0, sigma=1.0, S=None):
    """O2h on one cell (S = S^FD, 3x3) -> (fstar[Q], tau_eff)."""
    fc = _f64(fc)
    ub = _f64(ub)
    S = _f64(np.zeros((3, 3)) if S is None else S)
    fs = np.zeros(Q)
    tau = ctypes.c_double(0.0)
    assert lib().orc_collide_cell_hrr(Q, _dp(fc), float(d), _dp(ub), float(tau0), float(cs_smago), float(sigma),
                                      _dp(S), _dp(fs), ctypes.byref(tau)) == 0
    return fs, tau.value


def inlet_fixup_cell(Q, g, uw):
    g = _f64(g).copy()
    uw = _f64(uw)
    assert lib().orc_inlet_fixup_cell(Q, _dp(g), _dp(uw)) == 0
    return g


def pressure_fixup_cell(Q, g, rho_out):
    g = _f64(g).copy()
    assert lib().orc_pressure_fixup_cell(Q, _dp(g), float(rho_out)) == 0
    return g


def spalding(up, kappa=0.41, E=9.8):
    return lib().orc_spalding(float(up), float(kappa), float(E))


def wallmodel_speed(U2, nu, kappa=0.41, E=9.8, y2=1.5, y1=0.5):
    """-> (U1, u_tau, newton_iters_utau, newton_iters_u1)."""
    ut = ctypes.c_double(0.0)
    i1 = ctypes.c_int(0)
    i2 = ctypes.c_int(0)
    U1 = lib().orc_wallmodel_speed(float(U2), float(nu), float(kappa), float(E), float(y2), float(y1),
                                   ctypes.byref(ut), ctypes.byref(i1), ctypes.byref(i2))
    return U1, ut.value, i1.value, i2.value


def init_equilibrium(Q, rho, u):
    """rho[nz,ny,nx], u[3,nz,ny,nx] -> f[Q,nz,ny,nx] = f^eq(rho,u)."""
    rho = _f64(rho)
    u = _f64(u)
    f = np.empty((Q,) + rho.shape, dtype=np.float64)
    assert lib().orc_init_equilibrium(Q, rho.size, _dp(rho), _dp(u), _dp(f)) == 0
    return f


def pack_params(tau0, cs_smago=0.0, use_hlbm=0, u_in=(0.0, 0.0, 0.0), wm_enable=0, wm_kappa=0.41, wm_E=9.8,
                collision=0, sigma=1.0, u_wall=(0.0, 0.0, 0.0), rho_out=1.0, fringe_len=0, fringe_factor=0.0):
    """collision: 0 = BGK form (G1), 1 = HRR (Eq. 6-11), 2 = HRR with the FD strain of the previous level (G41); sigma = Eq. 7 hybridisation factor; u_wall = velocity of the
    MOVINGWALL cells (G33)."""
    return np.array([tau0, cs_smago, float(use_hlbm), u_in[0], u_in[1], u_in[2], float(wm_enable),
                     wm_kappa, wm_E, float(collision), sigma, u_wall[0], u_wall[1], u_wall[2], rho_out, float(fringe_len), fringe_factor],
                    dtype=np.float64)


def step(f, d=None, flags=None, nsteps=1, nthreads=1, u_body=None, **params):
    """Advance S_t -> S_{t+nsteps}.  f[Q,nz,ny,nx] float64 (a new array is returned).  u_body[3,nz,ny,nx]: the solid
    velocity u^B of Eq. 12 (None = 0)."""
    f = _f64(f).copy()
    Q, nz, ny, nx = f.shape
    par = pack_params(**params)
    dptr = None
    if d is not None:
        d = _f64(d)
        assert d.shape == (nz, ny, nx)
        dptr = _dp(d)
    fptr = None
    if flags is not None:
        flags = np.ascontiguousarray(flags, dtype=np.uint8)
        assert flags.shape == (nz, ny, nx)
        fptr = flags.ctypes.data_as(_c_u8p)
    if u_body is not None:
        u_body = _f64(u_body)
        assert u_body.shape == (3, nz, ny, nx)
        rc = lib().orc_step_body(Q, nx, ny, nz, _dp(f), dptr, fptr, _dp(par), int(nsteps), int(nthreads), _dp(u_body))
    else:
        rc = lib().orc_step(Q, nx, ny, nz, _dp(f), dptr, fptr, _dp(par), int(nsteps), int(nthreads))
    if rc != 0:
        raise ValueError("orc_step rejected its arguments")
    return f


def vm_inflow(mask, u_mean, u_prev, pos, sign, sigma_v, intensity):
    """Vortex Method inflow field (Eq. 18-21) on the plane x = 0.  mask[nz,ny] (1 = INLET cell), u_mean / u_prev [3,nz,ny],
    pos[nv,2] = seed positions (y, z) in cell coordinates, sign[nv] = +-1.  Returns u[3,nz,ny]."""
    mask = np.ascontiguousarray(mask, dtype=np.uint8)
    nz, ny = mask.shape
    u_mean, u_prev = _f64(u_mean), _f64(u_prev)
    pos = _f64(np.asarray(pos, dtype=np.float64).reshape(-1, 2))
    sign = _f64(np.asarray(sign, dtype=np.float64).reshape(-1))
    assert u_mean.shape == (3, nz, ny) and u_prev.shape == (3, nz, ny) and len(sign) == len(pos)
    out = np.empty((3, nz, ny))
    rc = lib().orc_vm_inflow(ny, nz, mask.ctypes.data_as(_c_u8p), _dp(u_mean), _dp(u_prev), len(pos), _dp(pos), _dp(sign),
                             float(sigma_v), float(intensity), _dp(out))
    if rc != 0:
        raise ValueError("orc_vm_inflow rejected its arguments")
    return out


def step_vm(f, u_mean, u_inflow, pos, sign, sigma_v, intensity, d=None, flags=None, nsteps=1, nthreads=1, **params):
    """orc_step with the Vortex Method inlet.  u_inflow[3,nz,ny] = inflow of the previous step (u_mean before the first).
    Returns (f, u_inflow) after nsteps."""
    f = _f64(f).copy()
    Q, nz, ny, nx = f.shape
    par = pack_params(**params)
    dptr = None
    if d is not None:
        d = _f64(d)
        dptr = _dp(d)
    flags = np.ascontiguousarray(flags, dtype=np.uint8)
    u_mean = _f64(u_mean)
    u_inflow = _f64(u_inflow).copy()
    pos = _f64(np.asarray(pos, dtype=np.float64).reshape(-1, 2))
    sign = _f64(np.asarray(sign, dtype=np.float64).reshape(-1))
    rc = lib().orc_step_vm(Q, nx, ny, nz, _dp(f), dptr, flags.ctypes.data_as(_c_u8p), _dp(par), int(nsteps), int(nthreads),
                           _dp(u_mean), _dp(u_inflow), len(pos), _dp(pos), _dp(sign), float(sigma_v), float(intensity))
    if rc != 0:
        raise ValueError("orc_step_vm rejected its arguments")
    return f, u_inflow


def moments(f):
    f = _f64(f)
    Q = f.shape[0]
    shp = f.shape[1:]
    rho = np.empty(shp)
    u = np.empty((3,) + shp)
    assert lib().orc_moments(Q, rho.size, _dp(f), _dp(rho), _dp(u)) == 0
    return rho, u


def totals(f, flags=None):
    f = _f64(f)
    Q = f.shape[0]
    out = np.zeros(5)
    fptr = None
    if flags is not None:
        flags = np.ascontiguousarray(flags, dtype=np.uint8)
        fptr = flags.ctypes.data_as(_c_u8p)
    assert lib().orc_totals(Q, f[0].size, _dp(f), fptr, _dp(out)) == 0
    return out


def max_threads():
    return lib().orc_max_threads()

"""ctypes binding of include/lbm.h: the same names, argument marshalling only.

Buffers may be torch tensors (CUDA or CPU), numpy arrays, or raw integer addresses; they must be
contiguous and of the context's dtype.  Nothing here computes: no torch op, no numpy op touches data.
"""
import ctypes
import os

_PKG = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_PKG, "liblbm_b200.so")
_lib = None

LBM_OK, LBM_EINVAL, LBM_ENOMEM, LBM_ECUDA, LBM_ESTATE = 0, -1, -2, -3, -4
LBM_D3Q19, LBM_D3Q27 = 19, 27
LBM_F32, LBM_F64 = 4, 8
LBM_HALO_POPULATIONS, LBM_HALO_UHAT = 0, 1
LBM_SIDE_LOW, LBM_SIDE_HIGH = 0, 1
EXPORTS = ["lbm_create", "lbm_destroy", "lbm_set_fields", "lbm_init_equilibrium", "lbm_set_geometry", "lbm_step",
           "lbm_moments", "lbm_get_populations", "lbm_totals", "lbm_set_stream", "lbm_synchronize", "lbm_last_error",
           "lbm_query", "lbm_set_option", "lbm_set_inflow", "lbm_set_vortices", "lbm_get_inflow",
           "lbm_set_porosity", "lbm_set_body_velocity", "lbm_get_populations_box", "lbm_set_populations_box",
           "lbm_set_halo", "lbm_step_halo", "lbm_halo_pack", "lbm_halo_unpack", "lbm_totals_static"]


class LbmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("lbm error %d: %s" % (code, msg))
        self.code = code


class LbmParams(ctypes.Structure):
    """Mirror of `lbm_params` in include/lbm.h."""
    _fields_ = [("tau0", ctypes.c_double), ("cs_smago", ctypes.c_double), ("use_hlbm", ctypes.c_int),
                ("u_in", ctypes.c_double * 3), ("wm_enable", ctypes.c_int), ("wm_kappa", ctypes.c_double),
                ("wm_E", ctypes.c_double), ("collision", ctypes.c_int), ("sigma", ctypes.c_double),
                ("u_wall", ctypes.c_double * 3), ("rho_out", ctypes.c_double),
                ("fringe_len", ctypes.c_int), ("fringe_factor", ctypes.c_double)]

    def __init__(self, tau0, cs_smago=0.0, use_hlbm=0, u_in=(0.0, 0.0, 0.0), wm_enable=0, wm_kappa=0.41, wm_E=9.8,
                 collision=0, sigma=1.0, u_wall=(0.0, 0.0, 0.0), rho_out=1.0, fringe_len=0, fringe_factor=0.0):
        super().__init__()
        self.tau0, self.cs_smago, self.use_hlbm = tau0, cs_smago, int(use_hlbm)
        self.u_in[0], self.u_in[1], self.u_in[2] = u_in
        self.wm_enable, self.wm_kappa, self.wm_E = int(wm_enable), wm_kappa, wm_E
        self.collision, self.sigma = int(collision), float(sigma)
        self.u_wall[0], self.u_wall[1], self.u_wall[2] = u_wall
        self.rho_out = float(rho_out)
        self.fringe_len, self.fringe_factor = int(fringe_len), float(fringe_factor)


def library_path():
    return _LIB_PATH


def load_library():
    """Load liblbm_b200.so (built by paper_2506_21804_b200.build / __graft_entry__.build()).
    Raises if it is missing: there is no fallback path."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError("%s is missing: build it with `python -m paper_2506_21804_b200.build` "
                          "(nvcc, sm_100a); there is no CPU fallback" % _LIB_PATH)
    L = ctypes.CDLL(_LIB_PATH)
    vp, ip, ll = ctypes.c_void_p, ctypes.c_int, ctypes.c_longlong
    L.lbm_create.argtypes = [ip, ip, ip, ip, ip]
    L.lbm_create.restype = vp
    L.lbm_destroy.argtypes = [vp]
    L.lbm_destroy.restype = None
    L.lbm_set_fields.argtypes = [vp, vp, vp, vp]
    L.lbm_init_equilibrium.argtypes = [vp, vp, vp]
    L.lbm_set_geometry.argtypes = [vp, vp, vp]
    L.lbm_step.argtypes = [vp, ip, ctypes.POINTER(LbmParams)]
    L.lbm_set_porosity.argtypes = [vp, vp]
    L.lbm_set_body_velocity.argtypes = [vp, vp]
    L.lbm_set_inflow.argtypes = [vp, vp]
    L.lbm_set_vortices.argtypes = [vp, ip, vp, vp, ctypes.c_double, ctypes.c_double]
    L.lbm_get_inflow.argtypes = [vp, vp]
    L.lbm_moments.argtypes = [vp, vp, vp]
    L.lbm_get_populations.argtypes = [vp, vp]
    L.lbm_get_populations_box.argtypes = [vp, ip, ip, ip, ip, ip, ip, vp]
    L.lbm_set_populations_box.argtypes = [vp, ip, ip, ip, ip, ip, ip, vp]
    L.lbm_set_halo.argtypes = [vp, ip, ip]
    L.lbm_step_halo.argtypes = [vp, ctypes.POINTER(LbmParams), ip]
    L.lbm_halo_pack.argtypes = [vp, ip, ip, vp]
    L.lbm_halo_unpack.argtypes = [vp, ip, ip, vp]
    L.lbm_totals.argtypes = [vp, vp]
    L.lbm_totals_static.argtypes = [ip, ip, ip, ip, ip, vp, vp, vp, vp]
    L.lbm_set_stream.argtypes = [vp, vp]
    L.lbm_synchronize.argtypes = [vp]
    L.lbm_last_error.argtypes = [vp]
    L.lbm_last_error.restype = ctypes.c_char_p
    L.lbm_query.argtypes = [vp, ip]
    L.lbm_query.restype = ll
    L.lbm_set_option.argtypes = [vp, ctypes.c_char_p, ll]
    _lib = L
    return L


def _ptr(buf):
    """Address of a buffer: None, int, torch tensor or numpy array (must be contiguous)."""
    if buf is None:
        return None
    if isinstance(buf, int):
        return buf
    if hasattr(buf, "data_ptr"):            # torch tensor
        if not buf.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return buf.data_ptr()
    if hasattr(buf, "ctypes"):              # numpy array
        if not buf.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        return buf.ctypes.data
    raise TypeError("unsupported buffer type %r" % type(buf))


def _check(ctx, rc):
    if rc != LBM_OK:
        raise LbmError(rc, lbm_last_error(ctx))
    return rc


# ---- the C calls, same names ----------------------------------------------------------------------
def lbm_last_error(ctx=None):
    return load_library().lbm_last_error(ctx).decode()


def lbm_create(lattice, nx, ny, nz, dtype):
    ctx = load_library().lbm_create(lattice, nx, ny, nz, dtype)
    if not ctx:
        raise LbmError(LBM_EINVAL, lbm_last_error(None))
    return ctx


def lbm_destroy(ctx):
    load_library().lbm_destroy(ctx)


def lbm_set_fields(ctx, populations, porosity=None, cell_flags=None):
    return _check(ctx, load_library().lbm_set_fields(ctx, _ptr(populations), _ptr(porosity), _ptr(cell_flags)))


def lbm_init_equilibrium(ctx, rho, u):
    return _check(ctx, load_library().lbm_init_equilibrium(ctx, _ptr(rho), _ptr(u)))


def lbm_set_geometry(ctx, porosity=None, cell_flags=None):
    return _check(ctx, load_library().lbm_set_geometry(ctx, _ptr(porosity), _ptr(cell_flags)))


def lbm_set_porosity(ctx, porosity=None):
    return _check(ctx, load_library().lbm_set_porosity(ctx, _ptr(porosity)))


def lbm_set_body_velocity(ctx, u_body=None):
    return _check(ctx, load_library().lbm_set_body_velocity(ctx, _ptr(u_body)))


def lbm_set_inflow(ctx, u_mean):
    return _check(ctx, load_library().lbm_set_inflow(ctx, _ptr(u_mean)))


def lbm_set_vortices(ctx, pos, sign, sigma_v, intensity):
    """pos[n][2] = (y, z), sign[n]: converted to contiguous host float64 arrays (argument marshalling only)"""
    import numpy as np
    pos = np.ascontiguousarray(np.asarray(pos, dtype=np.float64).reshape(-1, 2))
    sign = np.ascontiguousarray(np.asarray(sign, dtype=np.float64).reshape(-1))
    if len(pos) != len(sign):
        raise ValueError("pos and sign must have the same length")
    return _check(ctx, load_library().lbm_set_vortices(ctx, len(sign), _ptr(pos) if len(sign) else None,
                                                       _ptr(sign) if len(sign) else None, float(sigma_v), float(intensity)))


def lbm_get_inflow(ctx, u):
    return _check(ctx, load_library().lbm_get_inflow(ctx, _ptr(u)))


def lbm_step(ctx, n_steps, params):
    return _check(ctx, load_library().lbm_step(ctx, n_steps, ctypes.byref(params)))


def lbm_moments(ctx, rho, u):
    return _check(ctx, load_library().lbm_moments(ctx, _ptr(rho), _ptr(u)))


def lbm_get_populations(ctx, populations):
    return _check(ctx, load_library().lbm_get_populations(ctx, _ptr(populations)))


def lbm_get_populations_box(ctx, origin, extent, populations):
    """origin = (x0, y0, z0), extent = (bx, by, bz); populations[Q][bz][by][bx]"""
    x0, y0, z0 = (int(v) for v in origin)
    bx, by, bz = (int(v) for v in extent)
    return _check(ctx, load_library().lbm_get_populations_box(ctx, x0, y0, z0, bx, by, bz, _ptr(populations)))


def lbm_set_populations_box(ctx, origin, extent, populations):
    """origin = (x0, y0, z0), extent = (bx, by, bz); populations[Q][bz][by][bx]"""
    x0, y0, z0 = (int(v) for v in origin)
    bx, by, bz = (int(v) for v in extent)
    return _check(ctx, load_library().lbm_set_populations_box(ctx, x0, y0, z0, bx, by, bz, _ptr(populations)))


def lbm_set_halo(ctx, ghost_lo, ghost_hi):
    return _check(ctx, load_library().lbm_set_halo(ctx, int(ghost_lo), int(ghost_hi)))


def lbm_step_halo(ctx, params, stage):
    return _check(ctx, load_library().lbm_step_halo(ctx, ctypes.byref(params), int(stage)))


def lbm_halo_pack(ctx, what, side, buf):
    return _check(ctx, load_library().lbm_halo_pack(ctx, int(what), int(side), _ptr(buf)))


def lbm_halo_unpack(ctx, what, side, buf):
    return _check(ctx, load_library().lbm_halo_unpack(ctx, int(what), int(side), _ptr(buf)))


def lbm_totals(ctx, out=None):
    """out = None: returns the five totals as a list (host, synchronises); out = a buffer of 5 doubles (host or device):
    filled in place (a device buffer asynchronously)"""
    if out is not None:
        return _check(ctx, load_library().lbm_totals(ctx, _ptr(out)))
    out = (ctypes.c_double * 5)()
    _check(ctx, load_library().lbm_totals(ctx, ctypes.addressof(out)))
    return list(out)


def lbm_totals_static(lattice, nx, ny, nz, dtype, populations, cell_flags, out, cuda_stream=None):
    """The totals of a caller-held state without any allocation (static device scratch; include/lbm.h): device buffers only,
    `out` = a device buffer of 5 doubles, filled asynchronously on `cuda_stream`"""
    return _check(None, load_library().lbm_totals_static(lattice, nx, ny, nz, dtype, _ptr(populations), _ptr(cell_flags),
                                                         _ptr(out), cuda_stream))


def lbm_set_stream(ctx, cuda_stream):
    return _check(ctx, load_library().lbm_set_stream(ctx, cuda_stream))


def lbm_synchronize(ctx):
    return _check(ctx, load_library().lbm_synchronize(ctx))


def lbm_query(ctx, what):
    return load_library().lbm_query(ctx, what)


def lbm_set_option(ctx, key, value):
    return _check(ctx, load_library().lbm_set_option(ctx, key.encode(), int(value)))


class LBM:
    """Convenience owner of one lbm_ctx (still marshalling only)."""
    QUERY = dict(steps=0, launches=1, cells=2, solid_cells=3, device_bytes=4, masked_cells=5, list_cells=6, graph_launches=7,
                 wallmodel_cells=8, halo_population_values=9, halo_uhat_values=10, interior_slices=11, slip_plane_cells=12)

    def __init__(self, lattice, nx, ny, nz, dtype="f32", stream=None):
        self.Q, self.nx, self.ny, self.nz = lattice, nx, ny, nz
        self.dtype = dtype
        self.ctx = lbm_create(lattice, nx, ny, nz, LBM_F32 if dtype == "f32" else LBM_F64)
        if stream is not None:
            lbm_set_stream(self.ctx, stream)

    def close(self):
        if self.ctx:
            lbm_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def set_fields(self, populations, porosity=None, cell_flags=None):
        return lbm_set_fields(self.ctx, populations, porosity, cell_flags)

    def set_geometry(self, porosity=None, cell_flags=None):
        return lbm_set_geometry(self.ctx, porosity, cell_flags)

    def set_porosity(self, porosity=None):
        return lbm_set_porosity(self.ctx, porosity)

    def set_body_velocity(self, u_body=None):
        return lbm_set_body_velocity(self.ctx, u_body)

    def init_equilibrium(self, rho, u):
        return lbm_init_equilibrium(self.ctx, rho, u)

    def set_inflow(self, u_mean):
        return lbm_set_inflow(self.ctx, u_mean)

    def set_vortices(self, pos, sign, sigma_v, intensity):
        return lbm_set_vortices(self.ctx, pos, sign, sigma_v, intensity)

    def get_inflow(self, u):
        return lbm_get_inflow(self.ctx, u)

    def step(self, n_steps, params):
        return lbm_step(self.ctx, n_steps, params)

    def moments(self, rho, u):
        return lbm_moments(self.ctx, rho, u)

    def get_populations(self, populations):
        return lbm_get_populations(self.ctx, populations)

    def get_populations_box(self, origin, extent, populations):
        return lbm_get_populations_box(self.ctx, origin, extent, populations)

    def set_populations_box(self, origin, extent, populations):
        return lbm_set_populations_box(self.ctx, origin, extent, populations)

    def set_halo(self, ghost_lo, ghost_hi):
        return lbm_set_halo(self.ctx, ghost_lo, ghost_hi)

    def step_halo(self, params, stage):
        return lbm_step_halo(self.ctx, params, stage)

    def halo_pack(self, what, side, buf):
        return lbm_halo_pack(self.ctx, what, side, buf)

    def halo_unpack(self, what, side, buf):
        return lbm_halo_unpack(self.ctx, what, side, buf)

    def totals(self, out=None):
        return lbm_totals(self.ctx, out)

    def synchronize(self):
        return lbm_synchronize(self.ctx)

    def query(self, name):
        return lbm_query(self.ctx, self.QUERY[name])

    def set_option(self, key, value):
        return lbm_set_option(self.ctx, key, value)

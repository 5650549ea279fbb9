"""Seeded synthetic inputs for the LBM hot path (harness side; serves the oracle AND the CUDA path).

This module holds NONE of the method's arithmetic: it only writes macroscopic fields
(rho, u), the porosity field d, the flag field and the parameter set of each BASELINE.json
config.  Populations are obtained from (rho, u) by each side's own equilibrium routine
(oracle: orc_init_equilibrium; product: lbm_init_equilibrium).  The paper's own workloads need
city geometry, tree data and wind-tunnel data that are not available (PAPER.md refs [9], [34]);
these generators take their structure and stand in for them.

All randomness: numpy.random.Generator(numpy.random.PCG64(seed)), seed = 1000 + config number.
Array layouts: rho[nz,ny,nx], u[3,nz,ny,nx], d[nz,ny,nx] float64; flags[nz,ny,nx] uint8.
Flag byte: low nibble {0 FLUID, 1 SOLID, 2 INLET, 3 OUTLET, 4 WALLMODEL, 5 MOVINGWALL, 6 POUTLET, 7 SLIPWALL}; WALLMODEL carries the
wall-normal code in the high nibble {0:+x,1:-x,2:+y,3:-y,4:+z,5:-z}.
"""
import numpy as np

FLUID, SOLID, INLET, OUTLET, WALLMODEL, MOVINGWALL, POUTLET, SLIPWALL = 0, 1, 2, 3, 4, 5, 6, 7
WM_FLOOR = 0x44  # WALLMODEL with normal +z


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


# ------------------------------------------------------------------------------------------------
# config 1: 2-D Taylor-Green vortex extruded along z (reading R9)
# ------------------------------------------------------------------------------------------------
def taylor_green(nx, ny, nz, u0=0.05, modes=1):
    k = 2.0 * np.pi * modes / nx
    ky = 2.0 * np.pi * modes / ny
    x = np.arange(nx, dtype=np.float64)[None, None, :]
    y = np.arange(ny, dtype=np.float64)[None, :, None]
    one = np.ones((nz, 1, 1))
    u = np.zeros((3, nz, ny, nx))
    u[0] = u0 * np.sin(k * x) * np.cos(ky * y) * one
    u[1] = -u0 * np.cos(k * x) * np.sin(ky * y) * one
    rho = (1.0 - 0.75 * u0 * u0 * (np.cos(2 * k * x) + np.cos(2 * ky * y))) * one
    return rho, u


# ------------------------------------------------------------------------------------------------
# field F(N, k_max, M, rms): M divergence-free Fourier modes, shell energy ~ k^-5/3
# ------------------------------------------------------------------------------------------------
def spectral_modes(k_max, M, seed):
    """-> (k[M,3] int, e[M,3] unit polarisation with e.k = 0, phase[M], amp[M] = |k|^(-11/6))."""
    rng = _rng(seed)
    ks, es = [], []
    while len(ks) < M:
        k = rng.integers(-k_max, k_max + 1, size=3)
        k2 = int(k @ k)
        if k2 < 1 or k2 > k_max * k_max:
            continue
        r = rng.standard_normal(3)
        e = np.cross(k.astype(np.float64), r)
        n = np.linalg.norm(e)
        if n < 1e-8:
            continue
        ks.append(k)
        es.append(e / n)
    k = np.array(ks, dtype=np.int64)
    e = np.array(es)
    phase = rng.uniform(0.0, 2.0 * np.pi, size=M)
    amp = np.sqrt((k.astype(np.float64) ** 2).sum(axis=1)) ** (-11.0 / 6.0)
    return k, e, phase, amp


def spectral_field(shape, k_max, M, rms, seed):
    """u[3,nz,ny,nx] = sum_m a_m e_m cos(2 pi k_m.x/N + phi_m), rescaled to rms |u| = rms.

    Evaluated exactly through one inverse FFT per component (the field is a finite Fourier sum).
    The wave numbers count periods per box side along each axis."""
    import scipy.fft

    nz, ny, nx = shape
    k, e, phase, amp = spectral_modes(k_max, M, seed)
    u = np.empty((3, nz, ny, nx))
    for a in range(3):
        C = np.zeros((nz, ny, nx), dtype=np.complex128)
        coef = amp * e[:, a] * np.exp(1j * phase)
        np.add.at(C, (k[:, 2] % nz, k[:, 1] % ny, k[:, 0] % nx), coef)
        u[a] = scipy.fft.ifftn(C, workers=-1).real * (nz * ny * nx)
    cur = np.sqrt((u ** 2).sum(axis=0).mean())
    u *= rms / cur
    return u


# ------------------------------------------------------------------------------------------------
# geometry U(nx,ny,nz): urban channel (configs 3 and 5)
# ------------------------------------------------------------------------------------------------
def urban_channel(nx, ny, nz, seed, building_cover=0.15, tree_cover=0.05):
    """-> (flags[nz,ny,nx] uint8, d[nz,ny,nx] float64)."""
    rng = _rng(seed)
    flags = np.zeros((nz, ny, nx), dtype=np.uint8)
    d = np.zeros((nz, ny, nx))
    flags[0] = SOLID
    flags[nz - 1] = SOLID
    flags[1:nz - 1, :, 0] = INLET
    flags[1:nz - 1, :, nx - 1] = OUTLET
    x_lo = max(nx // 12, 1)
    x_hi = nx - max(nx // 6, 1)            # obstacles live in [x_lo, x_hi)
    # buildings: HLBM solids (d = 1), flag stays FLUID
    foot = np.zeros((ny, nx), dtype=bool)
    side_hi = max(min(32, (x_hi - x_lo) // 2, ny // 2), 2)
    side_lo = min(8, side_hi)
    h_hi = max(min(60, nz // 2), 2)
    h_lo = min(10, h_hi)
    guard = 0
    while foot.mean() < building_cover and guard < 100000:
        guard += 1
        sx = int(rng.integers(side_lo, side_hi + 1))
        sy = int(rng.integers(side_lo, side_hi + 1))
        h = int(rng.integers(h_lo, h_hi + 1))
        if x_hi - sx <= x_lo:
            continue
        x0 = int(rng.integers(x_lo, x_hi - sx + 1))
        y0 = int(rng.integers(0, ny))
        ys = (y0 + np.arange(sy)) % ny
        foot[np.ix_(ys, np.arange(x0, x0 + sx))] = True
        d[np.ix_(np.arange(1, min(1 + h, nz - 1)), ys, np.arange(x0, x0 + sx))] = 1.0
    # trees: porous blobs, one d per blob, written only where d is still 0
    z_top = max(min(40, nz // 3), 5)
    r_hi = max(min(8, nz // 6), 2)
    r_lo = min(3, r_hi)
    guard = 0
    zz, yy, xx = np.meshgrid(np.arange(-r_hi, r_hi + 1), np.arange(-r_hi, r_hi + 1),
                             np.arange(-r_hi, r_hi + 1), indexing="ij")
    dist2 = zz * zz + yy * yy + xx * xx
    porous = 0
    total = nx * ny * nz
    while porous < tree_cover * total and guard < 1000000:
        guard += 1
        r = rng.uniform(r_lo, r_hi)
        cx = rng.uniform(x_lo, x_hi)
        cy = rng.uniform(0, ny)
        cz = rng.uniform(4, z_top) if z_top > 4 else 4.0
        dv = rng.uniform(0.2, 0.6)
        ix, iy, iz = int(round(cx)), int(round(cy)), int(round(cz))
        m = dist2 <= r * r
        zs = iz + zz[m]
        ysel = (iy + yy[m]) % ny
        xs = ix + xx[m]
        ok = (zs >= 1) & (zs <= nz - 2) & (xs >= x_lo) & (xs < x_hi)
        zs, ysel, xs = zs[ok], ysel[ok], xs[ok]
        free = d[zs, ysel, xs] == 0.0
        d[zs[free], ysel[free], xs[free]] = dv
        porous += int(free.sum())
    # wall-model cells: every FLUID cell at z = 1 with d = 0 (reading R8 sets d := 1 there)
    wm = (flags[1] == FLUID) & (d[1] == 0.0)
    flags[1][wm] = WM_FLOOR
    d[1][wm] = 1.0
    return flags, d


# ------------------------------------------------------------------------------------------------
# config 4: random solid spheres in a periodic box
# ------------------------------------------------------------------------------------------------
def random_spheres(shape, seed, solid_fraction=0.10, r_lo=4.0, r_hi=12.0):
    nz, ny, nx = shape
    rng = _rng(seed)
    flags = np.zeros(shape, dtype=np.uint8)
    R = int(np.ceil(r_hi))
    zz, yy, xx = np.meshgrid(np.arange(-R, R + 1), np.arange(-R, R + 1), np.arange(-R, R + 1), indexing="ij")
    total = nx * ny * nz
    solid = 0
    guard = 0
    while solid < solid_fraction * total and guard < 10000000:
        guard += 1
        c = rng.uniform(0.0, 1.0, size=3) * np.array([nx, ny, nz])
        r = rng.uniform(r_lo, r_hi)
        i0 = np.floor(c).astype(int)
        fx, fy, fz = c - i0
        m = (xx - fx) ** 2 + (yy - fy) ** 2 + (zz - fz) ** 2 <= r * r
        zs = (i0[2] + zz[m]) % nz
        ys = (i0[1] + yy[m]) % ny
        xs = (i0[0] + xx[m]) % nx
        new = flags[zs, ys, xs] == FLUID
        solid += int(new.sum())
        flags[zs, ys, xs] = SOLID
    return flags


# ------------------------------------------------------------------------------------------------
# the BASELINE.json configs (optionally scaled down for tests)
# ------------------------------------------------------------------------------------------------
def make_config(number, shape=None, k_max=None, n_modes=None):
    """Return a dict: Q, dtype ('f32'/'f64'), shape (nz,ny,nx), steps, params (dict for lbm_params),
    rho, u, d (or None), flags (or None).  `shape` overrides the size for scaled-down tests;
    config 5 requires `shape`."""
    seed = 1000 + number
    tau_les = 0.5 + 3.0 * 1e-5      # nu = 1e-5 (configs 2 and 4)
    # configs 3 / 5 state no tau0.  With the wall-model coupling of reading R8 the run blows up (oracle and
    # CUDA path alike) for tau0 <= 0.505; 0.52 (nu = 6.7e-3) keeps all 2000 steps finite (G27).
    tau_urban = 0.52
    if number == 1:
        nz, ny, nx = shape or (32, 32, 32)
        rho, u = taylor_green(nx, ny, nz, u0=0.05)
        return dict(number=1, Q=19, dtype="f64", shape=(nz, ny, nx), steps=100, rho=rho, u=u, d=None, flags=None,
                    params=dict(tau0=0.6, cs_smago=0.0, use_hlbm=0))
    if number == 2:
        shape = shape or (256, 256, 256)
        u = spectral_field(shape, k_max or 32, n_modes or 256, 0.03, seed)
        return dict(number=2, Q=19, dtype="f32", shape=tuple(shape), steps=1000, rho=np.ones(shape), u=u, d=None,
                    flags=None, params=dict(tau0=tau_les, cs_smago=0.1, use_hlbm=0))
    if number in (3, 5):
        if number == 5 and shape is None:
            raise ValueError("config 5 is a sweep: pass shape")
        nz, ny, nx = shape or (128, 192, 384)
        flags, d = urban_channel(nx, ny, nz, seed)
        rho = np.ones((nz, ny, nx))
        u = np.zeros((3, nz, ny, nx))
        u[0][(flags & 0x0F) != SOLID] = 0.05
        return dict(number=number, Q=19, dtype="f32", shape=(nz, ny, nx), steps=2000 if number == 3 else 100,
                    rho=rho, u=u, d=d, flags=flags,
                    params=dict(tau0=tau_urban, cs_smago=0.1, use_hlbm=1, u_in=(0.05, 0.0, 0.0), wm_enable=1,
                                wm_kappa=0.41, wm_E=9.8))
    if number == 4:
        shape = shape or (512, 512, 512)
        flags = random_spheres(shape, seed)
        u = spectral_field(shape, k_max or 32, n_modes or 256, 0.03, seed + 500)
        u[:, (flags & 0x0F) == SOLID] = 0.0
        return dict(number=4, Q=27, dtype="f32", shape=tuple(shape), steps=200, rho=np.ones(shape), u=u, d=None,
                    flags=flags, params=dict(tau0=tau_les, cs_smago=0.12, use_hlbm=0))
    if number == 7:
        # the urban channel in the PAPER's boundary set (not a BASELINE.json config): config 3's
        # geometry with a fixed-pressure outlet + fringe zone, full-slip lateral walls (planes y = 0, ny-1) and top (z = nz-1),
        # wall-modelled bounce-back floor, velocity inlet (bench.py adds the Vortex Method to it)
        cfg = make_config(3, shape=shape)
        nz, ny, nx = cfg["shape"]
        fl = cfg["flags"]
        fl[(fl & 0x0F) == OUTLET] = POUTLET
        fl[nz - 1] = SLIPWALL
        fl[1:, 0] = SLIPWALL
        fl[1:, ny - 1] = SLIPWALL
        wall = is_wall(fl)
        cfg["d"][wall] = 0.0
        cfg["u"][:, wall] = 0.0
        cfg["number"] = 7
        cfg["params"] = dict(cfg["params"], rho_out=1.0, fringe_len=max(nx // 8, 1), fringe_factor=10.0)
        return cfg
    if number == 8:
        # config 7 with the wall model on the building faces as well ("wall-modelled"; SURVEY 8(f)-2 "wall model on
        # building faces of all six orientations"): every plain fluid cell (FLUID, d = 0) with a building cell (d = 1) as axis
        # neighbour becomes a WALLMODEL cell with the normal pointing away from that face (roofs first, then x, then y faces) and
        # d := 1 (reading R8), like the floor cells
        cfg = make_config(7, shape=shape)
        n_faces = wallmodel_faces(cfg["flags"], cfg["d"])
        cfg["number"] = 8
        cfg["wm_face_cells"] = n_faces
        return cfg
    if number == 6:
        # lid-driven cavity (the paper's scaling benchmark; not a BASELINE.json config):
        # closed box, five resting walls, the z = nz-1 plane moves with u_wall = (0.05, 0, 0); fluid at rest, rho = 1;
        # fp32 as in the paper ("base arithmetic type ... single-precision"); tau0 / Cs are this build's choice.
        shape = tuple(shape or (512, 512, 512))
        return dict(number=6, Q=19, dtype="f32", shape=shape, steps=200, rho=np.ones(shape), u=np.zeros((3,) + shape),
                    d=None, flags=cavity_flags(shape),
                    params=dict(tau0=0.52, cs_smago=0.1, use_hlbm=0, u_wall=(0.05, 0.0, 0.0)))
    raise ValueError("unknown config %r" % number)


def vm_inlet(shape, seed, n_vortices=256, sigma_v=6.0, intensity=0.15, u_ref=0.05, alpha=0.25):
    """Vortex Method inlet of the urban channel: an atmospheric power-law mean profile
    u_mean = u_ref ((z - 1/2)/(nz - 2))^alpha e_x over the floor z = 1/2 (stand-in for the paper's profile [23], which is not
    printed), seeded vortex positions (uniform over the inflow plane) and signs.  No method arithmetic: inputs only."""
    nz, ny, nx = shape
    rng = _rng(seed)
    u_mean = np.zeros((3, nz, ny))
    h = np.clip((np.arange(nz) - 0.5) / max(nz - 2, 1), 0.5 / max(nz - 2, 1), 1.0)
    u_mean[0] = (u_ref * h ** alpha)[:, None]
    pos = np.stack([rng.uniform(0.0, ny, n_vortices), rng.uniform(1.0, nz - 1.0, n_vortices)], axis=1)
    sign = rng.choice([-1.0, 1.0], n_vortices)
    return dict(u_mean=u_mean, pos=pos, sign=sign, sigma_v=float(sigma_v), intensity=float(intensity))


def body_velocity(cfg, seed, amp=0.02):
    """Solid velocity field u^B(x,t) of Eq. 12 for a workload: the partly porous cells
    (0 < d < 1: the trees of config 3) sway with a seeded smooth velocity (three plane waves per component), cells with d = 1
    (buildings) and d = 0 carry 0.  [3][nz][ny][nx] float64.  No method arithmetic: inputs only."""
    nz, ny, nx = cfg["shape"]
    rng = _rng(seed)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij", sparse=True)
    ub = np.zeros((3, nz, ny, nx))
    for a in range(3):
        for _ in range(3):
            k = rng.integers(1, 4, size=3)
            ph = rng.uniform(0.0, 2.0 * np.pi)
            ub[a] += (amp / 3.0) * np.sin(2.0 * np.pi * (k[0] * x / nx + k[1] * y / ny + k[2] * z / nz) + ph)
    d = cfg["d"]
    moving = (d > 0.0) & (d < 1.0) if d is not None else np.zeros((nz, ny, nx), dtype=bool)
    ub[:, ~moving] = 0.0
    return ub


def wallmodel_faces(flags, d):
    """Flag the plain fluid cells next to a building face (a FLUID cell with d = 1) as WALLMODEL cells, in place; the normal code
    {0:+x, 1:-x, 2:+y, 3:-y, 4:+z, 5:-z} points from the face into the fluid.  Returns the number of cells per normal code."""
    building = (d == 1.0) & ((flags & 0x0F) == FLUID)
    plain = (d == 0.0) & (flags == FLUID)
    taken = np.zeros_like(plain)
    cand = []
    # (normal code, axis, shift): the building lies at x - n, i.e. building rolled by +n along the axis
    order = [(4, 0, 1), (5, 0, -1), (0, 2, 1), (1, 2, -1), (2, 1, 1), (3, 1, -1)]
    for code, axis, sh in order:
        m = plain & ~taken & np.roll(building, sh, axis=axis)
        taken |= m
        cand.append(m)
    # the wall model samples the velocity at x + n: that cell must be plain fluid and not a candidate itself (a gap of one or two
    # cells between two buildings has no such point: two wall-model cells sampling each other feed back and blow up within 40 steps)
    free = plain & ~taken
    counts = {}
    chosen = np.zeros_like(plain)
    for (code, axis, sh), m in zip(order, cand):
        ok = m & np.roll(free, -sh, axis=axis)
        flags[ok] = WALLMODEL | (code << 4)
        chosen |= ok
        counts[code] = int(ok.sum())
    d[chosen] = 1.0
    return counts


def cavity_flags(shape):
    """closed box: SOLID on x = 0, nx-1, y = 0, ny-1, z = 0; MOVINGWALL on the whole plane z = nz-1 (the lid)"""
    flags = np.zeros(shape, dtype=np.uint8)
    flags[0] = SOLID
    flags[:, 0] = SOLID
    flags[:, -1] = SOLID
    flags[:, :, 0] = SOLID
    flags[:, :, -1] = SOLID
    flags[-1] = MOVINGWALL
    return flags


def is_wall(flags):
    """cells that are walls (resting SOLID or MOVINGWALL): inert, excluded from every comparison of fluid values"""
    t = flags & 0x0F
    return (t == SOLID) | (t == MOVINGWALL) | (t == SLIPWALL)

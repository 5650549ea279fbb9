"""Slab decomposition of the lattice in z over several contexts (Table 1): the
plumbing around lbm_set_halo / lbm_step_halo / lbm_halo_pack / lbm_halo_unpack.  No arithmetic of the method lives here: the
partition, the neighbour bookkeeping, the face buffers (torch tensors: device memory) and the transfer -- torch.distributed
send / recv between ranks (NCCL over NVLink between GPUs, gloo in the CPU tests of the host logic), or plain device copies between
several sub-domains held by ONE process on one GPU (`LocalGroup`, the single-GPU proof that the decomposed run equals the
undivided one).

Layout of a sub-domain: global slices [z0, z0 + count) plus one ghost slice below / above where the sub-domain has a neighbour
there.  A lattice that is closed in z (its planes z = 0 and z = nz-1 are walls throughout: channel floor / top, cavity bottom /
lid) has no neighbour across those planes; otherwise the z axis is periodic and the ranks form a ring.
"""
import numpy as np

from . import binding as B

POP, UHAT = B.LBM_HALO_POPULATIONS, B.LBM_HALO_UHAT
LOW, HIGH = B.LBM_SIDE_LOW, B.LBM_SIDE_HIGH


def partition(nz, world, min_slices=2):
    """[(z0, count)] per rank: contiguous, near-equal (the first nz % world ranks take one slice more)."""
    if world < 1 or nz < world * min_slices:
        raise ValueError("cannot cut %d slices into %d slabs of at least %d" % (nz, world, min_slices))
    base, extra = divmod(nz, world)
    out, z = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((z, n))
        z += n
    return out


def z_is_closed(flags):
    """True when the planes z = 0 and z = nz-1 are wall cells throughout (nothing crosses the periodic seam)."""
    if flags is None:
        return False
    t0, t1 = flags[0] & 0x0F, flags[-1] & 0x0F
    wall = lambda t: (t == 1) | (t == 5) | (t == 7)       # SOLID, MOVINGWALL, SLIPWALL
    return bool(wall(t0).all() and wall(t1).all())


class Slab:
    """One rank's share of the z axis and its neighbours."""

    def __init__(self, nz, rank, world, closed):
        self.nz, self.rank, self.world, self.closed = nz, rank, world, bool(closed)
        self.z0, self.count = partition(nz, world)[rank]
        if world == 1:
            self.lower = self.upper = None                 # undivided: the library's own periodic wrap serves the seam
        else:
            self.lower = rank - 1 if rank > 0 else (None if closed else world - 1)
            self.upper = rank + 1 if rank < world - 1 else (None if closed else 0)
        self.ghost_lo = 0 if self.lower is None else 1
        self.ghost_hi = 0 if self.upper is None else 1
        self.nz_local = self.count + self.ghost_lo + self.ghost_hi

    def local_z(self):
        """global z index of every local slice (ghost slices included, periodic wrap)"""
        return (np.arange(self.z0 - self.ghost_lo, self.z0 + self.count + self.ghost_hi)) % self.nz

    def take(self, arr, axis=0):
        """the local part (with ghost slices) of a global array whose z axis is `axis`"""
        return None if arr is None else np.ascontiguousarray(np.take(arr, self.local_z(), axis=axis))

    def interior(self):
        """slice object of the interior slices inside the local lattice"""
        return slice(self.ghost_lo, self.ghost_lo + self.count)


def exchange_faces(slab, send_low, send_high, recv_low, recv_high, group=None):
    """One halo exchange between ranks over torch.distributed: my low face goes to the lower neighbour (into its HIGH ghost), my
    high face to the upper one (into its LOW ghost).  Sends and receives are posted in one batch; between the same pair of ranks
    they match in posting order (and by tag where the backend has tags): data travelling DOWN first, then data travelling UP."""
    import torch.distributed as dist
    if send_low.is_cuda and dist.get_backend(group) == "gloo":
        # gloo moves host memory only (the CPU tests, and the single-GPU dry run of bench.py's decomposed path): stage through the host
        hs = [t.cpu() for t in (send_low, send_high, recv_low, recv_high)]
        exchange_faces(slab, hs[0], hs[1], hs[2], hs[3], group)
        if slab.lower is not None:
            recv_low.copy_(hs[2])
        if slab.upper is not None:
            recv_high.copy_(hs[3])
        return
    ops = []
    if slab.lower is not None:
        ops.append(dist.P2POp(dist.isend, send_low, slab.lower, group, 0))        # travels down
    if slab.upper is not None:
        ops.append(dist.P2POp(dist.isend, send_high, slab.upper, group, 1))       # travels up
    if slab.upper is not None:
        ops.append(dist.P2POp(dist.irecv, recv_high, slab.upper, group, 0))       # the upper neighbour's low face
    if slab.lower is not None:
        ops.append(dist.P2POp(dist.irecv, recv_low, slab.lower, group, 1))        # the lower neighbour's high face
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()


class SlabLBM:
    """A sub-domain: an LBM context of nz_local slices with ghost slices declared, its face buffers, and the stepping loop."""

    def __init__(self, lattice, nx, ny, nz_global, dtype, rank, world, closed, stream=None, group=None, device="cuda"):
        import torch
        self.slab = Slab(nz_global, rank, world, closed)
        self.sim = B.LBM(lattice, nx, ny, self.slab.nz_local, dtype, stream=stream)
        self.group = group
        self.dtype = dtype
        tdt = torch.float32 if dtype == "f32" else torch.float64
        self._buf = {}
        for what, key in ((POP, "halo_population_values"), (UHAT, "halo_uhat_values")):
            n = self.sim.query(key)
            self._buf[what] = {k: torch.empty(n, dtype=tdt, device=device) for k in ("send_low", "send_high", "recv_low", "recv_high")}
        self._halo_set = False

    # geometry and state of the LOCAL lattice (ghost slices included: copies of the neighbours' boundary slices)
    def set_fields(self, populations, porosity=None, cell_flags=None):
        self.sim.set_fields(populations, porosity, cell_flags)
        self._declare()

    def set_geometry(self, porosity=None, cell_flags=None):
        self.sim.set_geometry(porosity, cell_flags)

    def init_equilibrium(self, rho, u):
        self.sim.init_equilibrium(rho, u)
        self._declare()

    def _declare(self):
        if not self._halo_set:
            self.sim.set_halo(self.slab.ghost_lo, self.slab.ghost_hi)
            self._halo_set = True

    # the pieces of an exchange (LocalGroup drives them in lockstep over several sub-domains of one process)
    def pack(self, what):
        s, b = self.slab, self._buf[what]
        if s.lower is not None:
            self.sim.halo_pack(what, LOW, b["send_low"])
        if s.upper is not None:
            self.sim.halo_pack(what, HIGH, b["send_high"])

    def unpack(self, what):
        s, b = self.slab, self._buf[what]
        if s.lower is not None:
            self.sim.halo_unpack(what, LOW, b["recv_low"])
        if s.upper is not None:
            self.sim.halo_unpack(what, HIGH, b["recv_high"])

    def exchange(self, what):
        b = self._buf[what]
        self.pack(what)
        exchange_faces(self.slab, b["send_low"], b["send_high"], b["recv_low"], b["recv_high"], self.group)
        self.unpack(what)

    def step(self, n_steps, params):
        """n time steps of this rank's sub-domain, exchanging with the neighbouring ranks (every rank calls it)"""
        if self.slab.world == 1:
            return self.sim.step(n_steps, params)
        hrr = params.collision >= 1        # both HRR forms exchange u^ boundary slices in front of the fused step
        for _ in range(n_steps):
            self.sim.step_halo(params, 0)
            if hrr:
                self.exchange(UHAT)
            self.sim.step_halo(params, 1)
            self.exchange(POP)

    def close(self):
        self.sim.close()


class LocalGroup:
    """All sub-domains of a decomposition held by ONE process on one GPU: the halo transfer is a device copy between the face
    buffers.  The stages run in lockstep over the sub-domains, so nothing ever waits on another sub-domain inside a kernel."""

    def __init__(self, lattice, nx, ny, nz, dtype, world, closed, stream=None):
        self.parts = [SlabLBM(lattice, nx, ny, nz, dtype, r, world, closed, stream=stream) for r in range(world)]
        self.world = world

    def set_fields(self, populations, porosity=None, cell_flags=None):
        """global host arrays [Q][nz][ny][nx], [nz][ny][nx]: every sub-domain takes its slices (ghost slices included)"""
        for p in self.parts:
            p.set_fields(p.slab.take(populations, axis=1), p.slab.take(porosity), p.slab.take(cell_flags))

    def _exchange(self, what):
        for p in self.parts:
            p.pack(what)
        for p in self.parts:
            s, b = p.slab, p._buf[what]
            if s.upper is not None:
                b["recv_high"].copy_(self.parts[s.upper]._buf[what]["send_low"])
            if s.lower is not None:
                b["recv_low"].copy_(self.parts[s.lower]._buf[what]["send_high"])
        for p in self.parts:
            p.unpack(what)

    def step(self, n_steps, params):
        if self.world == 1:
            return self.parts[0].sim.step(n_steps, params)
        hrr = params.collision >= 1        # both HRR forms exchange u^ boundary slices in front of the fused step
        for _ in range(n_steps):
            for p in self.parts:
                p.sim.step_halo(params, 0)
            if hrr:
                self._exchange(UHAT)
            for p in self.parts:
                p.sim.step_halo(params, 1)
            self._exchange(POP)

    def get_populations(self, out):
        """assemble the global state S_t [Q][nz][ny][nx] (host numpy array) from the interiors"""
        for p in self.parts:
            loc = np.empty((out.shape[0], p.slab.nz_local) + out.shape[2:], dtype=out.dtype)
            p.sim.get_populations(loc)
            out[:, p.slab.z0:p.slab.z0 + p.slab.count] = loc[:, p.slab.interior()]
        return out

    def moments(self, rho, u):
        for p in self.parts:
            s = p.slab
            lr = np.empty((s.nz_local,) + rho.shape[1:], dtype=rho.dtype)
            lu = np.empty((3, s.nz_local) + rho.shape[1:], dtype=rho.dtype)
            p.sim.moments(lr, lu)
            rho[s.z0:s.z0 + s.count] = lr[s.interior()]
            u[:, s.z0:s.z0 + s.count] = lu[:, s.interior()]

    def totals(self):
        return np.sum([p.sim.totals() for p in self.parts], axis=0)

    def close(self):
        for p in self.parts:
            p.close()

"""Host logic of the slab decomposition (paper_2506_21804_b200/slab.py): partition, neighbours, ghost slices, the
indices a sub-domain takes from a global array, and the halo exchange over torch.distributed -- world sizes 2 and 3, gloo, CPU.
The exchange test emulates the pull across the cut: after one exchange every rank's ghost faces must hold exactly the boundary
slices of the neighbouring sub-domains of a global field cut along z (closed in z and periodic)."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2506_21804_b200 import slab as S  # noqa: E402


def test_partition_is_contiguous_balanced_and_complete():
    for nz in (8, 9, 31, 128, 513):
        for world in (1, 2, 3, 4, 8):
            if nz < 2 * world:
                with pytest.raises(ValueError):
                    S.partition(nz, world)
                continue
            parts = S.partition(nz, world)
            assert parts[0][0] == 0 and sum(n for _, n in parts) == nz
            assert all(parts[r][0] + parts[r][1] == parts[r + 1][0] for r in range(world - 1))
            counts = [n for _, n in parts]
            assert max(counts) - min(counts) <= 1 and min(counts) >= 2


def test_neighbours_and_ghost_slices():
    for closed in (True, False):
        for world in (2, 3, 5):
            slabs = [S.Slab(40, r, world, closed) for r in range(world)]
            for r, s in enumerate(slabs):
                assert s.ghost_lo == (0 if (closed and r == 0) else 1)
                assert s.ghost_hi == (0 if (closed and r == world - 1) else 1)
                if s.upper is not None:
                    assert slabs[s.upper].lower == r                    # neighbour relations are mutual
                if s.lower is not None:
                    assert slabs[s.lower].upper == r
                z = s.local_z()
                assert len(z) == s.nz_local == s.count + s.ghost_lo + s.ghost_hi
                assert list(z[s.interior()]) == list(range(s.z0, s.z0 + s.count))
                if s.ghost_lo:
                    assert z[0] == (s.z0 - 1) % 40
                if s.ghost_hi:
                    assert z[-1] == (s.z0 + s.count) % 40
    one = S.Slab(16, 0, 1, False)
    assert one.ghost_lo == one.ghost_hi == 0 and one.nz_local == 16 and one.lower is None and one.upper is None


def test_take_and_closed_detection():
    g = np.arange(10 * 3 * 4).reshape(10, 3, 4)
    s = S.Slab(10, 0, 3, False)                                         # periodic: the low ghost of rank 0 is the last slice
    loc = s.take(g)
    assert np.array_equal(loc[0], g[9]) and np.array_equal(loc[1:1 + s.count], g[:s.count]) and np.array_equal(loc[-1], g[s.count])
    f = np.arange(2 * 10 * 3 * 4).reshape(2, 10, 3, 4)
    assert np.array_equal(s.take(f, axis=1)[:, 0], f[:, 9])
    assert s.take(None) is None
    flags = np.zeros((6, 4, 4), dtype=np.uint8)
    assert not S.z_is_closed(flags) and not S.z_is_closed(None)
    flags[0] = 1
    flags[-1] = 5
    assert S.z_is_closed(flags)
    flags[-1, 2, 2] = 0
    assert not S.z_is_closed(flags)
    flags[-1] = 7
    flags[0] = 0x44
    assert not S.z_is_closed(flags)


def _worker(rank, world, port, closed, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    nz, plane = 6 * world + 1, 5
    # global field: value = 1000 z + k for plane element k; "down" faces carry it as is, "up" faces carry its negative, so a
    # face that lands in the wrong ghost is seen
    glob = 1000.0 * torch.arange(nz, dtype=torch.float64)[:, None] + torch.arange(plane, dtype=torch.float64)[None, :]
    s = S.Slab(nz, rank, world, closed)
    send_low = glob[s.z0].clone()                              # travels down: the first interior slice
    send_high = -glob[s.z0 + s.count - 1].clone()              # travels up: the last interior slice
    recv_low = torch.full((plane,), 7.0, dtype=torch.float64)
    recv_high = torch.full((plane,), 7.0, dtype=torch.float64)
    for _ in range(3):                                         # repeated exchanges stay matched
        S.exchange_faces(s, send_low, send_high, recv_low, recv_high)
    ok = True
    if s.upper is not None:
        ok = ok and torch.equal(recv_high, glob[(s.z0 + s.count) % nz])          # the upper neighbour's first slice, travelling down
    else:
        ok = ok and bool((recv_high == 7.0).all())
    if s.lower is not None:
        ok = ok and torch.equal(recv_low, -glob[(s.z0 - 1) % nz])                 # the lower neighbour's last slice, travelling up
    else:
        ok = ok and bool((recv_low == 7.0).all())
    dist.barrier()
    q.put((rank, bool(ok)))
    dist.destroy_process_group()


@pytest.mark.parametrize("world,closed,port", [(2, True, 29621), (2, False, 29622), (3, True, 29623), (3, False, 29624)])
def test_halo_exchange_over_gloo(world, closed, port):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, closed, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(r, True) for r in range(world)]

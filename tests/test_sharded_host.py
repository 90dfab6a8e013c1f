"""CPU tests of the host logic of the time-direction decomposition (paper_1311_4462_b200/sharded.py): slab geometry and the
ring exchange of the face buffers over torch.distributed (gloo, world size 2 and 3; no GPU, no kernels)."""
import os
import socket

import numpy as np
import pytest
import torch

import synth_inputs as si
from paper_1311_4462_b200 import sharded


def test_slab_geometry():
    assert sharded.slab_dims((8, 6, 4, 16), 2) == (8, 6, 4, 8)
    assert sharded.slab_dims((8, 6, 4, 16), 4) == (8, 6, 4, 4)
    for bad in (3, 8, 16):                      # odd split, slabs of 2 time slices, slabs of 1
        with pytest.raises(ValueError):
            sharded.slab_dims((8, 6, 4, 16), bad)
    # slabs are contiguous ranges of the lexicographic index and keep the global site parity
    dims, world = (4, 4, 4, 16), 2
    local = sharded.slab_dims(dims, world)
    for r in range(world):
        sl = sharded.slab_slice(dims, r, world)
        gp = np.zeros(si.volume(dims), dtype=int)
        gp[si.parity_sites(dims, 1)] = 1
        lp = np.zeros(si.volume(local), dtype=int)
        lp[si.parity_sites(local, 1)] = 1
        assert np.array_equal(gp[sl], lp)


def test_ring_exchange_world_1_is_the_periodic_wrap():
    a, b = torch.arange(6.0), torch.arange(6.0) + 10
    fp, fn = sharded.ring_exchange(a, b, 0, 1)
    assert torch.equal(fp, b) and torch.equal(fn, a)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        to_prev = torch.full((5,), 100.0 * rank + 1)          # what rank sends down / up the ring
        to_next = torch.full((5,), 100.0 * rank + 2)
        fp, fn = sharded.ring_exchange(to_prev, to_next, rank, world)
        q.put((rank, float(fp[0]), float(fn[0]), bool((fp == fp[0]).all() and (fn == fn[0]).all())))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_ring_exchange_gloo(world):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = {r: (fp, fn, ok) for r, fp, fn, ok in (q.get(timeout=120) for _ in range(world))}
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        fp, fn, ok = got[r]
        assert ok
        assert fp == 100.0 * ((r - 1) % world) + 2            # the previous slab's to_next
        assert fn == 100.0 * ((r + 1) % world) + 1            # the next slab's to_prev


def test_process_grid_geometry():
    """sub_sites / grid_coords / neighbours of a (py, pz, pt) grid: the sub-lattices tile the global lattice, keep the global
    site parity, and the neighbour tables are periodic rings per direction."""
    dims, grid = (4, 8, 12, 8), (2, 3, 2)
    world = 12
    assert sharded.grid_of(world, grid) == grid and sharded.grid_of(4) == (1, 1, 4)
    with pytest.raises(ValueError):
        sharded.grid_of(world, (2, 2, 2))
    local = sharded.sub_dims(dims, grid)
    assert local == (4, 4, 4, 4)
    with pytest.raises(ValueError):
        sharded.sub_dims((4, 8, 12, 8), (4, 1, 1))           # parts of 2 sites
    seen = np.zeros(si.volume(dims), dtype=int)
    gp = np.zeros(si.volume(dims), dtype=int)
    gp[si.parity_sites(dims, 1)] = 1
    lp = np.zeros(si.volume(local), dtype=int)
    lp[si.parity_sites(local, 1)] = 1
    for r in range(world):
        c = sharded.grid_coords(r, grid)
        assert sharded.grid_rank(c, grid) == r
        idx = sharded.sub_sites(dims, grid, c)
        seen[idx] += 1
        assert np.array_equal(gp[idx], lp)                  # local parity = global parity
    assert (seen == 1).all()
    # time slabs are the special case of the default grid
    assert np.array_equal(sharded.sub_sites(dims, (1, 1, 2), (0, 0, 1)), np.arange(si.volume(dims))[sharded.slab_slice(dims, 1, 2)])
    # neighbours: walking `n` steps forward in a direction returns to the start; prev / next are inverse
    for r in range(world):
        c = sharded.grid_coords(r, grid)
        for k, d in enumerate(sharded.DIRS):
            cc = list(c)
            cc[k] += 1
            nxt = sharded.grid_rank(cc, grid)
            cc[k] -= 2
            prev = sharded.grid_rank(cc, grid)
            back = list(sharded.grid_coords(nxt, grid))
            back[k] -= 1
            assert sharded.grid_rank(back, grid) == r
            assert (prev == nxt) == (grid[k] <= 2)


def _peer_worker(rank, world, port, q, n_iter):
    """The flag protocol of sharded.PeerRing between two processes, on CPU tensors in shared memory: 'pack' = write the face into
    the neighbour's receive buffer of slot epoch & 1, then the epoch into the neighbour's flag word; 'complete' = spin on the own
    flag word, then read.  Random delays on both sides; a slot that is overwritten before it was read, or read before it was
    written, shows up as a wrong payload."""
    import random
    import time
    import torch.distributed as dist
    import torch.multiprocessing as mp
    mp.set_sharing_strategy("file_system")
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ok, rnd = True, random.Random(rank)
    try:
        def allgather(obj):
            out = [None] * world
            dist.all_gather_object(out, obj)
            return out
        prev, nxt = (rank - 1) % world, (rank + 1) % world
        ring = sharded.PeerRing(rank, prev, nxt, 64, torch.float64, "cpu", allgather)
        dist.barrier()
        for it in range(n_iter):
            epoch, t = ring.begin()
            assert epoch == it + 1
            time.sleep(rnd.random() * 2e-3)
            t["to_prev"].fill_(1000.0 * rank + epoch + 0.25)          # what this rank sends down ...
            t["to_next"].fill_(1000.0 * rank + epoch + 0.5)           # ... and up the ring
            for name in ("flag_prev", "flag_next"):
                f, i = t[name]
                f[i] = epoch
            time.sleep(rnd.random() * 2e-3)
            for name, src, frac in (("wait_prev", prev, 0.5), ("wait_next", nxt, 0.25)):
                f, i = t[name]
                t0 = time.time()
                while int(f[i]) < epoch:
                    assert time.time() - t0 < 60, "flag never arrived"
                buf = t["from_prev" if name == "wait_prev" else "from_next"]
                ok = ok and bool((buf == 1000.0 * src + epoch + frac).all())
        dist.barrier()
        q.put((rank, ok, ring.epoch))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_peer_ring_flag_protocol_shared_memory(world):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    n_iter = 60
    procs = [ctx.Process(target=_peer_worker, args=(r, world, port, q, n_iter)) for r in range(world)]
    for p in procs:
        p.start()
    got = [q.get(timeout=180) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sorted(r for r, _, _ in got) == list(range(world))
    assert all(ok for _, ok, _ in got) and all(e == n_iter for _, _, e in got)


def test_peer_ring_single_rank_targets_are_its_own_buffers():
    ring = sharded.PeerRing(0, 0, 0, 8, torch.float32, "cpu", None)
    e1, t1 = ring.begin()
    e2, t2 = ring.begin()
    assert (e1, e2) == (1, 2)
    assert t1["to_prev"].data_ptr() == t1["from_next"].data_ptr() and t1["to_next"].data_ptr() == t1["from_prev"].data_ptr()
    assert t1["to_prev"].data_ptr() != t2["to_prev"].data_ptr()                  # double-buffered by epoch parity
    assert t1["flag_prev"][1] == t1["wait_next"][1] and t1["flag_next"][1] == t1["wait_prev"][1]
    assert {t1[k][1] for k in ("flag_prev", "flag_next")} | {t2[k][1] for k in ("flag_prev", "flag_next")} == {0, 1, 2, 3}

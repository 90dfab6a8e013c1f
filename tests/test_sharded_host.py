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

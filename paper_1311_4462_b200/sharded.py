"""Time-direction domain decomposition on top of the C-ABI (include/tm.h: tm_halo_pack / tm_halo_apply; SURVEY.md section 8f
NEXT-4): one slab X x Y x Z x T/world of the global lattice per rank (one process per GPU), face exchange
with torch.distributed point-to-point operations (NCCL over NVLink on GPUs; gloo in the CPU tests of the exchange logic).

Argument marshalling and the exchange only: projection, the U_4^dag multiply of the sent face, the interior kernels and the
completion of the boundary sites all run in the library's kernels.
"""
import torch

import paper_1311_4462_b200 as tm


def slab_dims(global_dims, world):
    """Local extents of one slab; T must split into even slabs of at least 4 time slices (local parity = global parity)."""
    X, Y, Z, T = (int(d) for d in global_dims)
    if T % world or (T // world) % 2 or T // world < 4:
        raise ValueError("T = %d does not split into %d even slabs of >= 4 time slices" % (T, world))
    return (X, Y, Z, T // world)


def slab_slice(global_dims, rank, world):
    """The slab's sites as a slice of the lexicographic site index (x4 is the slowest coordinate)."""
    X, Y, Z, T = (int(d) for d in global_dims)
    n = X * Y * Z * (T // world)
    return slice(rank * n, (rank + 1) * n)


def ring_exchange_start(to_prev, to_next, rank, world, group=None):
    """Post the sends of `to_prev` to rank-1 and `to_next` to rank+1 and the matching receives (periodic ring); returns a
    handle for ring_exchange_finish.  With NCCL the transfers are ordered after the work already queued on the current
    stream (the pack kernel) and run beside whatever is queued next (the interior kernel)."""
    if world == 1:          # the slab is its own neighbour
        return (to_next.clone(), to_prev.clone(), [])
    import torch.distributed as dist
    prev, nxt = (rank - 1) % world, (rank + 1) % world
    from_prev, from_next = torch.empty_like(to_next), torch.empty_like(to_prev)
    ops = [dist.P2POp(dist.isend, to_prev, prev, group, tag=1), dist.P2POp(dist.isend, to_next, nxt, group, tag=2),
           dist.P2POp(dist.irecv, from_next, nxt, group, tag=1), dist.P2POp(dist.irecv, from_prev, prev, group, tag=2)]
    if world == 2:          # both neighbours are the same rank: order the pairs so that sends and receives match by tag
        ops = [ops[0], ops[2], ops[1], ops[3]] if rank == 0 else [ops[2], ops[0], ops[3], ops[1]]
    return (from_prev, from_next, dist.batch_isend_irecv(ops))


def ring_exchange_finish(handle):
    """(from_prev, from_next) = (rank-1's to_next, rank+1's to_prev); later work on the current stream sees them."""
    from_prev, from_next, reqs = handle
    for req in reqs:
        req.wait()
    return from_prev, from_next


def ring_exchange(to_prev, to_next, rank, world, group=None):
    """Blocking form: all four tensors have one shape and dtype."""
    return ring_exchange_finish(ring_exchange_start(to_prev, to_next, rank, world, group))


class Slab:
    """One rank's part of a time-decomposed lattice: a Lattice on the local extents with open time hops."""

    def __init__(self, global_dims, rank, world, device=0, group=None):
        self.global_dims, self.rank, self.world, self.group = tuple(global_dims), int(rank), int(world), group
        self.dims = slab_dims(global_dims, world)
        self.lat = tm.Lattice(self.dims, device)
        tm.tm_set_open_time(self.lat.ctx, 1)
        self.device = torch.device("cuda", device)
        self._faces = {}

    def faces(self, prec, nf):
        key = (int(prec), int(nf))
        if key not in self._faces:
            n = tm.tm_halo_bytes(self.lat.ctx, prec, nf) // (8 if prec == tm.TM_DOUBLE else 4)
            dt = torch.float64 if prec == tm.TM_DOUBLE else torch.float32
            self._faces[key] = (torch.empty(n, dtype=dt, device=self.device), torch.empty(n, dtype=dt, device=self.device))
        return self._faces[key]

    def signs(self, p):
        """(sign_prev, sign_next): the time boundary condition where the face is the global boundary."""
        return (p.t_boundary if self.rank == 0 else 1, p.t_boundary if self.rank == self.world - 1 else 1)

    def pack(self, inp, gauge, parity, dagger):
        to_prev, to_next = self.faces(inp.prec, inp.nf)
        tm.tm_halo_pack(inp.h, gauge.h, parity, dagger, to_prev.data_ptr(), to_next.data_ptr())
        return to_prev, to_next

    def finish(self, out, from_prev, from_next, gauge, p, parity, dagger, kernel_type):
        sp, sn = self.signs(p)
        tm.tm_halo_apply(out.h, from_prev.data_ptr(), from_next.data_ptr(), gauge.h, p, parity, dagger, kernel_type, sp, sn)

    def dslash_apply(self, out, inp, x, gauge, p, parity, dagger, kernel_type):
        """The distributed form of tm.dslash_apply: faces out, interior kernel while they travel, boundary sites completed."""
        to_prev, to_next = self.pack(inp, gauge, parity, dagger)
        handle = ring_exchange_start(to_prev, to_next, self.rank, self.world, self.group)
        tm.dslash_apply(out, inp, x, gauge, p, parity, dagger, kernel_type)            # overlaps the transfer
        from_prev, from_next = ring_exchange_finish(handle)
        self.finish(out, from_prev, from_next, gauge, p, parity, dagger, kernel_type)

    def mat_pc(self, out_e, in_e, tmp_o, gauge, p, matpc_type, dagger=0):
        """LHS of Eq. 2.2 / 2.3 on the slab (same two launches as tm_mat_pc, each with its face exchange)."""
        if matpc_type == tm.TM_MATPC_SYM and dagger:
            raise NotImplementedError("sharded SYM dagger: apply tm.twist_apply and the two daggered hops explicitly")
        self.dslash_apply(tmp_o, in_e, None, gauge, p, tm.TM_ODD, dagger, tm.TM_TWIST_INV_DSLASH)
        self.dslash_apply(out_e, tmp_o, in_e, gauge, p, tm.TM_EVEN, dagger,
                          tm.TM_DSLASH_TWIST_XPAY if matpc_type == tm.TM_MATPC_ASYM else tm.TM_TWIST_INV_DSLASH_XPAY)

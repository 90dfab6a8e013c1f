"""Domain decomposition in y, z and t on top of the C-ABI (include/tm.h: tm_set_open_dirs / tm_halo_pack / tm_halo_apply;
SURVEY.md section 8f NEXT-4): one sub-lattice X x Y/py x Z/pz x T/pt of the global lattice per rank (one
process per GPU) on a process grid (py, pz, pt).  Two transports for the faces:
  * torch.distributed point-to-point operations (NCCL over NVLink on GPUs; gloo in the CPU tests): ring_exchange*;
  * peer-mapped receive buffers (PeerRing): every rank maps its neighbours' receive buffers and flag words with CUDA IPC, the
    pack kernel stores the faces straight into the neighbour's memory and publishes an epoch number there; the neighbour's
    completion kernel spins on that word.  No copy engine, no host synchronisation: pack = transport.

Argument marshalling and the exchange only: projection, the U^dag multiply of the sent face, the interior kernels and the
completion of the boundary sites all run in the library's kernels.
"""
import numpy as np
import torch

import paper_1311_4462_b200 as tm

DIRS = (1, 2, 3)          # y, z, t: the directions a lattice can be cut in (x carries the checkerboard index)


# ---- geometry ---------------------------------------------------------------------------------------------------------------
def grid_of(world, grid=None):
    """(py, pz, pt); default: time slabs."""
    g = (1, 1, int(world)) if grid is None else tuple(int(v) for v in grid)
    if len(g) != 3 or g[0] * g[1] * g[2] != world or min(g) < 1:
        raise ValueError("process grid %r does not have %d ranks" % (g, world))
    return g


def grid_coords(rank, grid):
    """rank = (ct * pz + cz) * py + cy  ->  (cy, cz, ct)."""
    py, pz, _ = grid
    return (rank % py, (rank // py) % pz, rank // (py * pz))


def grid_rank(coords, grid):
    py, pz, pt = grid
    cy, cz, ct = (coords[0] % py, coords[1] % pz, coords[2] % pt)
    return (ct * pz + cz) * py + cy


def sub_dims(global_dims, grid):
    """Local extents; every cut extent must split into even parts of at least 4 sites (local parity = global parity)."""
    dims = [int(d) for d in global_dims]
    for k, d in enumerate(DIRS):
        n = grid[k]
        if dims[d] % n or (dims[d] // n) % 2 or dims[d] // n < 4:
            raise ValueError("extent %d = %d does not split into %d even parts of >= 4 sites" % (d, dims[d], n))
        dims[d] //= n
    return tuple(dims)


def sub_sites(global_dims, grid, coords):
    """Global lexicographic site indices of the sub-lattice at grid position `coords`, in the sub-lattice's own lexicographic order."""
    X, Y, Z, T = (int(d) for d in global_dims)
    lx, ly, lz, lt = sub_dims(global_dims, grid)
    y0, z0, t0 = coords[0] * ly, coords[1] * lz, coords[2] * lt
    x = np.arange(lx)[None, None, None, :]
    y = (y0 + np.arange(ly))[None, None, :, None]
    z = (z0 + np.arange(lz))[None, :, None, None]
    t = (t0 + np.arange(lt))[:, None, None, None]
    return (x + X * (y + Y * (z + Z * t))).reshape(-1)


def slab_dims(global_dims, world):
    """Local extents of one time slab (the default grid)."""
    try:
        return sub_dims(global_dims, (1, 1, world))
    except ValueError:
        raise ValueError("T = %d does not split into %d even slabs of >= 4 time slices" % (global_dims[3], world))


def slab_slice(global_dims, rank, world):
    """A time slab's sites as a slice of the lexicographic site index (x4 is the slowest coordinate)."""
    X, Y, Z, T = (int(d) for d in global_dims)
    n = X * Y * Z * (T // world)
    return slice(rank * n, (rank + 1) * n)


# ---- transport 1: torch.distributed point-to-point ----------------------------------------------------------------------------
def neighbor_exchange_start(to_prev, to_next, me, prev, nxt, group=None, tag=0):
    """Post the sends of `to_prev` to rank `prev` and `to_next` to rank `nxt` and the matching receives; returns a handle for
    ring_exchange_finish.  With NCCL the transfers are ordered after the work already queued on the current stream (the pack
    kernel) and run beside whatever is queued next (the interior kernel)."""
    if prev == me and nxt == me:          # the sub-lattice is its own neighbour
        return (to_next.clone(), to_prev.clone(), [])
    import torch.distributed as dist
    from_prev, from_next = torch.empty_like(to_next), torch.empty_like(to_prev)
    ops = [dist.P2POp(dist.isend, to_prev, prev, group, tag=tag + 1), dist.P2POp(dist.isend, to_next, nxt, group, tag=tag + 2),
           dist.P2POp(dist.irecv, from_next, nxt, group, tag=tag + 1), dist.P2POp(dist.irecv, from_prev, prev, group, tag=tag + 2)]
    if prev == nxt:         # two ranks in this direction: order the pairs so that sends and receives match by tag
        ops = [ops[0], ops[2], ops[1], ops[3]] if me < prev else [ops[2], ops[0], ops[3], ops[1]]
    return (from_prev, from_next, dist.batch_isend_irecv(ops))


def ring_exchange_start(to_prev, to_next, rank, world, group=None):
    """The time-slab form: neighbours rank - 1 and rank + 1 on a periodic ring."""
    return neighbor_exchange_start(to_prev, to_next, rank, (rank - 1) % world, (rank + 1) % world, group)


def ring_exchange_finish(handle):
    """(from_prev, from_next) = (the previous rank's to_next, the next rank's to_prev); later work on the current stream sees them."""
    from_prev, from_next, reqs = handle
    for req in reqs:
        req.wait()
    return from_prev, from_next


def ring_exchange(to_prev, to_next, rank, world, group=None):
    """Blocking form: all four tensors have one shape and dtype."""
    return ring_exchange_finish(ring_exchange_start(to_prev, to_next, rank, world, group))


# ---- transport 2: peer-mapped receive buffers with flag words -------------------------------------------------------------------
def _share(t):
    """A picklable handle (bytes) of tensor `t` for another process on this node: CUDA IPC for device tensors, shared memory for
    CPU tensors (torch.multiprocessing's reductions)."""
    import torch.multiprocessing  # noqa: F401  (registers the tensor reductions with ForkingPickler)
    from multiprocessing.reduction import ForkingPickler
    if not t.is_cuda:
        t.share_memory_()
    return bytes(ForkingPickler.dumps(t))


def _open(handle):
    import pickle
    return pickle.loads(handle)


class PeerRing:
    """Receive buffers and flag words of one rank for one (direction, buffer key), double-buffered, and the views of the two
    neighbours' buffers.  Protocol per exchange (epoch e = 1, 2, ..., slot = e & 1):
        sender   : writes its to_prev face into prev.recv[slot]['from_next'] and its to_next face into next.recv[slot]['from_prev'],
                   then stores e to prev.flag[slot]['from_next'] and next.flag[slot]['from_prev'] (tm_halo_pack, release);
        receiver : waits until its own flag[slot][side] >= e (tm_halo_apply, acquire), then reads recv[slot][side].
    Slot reuse is safe without further handshakes: a rank packs epoch e + 2 only after its own completion of epoch e + 1, which
    waited for the neighbour's pack of e + 1, which the neighbour queued after its completion of epoch e (stream order).
    `allgather(obj) -> list` distributes the handles (torch.distributed.all_gather_object, or a local stand-in)."""

    SIDES = ("from_prev", "from_next")

    def __init__(self, me, prev, nxt, n_elems, dtype, device, allgather):
        self.me, self.prev, self.nxt, self.epoch = me, prev, nxt, 0
        self.recv = [{s: torch.zeros(n_elems, dtype=dtype, device=device) for s in self.SIDES} for _ in range(2)]
        self.flag = torch.zeros(4, dtype=torch.int32, device=device)          # [slot][side]
        mine = {"recv": self.recv, "flag": self.flag}
        if prev == me and nxt == me:
            self.peer = {me: mine}
        else:
            handles = allgather({"recv": [{s: _share(b[s]) for s in self.SIDES} for b in self.recv], "flag": _share(self.flag)})
            self.peer = {me: mine}
            for r in {prev, nxt} - {me}:
                self.peer[r] = {"recv": [{s: _open(h[s]) for s in self.SIDES} for h in handles[r]["recv"]], "flag": _open(handles[r]["flag"])}

    @staticmethod
    def flag_index(slot, side):
        return 2 * slot + PeerRing.SIDES.index(side)

    def begin(self):
        """Start the next exchange: returns (epoch, targets) with the tensors / flag indices the pack and completion kernels use."""
        self.epoch += 1
        slot = self.epoch & 1
        p, n, m = self.peer[self.prev], self.peer[self.nxt], self.peer[self.me]
        return self.epoch, {
            "to_prev": p["recv"][slot]["from_next"], "flag_prev": (p["flag"], self.flag_index(slot, "from_next")),
            "to_next": n["recv"][slot]["from_prev"], "flag_next": (n["flag"], self.flag_index(slot, "from_prev")),
            "from_prev": m["recv"][slot]["from_prev"], "wait_prev": (m["flag"], self.flag_index(slot, "from_prev")),
            "from_next": m["recv"][slot]["from_next"], "wait_next": (m["flag"], self.flag_index(slot, "from_next"))}


def _word_ptr(pair):
    t, i = pair
    return t.data_ptr() + 4 * i


# ---- one rank's sub-lattice ---------------------------------------------------------------------------------------------------
class Slab:
    """One rank's part of a decomposed lattice: a Lattice on the local extents with the cut directions open.
    grid = (py, pz, pt) (default: time slabs, (1, 1, world)); cut = the directions treated as cut (default: those with more than
    one rank, or time when there is a single rank: the sub-lattice is then its own neighbour).  peer = True: faces travel through
    peer-mapped buffers and flag words (PeerRing) instead of torch.distributed point-to-point operations."""

    def __init__(self, global_dims, rank, world, device=0, group=None, grid=None, cut=None, peer=False, host_sync=False):
        self.global_dims, self.rank, self.world, self.group = tuple(global_dims), int(rank), int(world), group
        self.grid = grid_of(world, grid)
        self.coords = grid_coords(self.rank, self.grid)
        self.dims = sub_dims(global_dims, self.grid)
        self.cut = tuple(cut) if cut is not None else (tuple(d for k, d in enumerate(DIRS) if self.grid[k] > 1) or (3,))
        self.lat = tm.Lattice(self.dims, device)
        tm.tm_set_open_dirs(self.lat.ctx, sum(1 << d for d in self.cut))
        self.device = torch.device("cuda", device)
        self.peer = bool(peer)
        # host_sync (with peer): no flag words; the ranks meet at a host barrier between the pack kernels and the completion kernels
        # instead.  For ranks that SHARE one GPU (tests), where a kernel spinning on a flag could starve the kernel that sets it.
        self.host_sync = bool(host_sync)
        self._faces, self._rings = {}, {}

    def sites(self):
        """Global lexicographic indices of this rank's sites (local lexicographic order)."""
        return sub_sites(self.global_dims, self.grid, self.coords)

    def neighbors(self, d):
        c = list(self.coords)
        k = DIRS.index(d)
        c[k] -= 1
        prev = grid_rank(c, self.grid)
        c[k] += 2
        return prev, grid_rank(c, self.grid)

    def faces(self, prec, nf, d=3):
        key = (int(prec), int(nf), int(d))
        if key not in self._faces:
            n = tm.tm_halo_bytes(self.lat.ctx, prec, nf, d) // (8 if prec == tm.TM_DOUBLE else 4)
            dt = torch.float64 if prec == tm.TM_DOUBLE else torch.float32
            self._faces[key] = (torch.empty(n, dtype=dt, device=self.device), torch.empty(n, dtype=dt, device=self.device))
        return self._faces[key]

    def ring(self, prec, nf, d):
        key = (int(prec), int(nf), int(d))
        if key not in self._rings:
            n = tm.tm_halo_bytes(self.lat.ctx, prec, nf, d) // (8 if prec == tm.TM_DOUBLE else 4)
            dt = torch.float64 if prec == tm.TM_DOUBLE else torch.float32
            prev, nxt = self.neighbors(d)

            def allgather(obj):
                import torch.distributed as dist
                out = [None] * self.world
                dist.all_gather_object(out, obj, group=self.group)
                return out
            self._rings[key] = PeerRing(self.rank, prev, nxt, n, dt, self.device, allgather)
        return self._rings[key]

    def signs(self, p, d=3):
        """(sign_prev, sign_next): the time boundary condition where the face is the global boundary; space is periodic."""
        if d != 3:
            return (1, 1)
        ct, pt = self.coords[2], self.grid[2]
        return (p.t_boundary if ct == 0 else 1, p.t_boundary if ct == pt - 1 else 1)

    def pack(self, inp, gauge, parity, dagger, d=3):
        to_prev, to_next = self.faces(inp.prec, inp.nf, d)
        tm.tm_halo_pack(inp.h, gauge.h, parity, dagger, to_prev.data_ptr(), to_next.data_ptr(), d)
        return to_prev, to_next

    def finish(self, out, from_prev, from_next, gauge, p, parity, dagger, kernel_type, d=3):
        sp, sn = self.signs(p, d)
        tm.tm_halo_apply(out.h, from_prev.data_ptr(), from_next.data_ptr(), gauge.h, p, parity, dagger, kernel_type, sp, sn, d)

    def dslash_apply(self, out, inp, x, gauge, p, parity, dagger, kernel_type):
        """The distributed form of tm.dslash_apply: faces out, interior kernel while they travel, boundary sites completed."""
        if self.peer:
            pending = []
            flags = not self.host_sync
            for d in self.cut:
                epoch, t = self.ring(inp.prec, inp.nf, d).begin()
                tm.tm_halo_pack(inp.h, gauge.h, parity, dagger, t["to_prev"].data_ptr(), t["to_next"].data_ptr(), d,
                                _word_ptr(t["flag_prev"]) if flags else None, _word_ptr(t["flag_next"]) if flags else None, epoch)
                pending.append((d, epoch, t))
            tm.dslash_apply(out, inp, x, gauge, p, parity, dagger, kernel_type)        # overlaps the neighbours' stores
            if self.host_sync:
                import torch.distributed as dist
                self.lat.sync()
                if self.world > 1:
                    dist.barrier(group=self.group)      # every rank's faces have landed
            for d, epoch, t in pending:
                sp, sn = self.signs(p, d)
                tm.tm_halo_apply(out.h, t["from_prev"].data_ptr(), t["from_next"].data_ptr(), gauge.h, p, parity, dagger, kernel_type,
                                 sp, sn, d, _word_ptr(t["wait_prev"]) if flags else None, _word_ptr(t["wait_next"]) if flags else None, epoch)
            if self.host_sync and self.world > 1:
                import torch.distributed as dist
                self.lat.sync()
                dist.barrier(group=self.group)          # every rank has read its faces: the slot may be reused two exchanges later
            return
        handles = []
        for d in self.cut:
            to_prev, to_next = self.pack(inp, gauge, parity, dagger, d)
            prev, nxt = self.neighbors(d)
            handles.append((d, neighbor_exchange_start(to_prev, to_next, self.rank, prev, nxt, self.group, tag=10 * d)))
        tm.dslash_apply(out, inp, x, gauge, p, parity, dagger, kernel_type)            # overlaps the transfers
        for d, h in handles:
            from_prev, from_next = ring_exchange_finish(h)
            self.finish(out, from_prev, from_next, gauge, p, parity, dagger, kernel_type, d)

    def mat_pc(self, out_e, in_e, tmp_o, gauge, p, matpc_type, dagger=0):
        """LHS of Eq. 2.2 / 2.3 on the sub-lattice (the launches of tm_mat_pc, each hopping term with its face exchange)."""
        if matpc_type == tm.TM_MATPC_SYM and dagger:
            # M^_sym^dag = 1 - kappa^2 D^dag_eo R^dag^-1_oo D^dag_oe R^dag^-1_ee (C7): the leading twist is local
            tm.twist_apply(out_e, in_e, p, 1, 1)
            self.dslash_apply(tmp_o, out_e, None, gauge, p, tm.TM_ODD, 1, tm.TM_TWIST_INV_DSLASH)
            self.dslash_apply(out_e, tmp_o, in_e, gauge, p, tm.TM_EVEN, 1, tm.TM_DSLASH_XPAY)
            return
        self.dslash_apply(tmp_o, in_e, None, gauge, p, tm.TM_ODD, dagger, tm.TM_TWIST_INV_DSLASH)
        self.dslash_apply(out_e, tmp_o, in_e, gauge, p, tm.TM_EVEN, dagger,
                          tm.TM_DSLASH_TWIST_XPAY if matpc_type == tm.TM_MATPC_ASYM else tm.TM_TWIST_INV_DSLASH_XPAY)

    # ---- the solver on the decomposed lattice (the paper's CG runs on many GPUs) -----------------------
    def allreduce_hook(self):
        """A tm.TM_ALLREDUCE_FN that sums the library's device scalars over the ranks with torch.distributed.all_reduce (NCCL) on
        the current stream; install with tm.tm_set_allreduce(self.lat.ctx, hook) and keep the reference."""
        group = self.group

        class _Words:
            def __init__(self, ptr, n):
                self.__cuda_array_interface__ = {"shape": (n,), "typestr": "<f8", "data": (int(ptr), False), "version": 2}

        def fn(dev_sums, n, stream, user):
            try:
                if self.world > 1:
                    import torch.distributed as dist
                    dist.all_reduce(torch.as_tensor(_Words(dev_sums, n), device=self.device), group=group)
                return 0
            except Exception:
                return 1
        return tm.TM_ALLREDUCE_FN(fn)

    def invert_cg(self, x_e, b_e, g_precise, g_sloppy, p, matpc_type, tol=1e-10, max_iter=10000, sloppy_precision=tm.TM_SINGLE, delta=0.1):
        """tm_invert_cg on this rank's part of the lattice: the operator is Slab.mat_pc (face exchange inside every hopping
        term), the dot products are summed over the ranks (allreduce_hook).  Every rank calls it with its part of b_e."""
        by_gauge = {g_precise.h.value if hasattr(g_precise.h, "value") else g_precise.h: g_precise}
        if g_sloppy is not None:
            by_gauge[g_sloppy.h.value if hasattr(g_sloppy.h, "value") else g_sloppy.h] = g_sloppy
        nf = x_e.nf

        class _F:                                  # a field the library hands to the callback: handle + what Slab.mat_pc reads
            def __init__(self, h, prec):
                self.h, self.prec, self.nf = h, prec, nf

        def op(out_e, in_e, tmp_o, g, pp, typ, dagger, user):
            try:
                gauge = by_gauge[g]
                self.mat_pc(_F(out_e, gauge.prec), _F(in_e, gauge.prec), _F(tmp_o, gauge.prec), gauge, pp.contents, typ, dagger)
                return 0
            except Exception:
                import traceback
                traceback.print_exc()
                return 1
        hook = self.allreduce_hook()
        tm.tm_set_allreduce(self.lat.ctx, hook)
        try:
            return tm.invert_cg(x_e, b_e, g_precise, g_sloppy, p, matpc_type, tol, max_iter, sloppy_precision, delta, op=tm.TM_CG_OP_FN(op))
        finally:
            tm.tm_set_allreduce(self.lat.ctx, None)

"""GPU parity of the domain decomposition in y, z, t (include/tm.h: tm_halo_pack / tm_halo_apply, tm_set_open_dirs) against the
oracle on the GLOBAL lattice.  One GPU: the slabs of a `world`-way split are processed one after the other in this process
(pack all, hand the face buffers over exactly as sharded.ring_exchange routes them, then interior kernel + completion per
slab), so no kernel ever waits for another rank; the transport itself is covered by tests/test_sharded_host.py (gloo)."""
import itertools

import numpy as np
import pytest

import oracle
import paper_1311_4462_b200 as tm
import synth_inputs as si
from gpu_util import TOL, PREC_NAME, rel_l2
from paper_1311_4462_b200 import sharded

pytestmark = pytest.mark.gpu

KAPPA = 0.1632
PRECS = [tm.TM_DOUBLE, tm.TM_SINGLE, tm.TM_HALF]


class Split:
    """The sub-lattices of one global lattice on a (py, pz, pt) process grid, all on one GPU, each with its part of the gauge field."""

    def __init__(self, dims, world, U, grid=None):
        self.dims, self.world, self.U = dims, world, U
        self.slabs = [sharded.Slab(dims, r, world, grid=grid) for r in range(world)]
        self.sl = [s.sites() for s in self.slabs]
        self._g = {}

    def gauge(self, r, prec, recon):
        key = (r, prec, recon)
        if key not in self._g:
            self._g[key] = self.slabs[r].lat.gauge(np.ascontiguousarray(self.U[:, self.sl[r]]), prec, recon)
        return self._g[key]

    def kernel(self, inp, x, p, parity, dagger, kt, prec, recon, nf):
        fin, fx, fout, faces = [], [], [], []
        for r, s in enumerate(self.slabs):
            fin.append(s.lat.field(prec, nf).upload(1 - parity, np.ascontiguousarray(inp[:, self.sl[r]])))
            fx.append(None if x is None else s.lat.field(prec, nf).upload(parity, np.ascontiguousarray(x[:, self.sl[r]])))
            fout.append(s.lat.field(prec, nf))
            faces.append({})
            for d in s.cut:
                to_prev, to_next = s.pack(fin[r], self.gauge(r, prec, recon), parity, dagger, d)
                faces[r][d] = (to_prev.clone(), to_next.clone())
        out = np.zeros_like(inp)
        for r, s in enumerate(self.slabs):
            g = self.gauge(r, prec, recon)
            tm.dslash_apply(fout[r], fin[r], fx[r], g, p, parity, dagger, kt)
            for d in s.cut:
                prev, nxt = s.neighbors(d)
                s.finish(fout[r], faces[prev][d][1], faces[nxt][d][0], g, p, parity, dagger, kt, d)      # = the exchange's routing
            s.lat.sync()
            out[:, self.sl[r]] = fout[r].download(parity)
        return out


_cache = {}


def split_for(dims, world, kind, seed, grid=None):
    key = (dims, world, kind, seed, grid)
    if key not in _cache:
        _cache[key] = Split(dims, world, si.gauge_field(dims, seed, kind), grid)
    return _cache[key]


@pytest.mark.parametrize("dims,world", [((4, 4, 4, 16), 2), ((4, 6, 4, 12), 3), ((6, 6, 6, 8), 1)])
@pytest.mark.parametrize("kw", [dict(mu=0.3, epsilon=0.0, twist_flavor=-1), dict(mu=0.15, epsilon=0.19, twist_flavor=0),
                                dict(mu=0.15, epsilon=0.19, twist_flavor=0, t_boundary=+1)], ids=["deg-", "ndeg", "ndeg-periodic"])
def test_h1_sharded_kernels_match_the_global_oracle(dims, world, kw):
    nf = 2 if kw["twist_flavor"] == 0 else 1
    sp = split_for(dims, world, "haar", 21)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    full_in, full_x = si.spinor_field(dims, nf, 22), si.spinor_field(dims, nf, 23)
    for parity, dagger, kt in itertools.product((0, 1), (0, 1), (0, 1, 2, 3, 4, 5)):
        inp = si.mask_parity(full_in, dims, 1 - parity)
        x = si.mask_parity(full_x, dims, parity)
        if kt < 4:
            want = oracle.kernel(inp, x, sp.U, po, parity, dagger, kt)
        else:
            want = oracle.hop_xpay(inp, x, sp.U, po, parity, dagger, -KAPPA ** 2 if kt == 4 else KAPPA)
        for prec in PRECS:
            recon = tm.TM_RECON_12 if prec != tm.TM_DOUBLE else tm.TM_RECON_18
            got = sp.kernel(inp, None if kt == 0 else x, pg, parity, dagger, kt, prec, recon, nf)
            assert rel_l2(got, want) <= TOL[prec], (PREC_NAME[prec], world, parity, dagger, kt)


@pytest.mark.parametrize("dims,grid", [((4, 4, 8, 8), (1, 2, 1)), ((4, 8, 4, 8), (2, 1, 1)), ((4, 4, 8, 8), (1, 2, 2)), ((6, 8, 8, 4), (2, 2, 1)),
                                       ((4, 12, 4, 8), (3, 1, 2)), ((8, 8, 8, 8), (1, 2, 2)), ((8, 16, 4, 8), (2, 1, 1))],
                         ids=["z2", "y2", "z2t2", "y2z2", "y3t2", "z2t2-tile-kernel", "y2-tile-kernel"])
@pytest.mark.parametrize("kw", [dict(mu=0.3, epsilon=0.0, twist_flavor=-1), dict(mu=0.15, epsilon=0.19, twist_flavor=0)], ids=["deg-", "ndeg"])
def test_h1b_spatial_and_mixed_splits_match_the_global_oracle(dims, grid, kw):
    """Cuts in non-temporal directions (the face gather is strided and flavor-aware) and in two directions at once:
    every kernel type, parity, dagger and precision against the oracle on the GLOBAL lattice, sub-lattices processed in turn.
    The last two cases have local extents 8 x 8 x 4 x 4 / 8 x 8 x 4 x 8, which the warp-per-tile half kernel covers (open z, t / y hops there)."""
    nf = 2 if kw["twist_flavor"] == 0 else 1
    world = grid[0] * grid[1] * grid[2]
    sp = split_for(dims, world, "haar", 31, grid)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    full_in, full_x = si.spinor_field(dims, nf, 32), si.spinor_field(dims, nf, 33)
    for parity, dagger, kt in itertools.product((0, 1), (0, 1), (0, 1, 2, 3, 4, 5)):
        inp = si.mask_parity(full_in, dims, 1 - parity)
        x = si.mask_parity(full_x, dims, parity)
        if kt < 4:
            want = oracle.kernel(inp, x, sp.U, po, parity, dagger, kt)
        else:
            want = oracle.hop_xpay(inp, x, sp.U, po, parity, dagger, -KAPPA ** 2 if kt == 4 else KAPPA)
        for prec in PRECS:
            recon = tm.TM_RECON_12 if prec != tm.TM_DOUBLE else tm.TM_RECON_18
            got = sp.kernel(inp, None if kt == 0 else x, pg, parity, dagger, kt, prec, recon, nf)
            assert rel_l2(got, want) <= TOL[prec], (PREC_NAME[prec], grid, parity, dagger, kt, rel_l2(got, want))


@pytest.mark.parametrize("cut", [(3,), (2,), (1, 2, 3)], ids=["t", "z", "yzt"])
def test_h5_peer_ring_flags_and_sym_dagger_world_1(cut):
    """The peer-buffer transport (PeerRing: the pack kernel stores into the receiver's buffer and publishes the epoch, the
    completion kernel waits on the flag word) with one rank, which is its own neighbour in every cut direction, so that both
    kernels run through the flag code in stream order; and Slab.mat_pc for every operator including the exact SYM adjoint."""
    dims = (4, 4, 4, 8)
    U = si.gauge_field(dims, 34, "haar")
    kw = dict(mu=0.15, epsilon=0.19, twist_flavor=0)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    psi_e = si.mask_parity(si.spinor_field(dims, 2, 35), dims, 0)
    for peer in (True, False):
        s = sharded.Slab(dims, 0, 1, cut=cut, peer=peer)
        for prec in PRECS:
            g = s.lat.gauge(U, prec, tm.TM_RECON_12)
            fin, ftmp, fout = s.lat.field(prec, 2).upload(0, psi_e), s.lat.field(prec, 2), s.lat.field(prec, 2)
            for rep in range(3):                  # epochs 1..: both buffer slots are used
                for typ, dagger in ((tm.TM_MATPC_ASYM, 0), (tm.TM_MATPC_ASYM, 1), (tm.TM_MATPC_SYM, 0), (tm.TM_MATPC_SYM, 1)):
                    s.mat_pc(fout, fin, ftmp, g, pg, typ, dagger)
                    s.lat.sync()
                    want = oracle.matpc_adjoint(psi_e, U, po, typ) if dagger else oracle.matpc(psi_e, U, po, typ, 0)
                    assert rel_l2(fout.download(0), want) <= TOL[prec], (PREC_NAME[prec], peer, typ, dagger, rep)
        if peer:
            ring = s.ring(tm.TM_HALF, 2, cut[0])
            assert ring.epoch == 3 * (2 + 2 + 2 + 2)          # two hopping terms per operator
            assert int(ring.flag.max().item()) == ring.epoch


def test_h2_sharded_mat_pc_world_1_and_8real():
    """Slab.mat_pc through ring_exchange itself (world = 1: the slab is its own neighbour) and 8-real links."""
    dims = (4, 4, 4, 8)
    U = si.gauge_field(dims, 24, "haar")
    kw = dict(mu=0.15, epsilon=0.19, twist_flavor=0)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    psi_e = si.mask_parity(si.spinor_field(dims, 2, 25), dims, 0)
    s = sharded.Slab(dims, 0, 1)
    for prec, recon in ((tm.TM_DOUBLE, tm.TM_RECON_8), (tm.TM_SINGLE, tm.TM_RECON_8), (tm.TM_HALF, tm.TM_RECON_12)):
        g = s.lat.gauge(U, prec, recon)
        fin, ftmp, fout = s.lat.field(prec, 2).upload(0, psi_e), s.lat.field(prec, 2), s.lat.field(prec, 2)
        for typ, dagger in ((tm.TM_MATPC_ASYM, 0), (tm.TM_MATPC_ASYM, 1), (tm.TM_MATPC_SYM, 0)):
            s.mat_pc(fout, fin, ftmp, g, pg, typ, dagger)
            s.lat.sync()
            want = oracle.matpc_adjoint(psi_e, U, po, typ) if dagger else oracle.matpc(psi_e, U, po, typ, 0)
            assert rel_l2(fout.download(0), want) <= TOL[prec], (PREC_NAME[prec], typ, dagger)


@pytest.mark.parametrize("extra", [[], ["--peer"]], ids=["sendrecv", "peer"])
def test_h3_torchrun_script_world_1(extra):
    """tests/run_sharded_torchrun.py (the multi-GPU check, NCCL) launched the way the driver launches bench.py, with one rank."""
    import os
    import socket
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "1", "--master-addr", "127.0.0.1",
                        "--master-port", str(port), os.path.join(root, "tests", "run_sharded_torchrun.py")] + extra,
                       capture_output=True, text=True, timeout=600, cwd=root)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    assert "sharded ok: world 1" in r.stdout


def test_h4_halo_api_sizes_and_error_paths():
    import torch
    dims = (4, 6, 4, 8)
    s = sharded.Slab(dims, 0, 1)
    lat, ctx = s.lat, s.lat.ctx
    vs2 = 4 * 6 * 4 // 2
    assert tm.tm_halo_bytes(ctx, tm.TM_DOUBLE, 1) == vs2 * 12 * 8
    assert tm.tm_halo_bytes(ctx, tm.TM_SINGLE, 2) == 2 * vs2 * 12 * 4
    assert tm.tm_halo_bytes(ctx, tm.TM_HALF, 2) == 2 * vs2 * 12 * 4          # half fields travel as float
    assert tm.tm_halo_bytes(ctx, 3, 1) == 0 and tm.tm_halo_bytes(ctx, tm.TM_DOUBLE, 3) == 0
    assert tm.tm_halo_bytes(ctx, tm.TM_DOUBLE, 1, 2) == (4 * 6 * 8 // 2) * 12 * 8 and tm.tm_halo_bytes(ctx, tm.TM_DOUBLE, 2, 1) == 2 * (4 * 4 * 8 // 2) * 12 * 8
    assert tm.tm_halo_bytes(ctx, tm.TM_DOUBLE, 1, 0) == 0 and tm.tm_halo_bytes(ctx, tm.TM_DOUBLE, 1, 4) == 0       # x is never cut
    U = si.gauge_field(dims, 26, "haar")
    g64, g32 = lat.gauge(U, tm.TM_DOUBLE, tm.TM_RECON_12), lat.gauge(U, tm.TM_SINGLE, tm.TM_RECON_12)
    f = lat.field(tm.TM_DOUBLE, 1)
    a, b = s.faces(tm.TM_DOUBLE, 1)
    p = tm.params(KAPPA, mu=0.1)
    for bad in (lambda: tm.tm_halo_pack(f.h, g32.h, 0, 0, a.data_ptr(), b.data_ptr()),                      # precision mismatch
                lambda: tm.tm_halo_pack(f.h, g64.h, 2, 0, a.data_ptr(), b.data_ptr()),                      # parity
                lambda: tm.tm_halo_pack(f.h, g64.h, 0, 0, 0, b.data_ptr()),                                 # NULL buffer
                lambda: tm.tm_halo_apply(f.h, a.data_ptr(), b.data_ptr(), g64.h, p, 0, 0, 7, 1, 1),         # kernel type
                lambda: tm.tm_halo_apply(f.h, a.data_ptr(), b.data_ptr(), g64.h, p, 0, 0, 0, 0, 1),         # boundary sign
                lambda: tm.tm_halo_apply(f.h, a.data_ptr(), b.data_ptr(), g64.h, p, 0, 0, 0, -1, 1, 2),     # antiperiodic in space
                lambda: tm.tm_halo_pack(f.h, g64.h, 0, 0, a.data_ptr(), b.data_ptr(), 0),                   # direction x
                lambda: tm.tm_set_open_dirs(ctx, 1)):                                                       # mask bit of x
        with pytest.raises(tm.TmError):
            bad()
    # open time hops off again: the context is an ordinary periodic / antiperiodic lattice
    psi = si.mask_parity(si.spinor_field(dims, 1, 27), dims, 0)
    po = oracle.params(dims, KAPPA, mu=0.1)
    fin, fout = lat.field(tm.TM_DOUBLE, 1).upload(0, psi), lat.field(tm.TM_DOUBLE, 1)
    tm.dslash_apply(fout, fin, None, g64, p, 1, 0, 0)
    lat.sync()
    open_result = fout.download(1)
    tm.tm_set_open_time(ctx, 0)
    tm.dslash_apply(fout, fin, None, g64, p, 1, 0, 0)
    lat.sync()
    want = oracle.kernel(psi, np.zeros_like(psi), U, po, 1, 0, 0)
    assert rel_l2(fout.download(1), want) <= 1e-12
    # with open time hops only the two boundary time slices differ from the closed lattice
    diff = np.abs(open_result - want).reshape(1, dims[3], -1).max(axis=2)[0]
    assert (diff[1:-1] < 1e-12).all() and diff[0] > 1e-3 and diff[-1] > 1e-3


@pytest.mark.parametrize("dims,grid", [((4, 4, 4, 16), (1, 1, 2)), ((4, 4, 8, 8), (1, 2, 2))], ids=["t2", "z2t2"])
def test_h6_sharded_half_tight_against_the_oracle_on_the_quantised_inputs(dims, grid):
    """T2d on the sharded path: the oracle is fed the inputs as stored (int16 + norms), which leaves the fp32 arithmetic and the
    output quantisation.  The completion kernel re-quantises the boundary sites (load, add the missing hops, store: a second
    rounding of at most 1/2 LSB of the new site norm), so boundary components may be off by up to ~2.5 LSB instead of 1.75."""
    from test_gpu_parity import _quantise_links, _quantise_spinor
    world = grid[0] * grid[1] * grid[2]
    sp = split_for(dims, world, "haar", 41, grid)
    Uq = _quantise_links(sp.U)
    kw = dict(mu=0.15, epsilon=0.19, twist_flavor=0)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    full_in, full_x = si.spinor_field(dims, 2, 42), si.spinor_field(dims, 2, 43)
    worst_l2 = worst_lsb = 0.0
    for parity, dagger, kt in itertools.product((0, 1), (0, 1), (0, 1, 2, 3)):
        inp, x = si.mask_parity(full_in, dims, 1 - parity), si.mask_parity(full_x, dims, parity)
        want = oracle.kernel(_quantise_spinor(inp), _quantise_spinor(x), Uq, po, parity, dagger, kt)
        got = sp.kernel(inp, None if kt == 0 else x, pg, parity, dagger, kt, tm.TM_HALF, tm.TM_RECON_18, 2)
        err = rel_l2(got, want)
        idx = si.parity_sites(dims, parity)
        w = want[:, idx].view(np.float64).reshape(2, len(idx), 24)
        g = got[:, idx].view(np.float64).reshape(2, len(idx), 24)
        lsb = np.abs(g - w) / (np.abs(w).max(axis=2, keepdims=True) / 32767.0 + 1e-300)
        worst_l2, worst_lsb = max(worst_l2, err), max(worst_lsb, float(lsb.max()))
        assert err <= 6e-5, (parity, dagger, kt, err)
        assert lsb.max() <= 2.75, (parity, dagger, kt, lsb.max())
    print("sharded half, quantised inputs: worst rel L2 %.2e, worst component %.2f LSB" % (worst_l2, worst_lsb))


def _ipc_worker(rank, world, port, q):
    """One process of H7: maps its neighbours' receive buffers with CUDA IPC (PeerRing), stores into them with ordinary device work,
    and checks what arrived in its own buffers after a HOST barrier (no kernel of one process ever waits for another process)."""
    import os
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ok = True
    try:
        torch.cuda.set_device(0)

        def allgather(obj):
            out = [None] * world
            dist.all_gather_object(out, obj)
            return out
        prev, nxt = (rank - 1) % world, (rank + 1) % world
        ring = sharded.PeerRing(rank, prev, nxt, 4096, torch.float32, torch.device("cuda", 0), allgather)
        dist.barrier()
        for it in range(4):                      # both buffer slots, twice
            epoch, t = ring.begin()
            t["to_prev"].fill_(1000.0 * rank + epoch + 0.25)
            t["to_next"].fill_(1000.0 * rank + epoch + 0.5)
            for name in ("flag_prev", "flag_next"):
                f, i = t[name]
                f[i] = epoch
            torch.cuda.synchronize()
            dist.barrier()                       # every rank's stores are complete
            ok = ok and bool((t["from_prev"] == 1000.0 * prev + epoch + 0.5).all()) and bool((t["from_next"] == 1000.0 * nxt + epoch + 0.25).all())
            ok = ok and int(t["wait_prev"][0][t["wait_prev"][1]]) == epoch and int(t["wait_next"][0][t["wait_next"][1]]) == epoch
            dist.barrier()                       # nobody overwrites a slot before everyone has read it
        q.put((rank, ok))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_h7_peer_buffers_map_across_processes_with_cuda_ipc(world):
    """The part of the peer-buffer transport that CPU tests cannot reach: the receive buffers and flag words of one PROCESS mapped
    into another with CUDA IPC (torch's tensor reductions through all_gather_object), routed as PeerRing routes them.  Two and three
    processes share this box's one GPU; they synchronise on the host only."""
    import socket
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_ipc_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = [q.get(timeout=300) for _ in range(world)]
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert sorted(r for r, _ in got) == list(range(world)) and all(ok for _, ok in got)


@pytest.mark.parametrize("extra", [["--peer", "--grid", "1,1,2", "--cg"], ["--peer", "--grid", "1,2,2"], ["--peer", "--grid", "2,1,2"]],
                         ids=["peer-t2-cg", "peer-z2t2", "peer-y2t2"])
def test_h8_two_and_four_processes_on_one_gpu(extra):
    """tests/run_sharded_torchrun.py with SEVERAL ranks, all on this box's one GPU (--one-gpu: gloo; the peer transport with host
    barriers in place of the flag words, so that no kernel waits for another process): every rank holds its sub-lattice in its own
    process, the pack kernels store the faces straight into the neighbour PROCESS's memory through CUDA IPC, and the gathered
    Eq. 2.2 / 2.3 / adjoint results match the oracle on the global lattice in all three precisions.  (The send / recv transport needs
    NCCL, which does not run two ranks on one GPU, and gloo does not move device tensors point to point: that transport is covered
    by the gloo ring tests on CPU tensors and by H3 with one rank.)"""
    import os
    import socket
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    n = 1
    for v in extra[extra.index("--grid") + 1].split(","):
        n *= int(v)
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n), "--master-addr", "127.0.0.1",
                        "--master-port", str(port), os.path.join(root, "tests", "run_sharded_torchrun.py"), "--one-gpu"] + extra,
                       capture_output=True, text=True, timeout=900, cwd=root)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    assert "sharded ok: world %d" % n in r.stdout
    if "--cg" in extra:                # the solver across two processes: operator callback + all-reduce hook (gloo on device scalars)
        assert "sharded cg ok" in r.stdout

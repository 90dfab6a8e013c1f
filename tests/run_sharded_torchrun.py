"""Multi-GPU check of the domain decomposition, one rank per GPU:

    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P tests/run_sharded_torchrun.py [--grid PY,PZ,PT] [--peer]

(default grid: time slabs (1, 1, N); --peer: faces through peer-mapped buffers and flag words instead of NCCL send / recv;
--one-gpu: every rank on cuda:0 over gloo, with --peer the ranks meet at host barriers instead of spinning on flag words;
--cg: also solve M^dag M x = b with Slab.invert_cg and check the gathered solution under the oracle's operator.)
Every rank cuts its sub-lattice out of the same seeded global inputs, applies the LHS of Eq. 2.2 and Eq. 2.3 through
paper_1311_4462_b200.sharded.Slab.mat_pc (NCCL face exchange), the slabs are gathered on rank 0 and compared with the oracle
on the global lattice (fp64 1e-12, fp32 1e-5, half 5e-3).  Test infrastructure: pytest runs it with N = 1 (test_gpu_sharded.py);
boxes with more GPUs run it with N > 1 by hand or from the driver.
"""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import paper_1311_4462_b200 as tm                      # noqa: E402
import synth_inputs as si                              # noqa: E402
from paper_1311_4462_b200 import sharded               # noqa: E402

TOL = {tm.TM_DOUBLE: 1e-12, tm.TM_SINGLE: 1e-5, tm.TM_HALF: 5e-3}


def main():
    rank, world, local = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1)), int(os.environ.get("LOCAL_RANK", 0))
    if "--one-gpu" in sys.argv:
        local = 0
        torch.cuda.set_device(0)
        dist.init_process_group("gloo")
    else:
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    grid = tuple(int(v) for v in sys.argv[sys.argv.index("--grid") + 1].split(",")) if "--grid" in sys.argv else (1, 1, world)
    peer = "--peer" in sys.argv
    one_gpu = "--one-gpu" in sys.argv          # all ranks on cuda:0, gloo, host barriers instead of flag words (tests on a 1-GPU box)
    dims, kappa = (8, 8 * grid[0], 8 * grid[1], 8 * grid[2]), 0.1632
    kw = dict(mu=0.15, epsilon=0.19, twist_flavor=0)
    U = si.gauge_field(dims, 31, "haar")
    psi_e = si.mask_parity(si.spinor_field(dims, 2, 32), dims, 0)
    slab = sharded.Slab(dims, rank, world, local, grid=grid, peer=peer, host_sync=one_gpu)
    sl = slab.sites()
    order = np.concatenate([sharded.sub_sites(dims, grid, sharded.grid_coords(r, grid)) for r in range(world)])
    pg = tm.params(kappa, **kw)
    worst = {}
    for prec in (tm.TM_DOUBLE, tm.TM_SINGLE, tm.TM_HALF):
        g = slab.lat.gauge(np.ascontiguousarray(U[:, sl]), prec, tm.TM_RECON_12)
        fin = slab.lat.field(prec, 2).upload(0, np.ascontiguousarray(psi_e[:, sl]))
        ftmp, fout = slab.lat.field(prec, 2), slab.lat.field(prec, 2)
        for typ, dagger in ((tm.TM_MATPC_ASYM, 0), (tm.TM_MATPC_SYM, 0), (tm.TM_MATPC_SYM, 1)):
            slab.mat_pc(fout, fin, ftmp, g, pg, typ, dagger)
            slab.lat.sync()
            mine = torch.from_numpy(fout.download(0).view(np.float64).copy())
            if not one_gpu:
                mine = mine.cuda()
            parts = [torch.empty_like(mine) for _ in range(world)] if rank == 0 else None
            dist.gather(mine, parts, dst=0)
            if rank == 0:
                import oracle
                got = np.empty_like(psi_e)
                got[:, order] = np.concatenate([p.cpu().numpy().view(np.complex128).reshape(2, -1, 4, 3) for p in parts], axis=1)
                po = oracle.params(dims, kappa, **kw)
                want = oracle.matpc_adjoint(psi_e, U, po, typ) if dagger else oracle.matpc(psi_e, U, po, typ, 0)
                err = float(np.linalg.norm(got - want) / np.linalg.norm(want))
                worst[(prec, typ, dagger)] = err
                assert err <= TOL[prec], (prec, typ, dagger, err)
    if "--cg" in sys.argv:
        # the solver on the decomposed lattice: M^dag M x = b with the distributed operator and the dot products summed over the ranks
        import oracle
        po = oracle.params(dims, kappa, **kw)
        typ = tm.TM_MATPC_SYM
        A = lambda v: oracle.matpc_adjoint(oracle.matpc(v, U, po, typ), U, po, typ)
        b = A(psi_e)
        gd = slab.lat.gauge(np.ascontiguousarray(U[:, sl]), tm.TM_DOUBLE, tm.TM_RECON_12)
        gs = slab.lat.gauge(np.ascontiguousarray(U[:, sl]), tm.TM_SINGLE, tm.TM_RECON_12)
        fb = slab.lat.field(tm.TM_DOUBLE, 2).upload(0, np.ascontiguousarray(b[:, sl]))
        fx = slab.lat.field(tm.TM_DOUBLE, 2)
        info = slab.invert_cg(fx, fb, gd, gs, pg, typ, tol=1e-9, max_iter=2000, sloppy_precision=tm.TM_SINGLE, delta=0.1)
        mine = torch.from_numpy(fx.download(0).view(np.float64).copy())
        if not one_gpu:
            mine = mine.cuda()
        parts = [torch.empty_like(mine) for _ in range(world)] if rank == 0 else None
        dist.gather(mine, parts, dst=0)
        if rank == 0:
            x = np.empty_like(psi_e)
            x[:, order] = np.concatenate([p.cpu().numpy().view(np.complex128).reshape(2, -1, 4, 3) for p in parts], axis=1)
            res = float(np.linalg.norm(A(x) - b) / np.linalg.norm(b))
            err = float(np.linalg.norm(x - psi_e) / np.linalg.norm(psi_e))
            assert info["converged"] and res <= 5e-9 and err <= 1e-6, (info, res, err)
            print("sharded cg ok: %d iterations, %d reliable updates, residual under the oracle's operator %.2e" % (info["iterations"], info["restarts"], res))
    if rank == 0:
        print("sharded ok: world %d, grid %s, %s, rel L2 %s" % (world, grid, "peer buffers" if peer else "send / recv", {k: "%.2e" % v for k, v in worst.items()}))
        print("sharded ok: world %d, rel L2 %s" % (world, {k: "%.2e" % v for k, v in worst.items()}))
    dist.destroy_process_group()


if __name__ == "__main__":
    main()

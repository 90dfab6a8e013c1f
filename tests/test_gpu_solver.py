"""GPU tests of the vector operations and the mixed-precision CG.

The CG is an iteration, but what it reaches has a plain definition: the solution of M^dag M x = b.  The tests build b
from a known psi_e with the ORACLE's operators, solve on the GPU, and check (a) the residual of the GPU's x under the
oracle's fp64 operator and (b) the distance to psi_e, for plain double and for double-single / double-half.
"""
import itertools

import numpy as np
import pytest

import oracle
import paper_1311_4462_b200 as tm
import synth_inputs as si
from gpu_util import Bench, rel_l2

pytestmark = pytest.mark.gpu

KAPPA = 0.1632
FLAVORS = [dict(mu=0.05, epsilon=0.0, twist_flavor=1), dict(mu=0.15, epsilon=0.19, twist_flavor=0)]


def nf_of(kw):
    return 2 if kw["twist_flavor"] == 0 else 1


@pytest.mark.parametrize("nf", [1, 2])
def test_s1_axpby_and_redot_match_numpy(nf):
    dims = (6, 6, 6, 6)                        # ragged last tile: the padding must not leak into the sums
    lat = tm.Lattice(dims)
    x = si.mask_parity(si.spinor_field(dims, nf, 31), dims, 0)
    y = si.mask_parity(si.spinor_field(dims, nf, 32), dims, 0)
    a, b = 0.37, -1.21
    for prec, tol in ((tm.TM_DOUBLE, 1e-14), (tm.TM_SINGLE, 1e-6), (tm.TM_HALF, 2e-4)):
        fx, fy, fz = lat.field(prec, nf).upload(0, x), lat.field(prec, nf).upload(0, y), lat.field(prec, nf)
        tm.field_axpby(fz, a, fx, b, fy)
        assert rel_l2(fz.download(0), a * x + b * y) <= tol
        tm.field_axpby(fy, a, fx, b, fy)       # in place
        assert rel_l2(fy.download(0), a * x + b * y) <= tol
        want = np.vdot(x, a * x + b * y).real
        assert abs(tm.field_redot(fx, fz) - want) <= max(tol, 1e-13) * 10 * np.linalg.norm(x) * np.linalg.norm(a * x + b * y)
        assert abs(tm.field_redot(fx, fx) - np.vdot(x, x).real) <= max(tol, 1e-13) * 10 * np.vdot(x, x).real
    # mixed precisions: double += a * sloppy ; sloppy = a * double
    for ps, tol in ((tm.TM_SINGLE, 1e-6), (tm.TM_HALF, 2e-4)):
        fd, fs = lat.field(tm.TM_DOUBLE, nf).upload(0, y), lat.field(ps, nf).upload(0, x)
        tm.field_axpby(fd, a, fs, 1.0, fd)
        assert rel_l2(fd.download(0), a * x + y) <= tol
        fs2 = lat.field(ps, nf)
        tm.field_axpby(fs2, b, fd)
        assert rel_l2(fs2.download(0), b * (a * x + y)) <= tol
    with pytest.raises(tm.TmError) as e:
        tm.field_axpby(lat.field(tm.TM_SINGLE, nf), 1.0, lat.field(tm.TM_HALF, nf))
    assert e.value.status == tm.TM_ERR_UNSUPPORTED


@pytest.mark.parametrize("kw", FLAVORS, ids=["deg", "ndeg"])
@pytest.mark.parametrize("typ", [tm.TM_MATPC_ASYM, tm.TM_MATPC_SYM], ids=["asym", "sym"])
def test_s2_cg_solves_the_normal_equations(kw, typ):
    dims = (4, 4, 4, 8)
    nf = nf_of(kw)
    U = si.gauge_field(dims, 1, "near_identity")
    bench = Bench(dims, U)
    lat = bench.lat
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    psi_e = si.mask_parity(si.spinor_field(dims, nf, 33), dims, 0)
    A = lambda v: oracle.matpc_adjoint(oracle.matpc(v, U, po, typ), U, po, typ)      # M^dag M, oracle, fp64
    b = A(psi_e)
    gd = bench.gauge(tm.TM_DOUBLE, tm.TM_RECON_12)
    fb = lat.field(tm.TM_DOUBLE, nf).upload(0, b)
    tol = 1e-10
    iters = {}
    for ps, delta in ((tm.TM_DOUBLE, 0.5), (tm.TM_SINGLE, 0.1), (tm.TM_HALF, 0.3)):
        gs = None if ps == tm.TM_DOUBLE else bench.gauge(ps, tm.TM_RECON_12)
        fx = lat.field(tm.TM_DOUBLE, nf).upload(0, b)          # content on entry is ignored
        info = tm.invert_cg(fx, fb, gd, gs, pg, typ, tol=tol, max_iter=4000, sloppy_precision=ps, delta=delta)
        assert info["converged"] and info["residual"] <= tol, (ps, info)
        x = fx.download(0)
        assert rel_l2(A(x), b) <= 5 * tol, (ps, info)           # residual under the ORACLE's operator
        assert rel_l2(x, psi_e) <= 1e-7, (ps, info)             # and the solution itself
        iters[ps] = info["iterations"]
    # the low-precision solvers may need more iterations, not many times more
    assert iters[tm.TM_SINGLE] <= 2 * iters[tm.TM_DOUBLE] + 20
    assert iters[tm.TM_HALF] <= 4 * iters[tm.TM_DOUBLE] + 40


def test_s3_cg_edge_cases():
    dims = (4, 4, 4, 8)
    U = si.gauge_field(dims, 1, "near_identity")
    bench = Bench(dims, U)
    lat = bench.lat
    pg = tm.params(KAPPA, 0.05)
    gd = bench.gauge(tm.TM_DOUBLE, tm.TM_RECON_18)
    gs = bench.gauge(tm.TM_SINGLE, tm.TM_RECON_18)
    fb, fx = lat.field(tm.TM_DOUBLE, 1), lat.field(tm.TM_DOUBLE, 1)
    info = tm.invert_cg(fx, fb, gd, gs, pg, tm.TM_MATPC_ASYM)              # b = 0 -> x = 0, no iterations
    assert info["converged"] and info["iterations"] == 0 and np.abs(fx.download(0)).max() == 0
    b = si.mask_parity(si.spinor_field(dims, 1, 34), dims, 0)
    fb.upload(0, b)
    info = tm.invert_cg(fx, fb, gd, gs, pg, tm.TM_MATPC_ASYM, tol=1e-12, max_iter=3)   # iteration cap
    assert not info["converged"] and info["iterations"] == 3 and info["residual"] > 1e-12

    def status(fn):
        with pytest.raises(tm.TmError) as e:
            fn()
        return e.value.status
    assert status(lambda: tm.invert_cg(fx, fx, gd, gs, pg, tm.TM_MATPC_ASYM)) == tm.TM_ERR_ALIAS
    assert status(lambda: tm.invert_cg(fx, fb, gs, gs, pg, tm.TM_MATPC_ASYM)) == tm.TM_ERR_MISMATCH
    assert status(lambda: tm.invert_cg(fx, fb, gd, None, pg, tm.TM_MATPC_ASYM)) == tm.TM_ERR_MISMATCH
    assert status(lambda: tm.invert_cg(fx, fb, gd, gs, pg, tm.TM_MATPC_ASYM, delta=1.5)) == tm.TM_ERR_ARG


@pytest.mark.parametrize("kw,typ", [(FLAVORS[0], tm.TM_MATPC_SYM), (FLAVORS[1], tm.TM_MATPC_ASYM)], ids=["deg-sym", "ndeg-asym"])
def test_s4_cg_16c16_reliable_updates_and_workspace_reuse(kw, typ):
    """16^4 (beyond the 4^3 x 8 toy): the solution of every precision mix has residual <= 5 tol under the ORACLE's
    fp64 M^dag M; reliable updates keep one recurrence going (the sloppy solvers need about as many iterations as plain double,
    where defect-correction restarts needed many more); the work fields live on the context: no device allocation after the
    first solve of a precision mix."""
    import torch
    dims = (16, 16, 16, 16)
    nf = nf_of(kw)
    U = si.gauge_field(dims, 36, "near_identity")
    bench = Bench(dims, U)
    lat = bench.lat
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    A = lambda v: oracle.matpc_adjoint(oracle.matpc(v, U, po, typ), U, po, typ)
    psi_e = si.mask_parity(si.spinor_field(dims, nf, 37), dims, 0)
    b = A(psi_e)
    gd = bench.gauge(tm.TM_DOUBLE, tm.TM_RECON_12)
    fb = lat.field(tm.TM_DOUBLE, nf).upload(0, b)
    fx = lat.field(tm.TM_DOUBLE, nf)
    tol, iters = 1e-9, {}
    for ps, delta in ((tm.TM_DOUBLE, 0.1), (tm.TM_SINGLE, 0.1), (tm.TM_HALF, 0.3)):
        gs = None if ps == tm.TM_DOUBLE else bench.gauge(ps, tm.TM_RECON_12)
        info = tm.invert_cg(fx, fb, gd, gs, pg, typ, tol=tol, max_iter=5000, sloppy_precision=ps, delta=delta)
        assert info["converged"] and info["residual"] <= tol, (ps, info)
        x = fx.download(0)
        assert rel_l2(A(x), b) <= 5 * tol, (ps, info)
        assert rel_l2(x, psi_e) <= 1e-6, (ps, info)
        iters[ps] = info
        lat.sync()
        free0 = torch.cuda.mem_get_info()[0]
        again = tm.invert_cg(fx, fb, gd, gs, pg, typ, tol=tol, max_iter=5000, sloppy_precision=ps, delta=delta)
        lat.sync()
        assert torch.cuda.mem_get_info()[0] == free0                     # the second solve allocates nothing
        assert again["iterations"] == info["iterations"] and again["residual"] == info["residual"]      # and is deterministic
    print("16^4 iterations / reliable updates:", {k: (v["iterations"], v["restarts"]) for k, v in iters.items()})
    assert iters[tm.TM_SINGLE]["iterations"] <= 1.15 * iters[tm.TM_DOUBLE]["iterations"] + 5
    assert iters[tm.TM_HALF]["iterations"] <= 1.6 * iters[tm.TM_DOUBLE]["iterations"] + 10
    tm.tm_cg_release(lat.ctx)
    lat.sync()


def test_s5_cg_on_the_decomposed_lattice_world_1():
    """Slab.invert_cg: the solver with the distributed operator (face exchange inside every hopping term, through the peer-buffer
    transport) and the dot products passed through the all-reduce hook; one rank that is its own neighbour in z and t.  The
    solution equals the undecomposed solver's and solves the oracle's normal equations."""
    from paper_1311_4462_b200 import sharded
    dims = (8, 8, 8, 8)
    kw = FLAVORS[1]
    U = si.gauge_field(dims, 38, "near_identity")
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    typ = tm.TM_MATPC_SYM
    A = lambda v: oracle.matpc_adjoint(oracle.matpc(v, U, po, typ), U, po, typ)
    b = A(si.mask_parity(si.spinor_field(dims, 2, 39), dims, 0))
    s = sharded.Slab(dims, 0, 1, cut=(2, 3), peer=True)
    lat = s.lat
    gd, gs = lat.gauge(U, tm.TM_DOUBLE, tm.TM_RECON_12), lat.gauge(U, tm.TM_SINGLE, tm.TM_RECON_12)
    fb, fx = lat.field(tm.TM_DOUBLE, 2).upload(0, b), lat.field(tm.TM_DOUBLE, 2)
    n0 = lat.launches()
    info = s.invert_cg(fx, fb, gd, gs, pg, typ, tol=1e-9, max_iter=2000, sloppy_precision=tm.TM_SINGLE, delta=0.1)
    assert info["converged"], info
    x = fx.download(0)
    assert rel_l2(A(x), b) <= 5e-9, info
    assert lat.launches() - n0 > info["iterations"] * (4 + 2 * 4 * 2)      # 4 hopping terms, each with 2 directions x (pack + completion)
    plain = tm.Lattice(dims)
    gd2, gs2 = plain.gauge(U, tm.TM_DOUBLE, tm.TM_RECON_12), plain.gauge(U, tm.TM_SINGLE, tm.TM_RECON_12)
    fb2, fx2 = plain.field(tm.TM_DOUBLE, 2).upload(0, b), plain.field(tm.TM_DOUBLE, 2)
    info2 = tm.invert_cg(fx2, fb2, gd2, gs2, pg, typ, tol=1e-9, max_iter=2000, sloppy_precision=tm.TM_SINGLE, delta=0.1)
    assert abs(info2["iterations"] - info["iterations"]) <= 2
    assert rel_l2(x, fx2.download(0)) <= 1e-7

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

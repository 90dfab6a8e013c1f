"""Full-size GPU parity (BASELINE.json configs[1..4]) in the launch configuration bench.py times.

At 32^3x64 (configs[2], configs[3]: the lattice bench.py times) the composites are compared with the oracle on the WHOLE
lattice (the oracle needs well under a second per composite on the GPU box's host cores): relative L2 over the output field
with the north_star tolerances, and the largest component error of any site in units of that site's norm (MAXC below),
so that a defect confined to a few sites cannot hide in the L2 norm.  At 24^3x48 kernels, 48^3x96 and 64^4 the outputs are
SAMPLED: the oracle computes the composite (or the kernel) at a few thousand seeded output sites one by one
(oracle.matpc_sites / oracle.kernel_sites), always including the lattice corners and the first / last time slice where the
periodic wrap and the antiperiodic time sign act (relative L2 over the sampled sites).  Properties that hold at any size are checked on the whole field:
the other parity stays untouched and finite, and repeated application is bit-for-bit reproducible.

configs[4] (48^3x96, "applied 100 times back to back") is `test_config5_...` (~25 GB of host memory, about a minute on the
B200 box); `test_64c64_...` is the maximum-size case of the addressing (gauge parity blocks beyond 4 GiB, ~35 GB of host
memory, half a minute).  Both run by default and are skipped only when the host is short of memory or TM_TEST_HUGE=0.
"""
import os

import numpy as np
import pytest

import oracle
import paper_1311_4462_b200 as tm
import synth_inputs as si
from gpu_util import TOL, PREC_NAME

pytestmark = pytest.mark.gpu

KAPPA = 0.1632
N_SAMPLE = 2048
# largest |got - want| of a site's 12 (x flavors) components over that site's norm: fp64 / fp32 rounding of a ~1400-flop sum;
# half: the inputs are quantised to 1 / 32767 of their site norms and the output once more (measured 2.5e-4 on these configs)
# (measured 2.1e-14 / 1.3e-7 / 4.5e-5 with 12- and 18-real links).  8-real links: the rebuild's error grows like eps / N towards
# the chart's singular point (tm_gauge_load bounds N per precision); measured 7.8e-14 / 1.4e-5 / 7.5e-4 on the Haar field
MAXC = {tm.TM_DOUBLE: 1e-13, tm.TM_SINGLE: 1e-6, tm.TM_HALF: 2e-4}
MAXC8 = {tm.TM_DOUBLE: 1e-12, tm.TM_SINGLE: 1e-4, tm.TM_HALF: 5e-3}


def sample_sites(dims, parity, seed, n=N_SAMPLE):
    """Seeded lexicographic output sites of `parity`: random ones plus every lattice corner / boundary slice."""
    X, Y, Z, T = dims
    rng = np.random.Generator(np.random.Philox(key=[seed, 99]))
    all_p = si.parity_sites(dims, parity)
    pick = set(int(s) for s in rng.choice(all_p, size=n, replace=False))
    edge = [0, 1, X - 2, X - 1]
    for t in (0, T - 1):
        for z in (0, Z - 1):
            for y in (0, Y - 1):
                for x in edge:
                    if (x + y + z + t) % 2 == parity:
                        pick.add(x + X * (y + Y * (z + Z * t)))
    pick.add(int(all_p[-1]))
    pick.add(int(all_p[0]))
    return np.array(sorted(pick), dtype=np.int64)


def rel_l2_sites(got_full, want_sites, sites):
    got = got_full[:, sites].transpose(1, 0, 2, 3)
    return float(np.linalg.norm((got - want_sites).ravel()) / np.linalg.norm(want_sites.ravel()))


class Case:
    def __init__(self, dims, kind, seed, nf):
        self.dims, self.nf = dims, nf
        self.U = si.gauge_field(dims, seed, kind)
        self.psi_e = si.mask_parity(si.spinor_field(dims, nf, seed), dims, 0)
        self.lat = tm.Lattice(dims)
        self._want = {}

    def full_oracle(self, po, kw, typ, dagger):
        key = (tuple(sorted(kw.items())), typ, dagger)
        if key not in self._want:
            self._want[key] = oracle.matpc_adjoint(self.psi_e, self.U, po, typ) if dagger else oracle.matpc(self.psi_e, self.U, po, typ, 0)
        return self._want[key]

    def check_matpc(self, kw, prec, recon, typ, dagger, seed, full=False):
        lat, nf, dims = self.lat, self.nf, self.dims
        po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
        g = lat.gauge(self.U, prec, recon)
        fin = lat.field(prec, nf).upload(tm.TM_EVEN, self.psi_e)
        ftmp, fout = lat.field(prec, nf), lat.field(prec, nf)
        n0 = lat.launches()
        tm.mat_pc(fout, fin, ftmp, g, pg, typ, dagger)
        lat.sync()
        assert lat.launches() - n0 == 2                       # two fused launches, nothing else on the path
        got = fout.download(tm.TM_EVEN)
        if full:
            want = self.full_oracle(po, kw, typ, dagger)
            ev = si.parity_sites(dims, 0)
            d, w = (got - want)[:, ev], want[:, ev]
            err = float(np.linalg.norm(d.ravel()) / np.linalg.norm(w.ravel()))
            site_norm = np.sqrt((np.abs(w) ** 2).sum(axis=(0, 2, 3)))                       # per site, both flavors together
            maxc = float((np.abs(d).max(axis=(0, 2, 3)) / site_norm).max())
            print("full lattice: rel L2 %.3e, max component error / site norm %.3e" % (err, maxc))
            assert maxc <= (MAXC8 if recon == tm.TM_RECON_8 else MAXC)[prec], (PREC_NAME[prec], recon, typ, dagger, maxc)
        else:
            sites = sample_sites(dims, 0, seed)
            want = oracle.matpc_sites(sites, self.psi_e, self.U, po, typ, dagger)
            err = rel_l2_sites(got, want, sites)
        assert err <= TOL[prec], (PREC_NAME[prec], recon, typ, dagger, err)
        assert np.isfinite(got.view(np.float64)).all()
        assert np.abs(got[:, si.parity_sites(dims, 1)]).max() == 0
        # reproducibility: a second application gives the same bits
        first = fout.storage.clone()
        tm.mat_pc(fout, fin, ftmp, g, pg, typ, dagger)
        lat.sync()
        assert bool((first == fout.storage).all())
        return err


@pytest.fixture(scope="module")
def case2():
    return Case((24, 24, 24, 48), "near_identity", 2, 1)


@pytest.fixture(scope="module")
def case3():
    return Case((32, 32, 32, 64), "haar", 3, 1)


@pytest.fixture(scope="module")
def case4():
    return Case((32, 32, 32, 64), "near_identity", 4, 2)


def test_config2_24c48_fp32_18real_kernels_plain_and_dagger(case2):
    """configs[1]: kernels R_oo^-1 D_oe and (R_ee - kappa^2 D_eo), plain and dagger, 18-real, fp32."""
    c, dims = case2, case2.dims
    kw = dict(mu=0.004, epsilon=0.0, twist_flavor=1)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    g = c.lat.gauge(c.U, tm.TM_SINGLE, tm.TM_RECON_18)
    x_e = si.mask_parity(si.spinor_field(dims, 1, 22), dims, 0)
    in_o = si.mask_parity(si.spinor_field(dims, 1, 23), dims, 1)
    f_e = c.lat.field(tm.TM_SINGLE, 1).upload(0, c.psi_e)
    f_x = c.lat.field(tm.TM_SINGLE, 1).upload(0, x_e)
    f_o = c.lat.field(tm.TM_SINGLE, 1).upload(1, in_o)
    out = c.lat.field(tm.TM_SINGLE, 1)
    for dagger in (0, 1):
        # A on the odd sites from the even input
        tm.dslash_apply(out, f_e, None, g, pg, 1, dagger, tm.TM_TWIST_INV_DSLASH)
        c.lat.sync()
        sites = sample_sites(dims, 1, 5 + dagger)
        want = oracle.kernel_sites(sites, c.psi_e, None, c.U, po, dagger, oracle.A)
        assert rel_l2_sites(out.download(1), want, sites) <= TOL[tm.TM_SINGLE]
        # B on the even sites from the odd input and the even x
        tm.dslash_apply(out, f_o, f_x, g, pg, 0, dagger, tm.TM_DSLASH_TWIST_XPAY)
        c.lat.sync()
        sites = sample_sites(dims, 0, 7 + dagger)
        want = oracle.kernel_sites(sites, in_o, x_e, c.U, po, dagger, oracle.B)
        assert rel_l2_sites(out.download(0), want, sites) <= TOL[tm.TM_SINGLE]


@pytest.mark.parametrize("prec", [tm.TM_DOUBLE, tm.TM_SINGLE, tm.TM_HALF], ids=["fp64", "fp32", "half"])
@pytest.mark.parametrize("typ", [tm.TM_MATPC_ASYM, tm.TM_MATPC_SYM], ids=["eq2.2", "eq2.3"])
def test_config3_32c64_degenerate_precision_sweep(case3, prec, typ):
    """configs[2]: full Eq. 2.2 and Eq. 2.3 operators, 12-real Haar links, mu = 0.0015 (bench.py's degenerate leg)."""
    err = case3.check_matpc(dict(mu=0.0015, epsilon=0.0, twist_flavor=1), prec, tm.TM_RECON_12, typ, 0, 31, full=True)
    print("config3", PREC_NAME[prec], typ, "rel L2 on the whole lattice = %.3e" % err)


@pytest.mark.parametrize("prec", [tm.TM_DOUBLE, tm.TM_SINGLE, tm.TM_HALF], ids=["fp64", "fp32", "half"])
def test_config3_32c64_8real_links(case3, prec):
    """The same Eq. 2.2 operator with 8-real links (Table 1's "8" rows; `python bench.py --recon 8` times this launch
    configuration): fp64 = scalar kernel, fp32 = packed kernel with the fast special-function rebuild."""
    err = case3.check_matpc(dict(mu=0.0015, epsilon=0.0, twist_flavor=1), prec, tm.TM_RECON_8, tm.TM_MATPC_ASYM, 0, 33, full=True)
    print("config3 8-real", PREC_NAME[prec], "rel L2 on the whole lattice = %.3e" % err)


@pytest.mark.parametrize("prec", [tm.TM_SINGLE, tm.TM_HALF], ids=["fp32", "half"])
@pytest.mark.parametrize("dagger", [0, 1], ids=["plain", "dagger"])
def test_config4_32c64_nondegenerate_doublet(case4, prec, dagger):
    """configs[3]: flavor-coupled 2x2 R^-1 fused kernels, plain and dagger (bench.py's non-degenerate leg)."""
    err = case4.check_matpc(dict(mu=0.15, epsilon=0.19, twist_flavor=0), prec, tm.TM_RECON_12, tm.TM_MATPC_ASYM, dagger, 41, full=True)
    print("config4", PREC_NAME[prec], "dagger" if dagger else "plain", "rel L2 on the whole lattice = %.3e" % err)


def test_config4_doublet_fp64_sampled(case4):
    """The fp64 doublet kernels (configs[4]'s kernels) at 32^3x64, 18-real, SYM (Eq. 2.3)."""
    case4.check_matpc(dict(mu=0.135, epsilon=0.17, twist_flavor=0), tm.TM_DOUBLE, tm.TM_RECON_18, tm.TM_MATPC_SYM, 0, 51, full=True)


def _host_gb():
    try:
        import psutil
        return psutil.virtual_memory().available / 2 ** 30
    except Exception:
        return 0.0


# ~1 minute on the B200 box (196 GB of host memory); needs ~25 GB of host memory for the 48^3x96 double inputs
@pytest.mark.skipif(os.environ.get("TM_TEST_HUGE", "1") == "0" or _host_gb() < 40,
                    reason="48^3x96 host inputs need ~25 GB of host memory (or TM_TEST_HUGE=0)")
def test_config5_48c96_nondegenerate_fp64_sym_100_applications():
    """configs[4]: Eq. 2.3 operator, Haar 18-real links, applied 100 times back to back; sampled parity on the
    first application and bit-identical output on the 100th."""
    dims = (48, 48, 48, 96)
    c = Case(dims, "haar", 5, 2)
    kw = dict(mu=0.135, epsilon=0.17, twist_flavor=0)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    g = c.lat.gauge(c.U, tm.TM_DOUBLE, tm.TM_RECON_18)
    fin = c.lat.field(tm.TM_DOUBLE, 2).upload(0, c.psi_e)
    ftmp, fout = c.lat.field(tm.TM_DOUBLE, 2), c.lat.field(tm.TM_DOUBLE, 2)
    tm.mat_pc(fout, fin, ftmp, g, pg, tm.TM_MATPC_SYM, 0)
    c.lat.sync()
    first = fout.storage.clone()
    sites = sample_sites(dims, 0, 55, n=512)
    want = oracle.matpc_sites(sites, c.psi_e, c.U, po, oracle.SYM, 0)
    assert rel_l2_sites(fout.download(0), want, sites) <= TOL[tm.TM_DOUBLE]
    for _ in range(99):
        tm.mat_pc(fout, fin, ftmp, g, pg, tm.TM_MATPC_SYM, 0)
    c.lat.sync()
    assert bool((first == fout.storage).all())


@pytest.mark.skipif(os.environ.get("TM_TEST_HUGE", "1") == "0" or _host_gb() < 60,
                    reason="64^4 host inputs need ~35 GB of host memory (or TM_TEST_HUGE=0)")
def test_64c64_fp64_gauge_blocks_beyond_4_gib():
    """Maximum-size case for the addressing: at 64^4 one parity block of the fp64 18-real gauge field is 4.8 GB, so link
    offsets pass 2^32 bytes (no BASELINE.json config does: 48^3x96 stops at 3.1 GB per block).  Kernels A (odd output) and
    B (even output) against the oracle at sampled sites, which include the last sites of both parities.  The gauge field is
    a 64^3 x 8 Haar block repeated along x4 (a valid SU(3) field; generating 67 M independent links would take minutes)."""
    dims, small = (64, 64, 64, 64), (64, 64, 64, 8)
    U = np.ascontiguousarray(np.tile(si.gauge_field(small, 6, "haar"), (1, 8, 1, 1)))
    lat = tm.Lattice(dims)
    g = lat.gauge(U, tm.TM_DOUBLE, tm.TM_RECON_18)
    assert 4 * lat.Vh * 18 * 8 > 2 ** 32
    kw = dict(mu=0.004, epsilon=0.0, twist_flavor=1)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    psi = si.spinor_field(dims, 1, 6)
    for parity, kt in ((1, 0), (0, 2)):
        inp = si.mask_parity(psi, dims, 1 - parity)
        x = si.mask_parity(psi, dims, parity)
        fin = lat.field(tm.TM_DOUBLE, 1).upload(1 - parity, inp)
        fx = lat.field(tm.TM_DOUBLE, 1).upload(parity, x)
        fout = lat.field(tm.TM_DOUBLE, 1)
        tm.dslash_apply(fout, fin, None if kt == 0 else fx, g, pg, parity, 0, kt)
        lat.sync()
        sites = sample_sites(dims, parity, 60 + parity, n=1024)
        want = oracle.kernel_sites(sites, inp, x, U, po, 0, kt)
        err = rel_l2_sites(fout.download(parity), want, sites)
        assert err <= TOL[tm.TM_DOUBLE], (parity, kt, err)
        del fin, fx, fout

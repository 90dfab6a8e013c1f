"""Helpers of the GPU parity tests: run one C-ABI call on full-lattice numpy arrays, compare with the oracle."""
import numpy as np

import paper_1311_4462_b200 as tm

TOL = {tm.TM_DOUBLE: 1e-12, tm.TM_SINGLE: 1e-5, tm.TM_HALF: 5e-3}    # BASELINE.json north_star
PREC_NAME = {tm.TM_DOUBLE: "fp64", tm.TM_SINGLE: "fp32", tm.TM_HALF: "half"}


def rel_l2(got, want):
    return float(np.linalg.norm((got - want).ravel()) / max(np.linalg.norm(want.ravel()), 1e-300))


class Bench:
    """One lattice + cached gauge handles per (precision, recon)."""

    def __init__(self, dims, U):
        self.dims = tuple(dims)
        self.lat = tm.Lattice(dims)
        self.U = U
        self._g = {}

    def gauge(self, prec, recon):
        key = (prec, recon)
        if key not in self._g:
            self._g[key] = self.lat.gauge(self.U, prec, recon)
        return self._g[key]

    def kernel(self, inp, x, p, parity, dagger, kt, prec, recon, nf):
        """GPU version of oracle.kernel(): full-lattice arrays in, full-lattice result (only `parity` filled)."""
        lat = self.lat
        fin = lat.field(prec, nf).upload(1 - parity, inp)
        fx = None if x is None else lat.field(prec, nf).upload(parity, x)
        fout = lat.field(prec, nf)
        tm.dslash_apply(fout, fin, fx, self.gauge(prec, recon), p, parity, dagger, kt)
        lat.sync()
        return fout.download(parity)

    def matpc(self, inp, p, typ, dagger, prec, recon, nf):
        lat = self.lat
        fin = lat.field(prec, nf).upload(tm.TM_EVEN, inp)
        ftmp, fout = lat.field(prec, nf), lat.field(prec, nf)
        tm.mat_pc(fout, fin, ftmp, self.gauge(prec, recon), p, typ, dagger)
        lat.sync()
        return fout.download(tm.TM_EVEN)

    def reconstruct_odd(self, psi_e, b_o, p, prec, recon, nf):
        lat = self.lat
        fe = lat.field(prec, nf).upload(tm.TM_EVEN, psi_e)
        fb = lat.field(prec, nf).upload(tm.TM_ODD, b_o)
        fo = lat.field(prec, nf)
        tm.reconstruct_odd(fo, fe, fb, self.gauge(prec, recon), p)
        lat.sync()
        return fo.download(tm.TM_ODD)

    def twist(self, inp, parity, p, inverse, dagger, prec, nf, in_place=False):
        lat = self.lat
        fin = lat.field(prec, nf).upload(parity, inp)
        fout = fin if in_place else lat.field(prec, nf)
        tm.twist_apply(fout, fin, p, inverse, dagger)
        lat.sync()
        return fout.download(parity)

    def prepare_rhs(self, b, p, typ, prec, recon, nf, alias=False):
        lat = self.lat
        fbe = lat.field(prec, nf).upload(tm.TM_EVEN, b)
        fbo = lat.field(prec, nf).upload(tm.TM_ODD, b)
        ftmp = lat.field(prec, nf)
        frhs = fbe if alias else lat.field(prec, nf)
        tm.prepare_rhs(frhs, fbe, fbo, ftmp, self.gauge(prec, recon), p, typ)
        lat.sync()
        return frhs.download(tm.TM_EVEN)

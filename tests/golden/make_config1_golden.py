"""Writes tests/golden/config1_matpc_asym.txt: sampled outputs of the ORACLE (and nothing else) on BASELINE.json
configs[0] -- 4^3 x 8, degenerate twisted mass, Haar links seed 1, Gaussian spinor seed 1 on the even sites,
kappa = 0.1632, mu = 0.004, antiperiodic time -- for the left-hand side of Eq. 2.2 and, with a
Gaussian b_o (seed 2), the reconstruction of Eq. 2.4.

The paper prints no worked example (no values to cite), so this file is not a pin of the oracle: the pins are the
closed forms and invariants of tests/test_oracle_pins.py.  It is a regression guard -- a later change to the oracle's
arithmetic has to change this file in the same commit and say why -- and a second, stored target for the GPU parity
test of configs[0].  Run from the repository root:   python tests/golden/make_config1_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle                      # noqa: E402
import synth_inputs as si          # noqa: E402

DIMS, KAPPA, MU = (4, 4, 4, 8), 0.1632, 0.004
OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_matpc_asym.txt")


def compute():
    U = si.gauge_field(DIMS, 1, "haar")
    p = oracle.params(DIMS, KAPPA, mu=MU, epsilon=0.0, twist_flavor=1)
    psi_e = si.mask_parity(si.spinor_field(DIMS, 1, 1), DIMS, 0)
    b_o = si.mask_parity(si.spinor_field(DIMS, 1, 2), DIMS, 1)
    return oracle.matpc(psi_e, U, p, oracle.ASYM), oracle.reconstruct_odd(psi_e, b_o, U, p)


def samples(dims, parity, n=12):
    idx = si.parity_sites(dims, parity)
    pick = idx[np.linspace(0, len(idx) - 1, n).astype(int)]
    return [(int(s), int(k % 4), int(k % 3)) for k, s in enumerate(pick)]


def main():
    m, r = compute()
    with open(OUT, "w") as f:
        f.write("# written by tests/golden/make_config1_golden.py from oracle/ only; BASELINE.json configs[0]\n")
        f.write("# columns: field  lex_site  spin  color  re  im      (field norm: site = -1)\n")
        for name, a, parity in (("matpc_asym", m, 0), ("reconstruct_odd", r, 1)):
            f.write("%s -1 0 0 %.17e 0\n" % (name, np.linalg.norm(a.ravel())))
            for s, sp, c in samples(DIMS, parity):
                v = a[0, s, sp, c]
                f.write("%s %d %d %d %.17e %.17e\n" % (name, s, sp, c, v.real, v.imag))
    print("wrote", OUT)


if __name__ == "__main__":
    main()

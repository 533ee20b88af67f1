"""Writes tests/golden/oracle_2x2x2x2_L5_4.txt.  Calls ONLY oracle/ and the seeded input generator.

The paper (arXiv:1701.07559) prints no worked numeric example of the operator, so this file is not
a paper value: it is a regression fixture of the pinned oracle (SURVEY.md 8(c) P1-P9 pin it) on the
seeded inputs, guarding the oracle AND the input generator against silent change.
Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle.mdwf_oracle import MdwfOracle  # noqa: E402
from paper_1701_07559_b200 import inputs  # noqa: E402

PARAMS = dict(L=(2, 2, 2, 2), L5=4, M5=1.3, b5=1.5, c5=0.5, mf=0.05, eps=0.3, seed=0)


def compute():
    p = PARAMS
    U = inputs.gauge_field(p["L"], p["eps"], p["seed"]).numpy()
    orc = MdwfOracle(p["L"], p["L5"], p["M5"], p["b5"], p["c5"], p["mf"], U)
    b = inputs.gaussian_source(p["L"], p["L5"], p["seed"]).numpy()
    rows = []
    for name, v in (("U", U), ("b", b), ("D b", orc.D(b)), ("Mpc b_o", orc.Mpc(orc.parity_part(b, 1))),
                    ("Mpcdag b_o", orc.Mpcdag(orc.parity_part(b, 1)))):
        f = v.ravel()
        rows.append((name + " norm2", float(np.vdot(f, f).real), 0.0))
        # sample non-zero entries only (the single-parity results vanish on every even site): first, 8th, middle, last
        nz = np.flatnonzero(f)
        for k in (nz[0], nz[7], nz[nz.size // 2 + 5], nz[-1]):
            rows.append((f"{name} [{k}]", float(f[k].real), float(f[k].imag)))
    return rows


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_2x2x2x2_L5_4.txt")
    with open(out, "w") as fh:
        fh.write("# written by tests/golden/make_golden.py from oracle/ only; params: %r\n" % (PARAMS,))
        for name, re, im in compute():
            fh.write("%s | %.17e | %.17e\n" % (name, re, im))
    print(out)

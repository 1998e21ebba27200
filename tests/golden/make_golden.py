"""Writes tests/golden/config1_oracle.txt from the oracle ALONE (never from the CUDA path).

Run:  python tests/golden/make_golden.py
Stored values: config 1 (BASELINE.json: 4^4, fp64, csw=1.0, m0=-0.1, antiperiodic t,
eps=0.3, omega=1.0): ||D_S b_e||, the 4-sweep Richardson residual history from x0 = 0
(reading R14), and GMRES(2,5) history.  They guard the oracle against accidental change;
a deliberate change must cite the passage / DESIGN.md reading in its commit message.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import oracle  # noqa: E402
from helpers import CONFIGS, config_gauge, config_spinor, even_part  # noqa: E402


def compute():
    c = CONFIGS[1]
    op = oracle.WilsonClover(c["L"], c["T"], c["csw"], c["m0"], c["bc"], config_gauge(1).numpy())
    b = config_spinor(1, 0).numpy()
    bhat = op.prepare_rhs(b)
    y = op.apply_schur(even_part(b, op.par))
    _, rich = oracle.richardson(op.apply_schur, bhat, np.zeros_like(bhat), 4, c["omega"])
    _, gm = oracle.gmres(op.apply_schur, bhat, np.zeros_like(bhat), 5, 2)
    return {
        "norm_schur_apply": [float(np.linalg.norm(y))],
        "norm_bhat": [float(np.linalg.norm(bhat))],
        "richardson_hist": rich,
        "gmres_2x5_hist": gm,
    }


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_oracle.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_golden.py (oracle only); config 1 of BASELINE.json\n")
        for k, v in compute().items():
            f.write(k + " " + " ".join("%.17e" % x for x in v) + "\n")
    print(open(out).read())

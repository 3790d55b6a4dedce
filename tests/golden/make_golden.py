"""Writes tests/golden/config1_oracle.txt: sampled values of the CPU oracle on config 1 (BASELINE.json configs[0]).

    python tests/golden/make_golden.py

Calls only ``oracle/`` and the seeded input recipe (never the CUDA path).  PAPER.md prints no worked numerical example
of the right-hand side, so these are NOT paper values: they freeze the pinned oracle (pins P1-P13
in tests/test_oracle_pins.py) so that a later accidental change of its arithmetic is caught on CPU.  A deliberate
change of the oracle must regenerate this file and name the PAPER.md passage or DESIGN.md reading in its commit.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle as orc                                   # noqa: E402
from paper_1812_00525_b200 import inputs               # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_oracle.txt")
# (field, j, k, i) sample nodes: interior, next to the frozen layers, and across the phi wrap
SAMPLES = [(f, j, k, i) for f in range(8) for (j, k, i) in [(0, 2, 2), (15, 16, 13), (7, 29, 29), (3, 10, 20)]]


def compute():
    prob = inputs.make_problem(1)
    c = prob.cfg
    rows = []
    for tag, kw in (("fd4", {}), ("hall", dict(d_i=0.05)), ("spectral", dict(phi_scheme=1))):
        o = orc.Oracle(c.nR, c.nphi, c.nZ, c.Rmin, c.Rmax, c.Zmin, c.Zmax, c.phi_extent, gamma=c.gamma, eta=c.eta, nu=c.nu,
                       D=c.D, kappa=c.kappa, dt=prob.dt, **kw)
        o.set_equilibrium(prob.U0)
        o.set_state(prob.U)
        K = o.rhs()
        for (f, j, k, i) in SAMPLES:
            rows.append((f"{tag}.K[{f}][{j}][{k}][{i}]", K[f, j, k, i]))
        if tag == "fd4":
            for name, v in o.diagnostics().items():
                rows.append((f"{tag}.diag0.{name}", v))
            rows.append((f"{tag}.setdt(0.5)", o.setdt(0.5)))
            o.step(c.steps)
            U = o.get_state()
            for (f, j, k, i) in SAMPLES:
                rows.append((f"{tag}.U{c.steps}[{f}][{j}][{k}][{i}]", U[f, j, k, i]))
            for name, v in o.diagnostics().items():
                rows.append((f"{tag}.diag{c.steps}.{name}", v))
    return rows


if __name__ == "__main__":
    with open(OUT, "w") as fh:
        fh.write("# written by tests/golden/make_golden.py from oracle/ only (config 1, seed 181200526); hex = exact bits\n")
        for name, v in compute():
            fh.write(f"{name} {float(v).hex()} {v:.17e}\n")
    print(OUT)

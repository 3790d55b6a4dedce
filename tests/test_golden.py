"""The oracle against its frozen sample values (tests/golden/config1_oracle.txt, written by tests/golden/make_golden.py
from oracle/ only).  CPU.  Not paper values (PAPER.md prints none for this path): a regression fence around the pinned
oracle.  Tolerance 1e-13 relative to the field scale: libm / OpenMP scheduling may differ between boxes by an ulp."""
import importlib.util
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_reproduces_its_golden_samples():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
    want = {}
    for line in open(os.path.join(HERE, "golden", "config1_oracle.txt")):
        if line.startswith("#"):
            continue
        name, hx, _dec = line.split()
        want[name] = float.fromhex(hx)
    got = dict(mg.compute())
    assert set(got) == set(want)
    def family(name):          # samples of the same quantity and field share one scale, e.g. "fd4.K[3]"
        return name[:name.find("]") + 1] if "[" in name else name

    scale = {}
    for name, w in want.items():
        scale[family(name)] = max(scale.get(family(name), 0.0), abs(w))
    for name, w in want.items():
        assert abs(got[name] - w) <= 1e-13 * scale[family(name)] + 1e-300, (name, got[name], w)

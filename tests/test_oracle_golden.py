"""Regression of the oracle against tests/golden/*.txt (written by tests/golden/make_golden.py, which calls
only oracle/) and consistency of the byte/flop accounting in DESIGN.md with the paper's Table 1
(tests/golden/paper_table1.txt).  CPU only."""
import os

import numpy as np
import pytest

import oracle
from paper_1206_0675_b200 import inputs

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_trajectory(name):
    rows, it, plaq, final = [], None, None, None
    for line in open(os.path.join(GOLD, name)):
        p = line.split()
        if not p or p[0].startswith("#"):
            continue
        if p[0] == "iterations":
            it = int(p[1])
        elif p[0] == "plaquette":
            plaq = float(p[1])
        elif p[0] == "final":
            final = (int(p[1]), float(p[2]), float(p[3]))
        else:
            rows.append((int(p[0]), float(p[1]), float(p[2])))
    return it, plaq, rows, final


@pytest.mark.parametrize("name,cfg", [("c1_trajectory.txt", "C1"), ("c2pg_trajectory.txt", "C2pg")])
def test_oracle_reproduces_golden_trajectory(name, cfg):
    it, plaq, rows, final = read_trajectory(name)
    c = inputs.CONFIGS[cfg]
    U = inputs.make_config(cfg)
    assert abs(oracle.plaquette(c["dims"], U) - plaq) < 1e-14
    _, Fh, Th = oracle.iterate(c["dims"], U, c["alpha"], 20)
    for n, F, th in rows:
        assert abs(Fh[n] - F) <= 1e-12 * abs(F)
        assert abs(Th[n] - th) <= 1e-12 * abs(th)


def test_table1_reconciles_with_definitions():
    """Table 1 against the definitions: k2 loads 8 links and stores Delta + 2 partials,
    k6 loads 4 links + 5 g's and stores 4 links; the 12-real extra flops are whole third-row
    reconstructions of 42 flops.  This is the accounting DESIGN.md's algorithmic bytes are derived from."""
    t = {}
    for line in open(os.path.join(GOLD, "paper_table1.txt")):
        if line.startswith("#"):
            continue
        p = line.split()
        t[p[0]] = [int(v) for v in p[1:]]
    assert t["k2"][0] == 8 * 18 and t["k2"][1] == 18 + 2
    assert t["k2"][3] == 8 * 12 and t["k2"][4] == 12 + 2
    assert t["k6"][0] == 4 * 18 + 5 * 18 and t["k6"][1] == 4 * 18
    assert t["k6"][3] == 4 * 12 + 5 * 12 and t["k6"][4] == 4 * 12
    recon = 3 * (2 * 6 + 2)                      # 3 components x (2 complex mul + 1 complex sub)
    assert recon == 42
    assert t["k2"][5] - t["k2"][2] == 8 * recon
    assert t["k6"][5] - t["k6"][2] == 9 * recon
    assert t["k6"][2] == 8 * (27 * 6 + 18 * 2)   # 8 complex 3x3 matmuls

"""Writes the stored expected values under tests/golden/ by calling ONLY oracle/ (and the seeded input
generator).  Nothing here touches the CUDA path.  Re-run with:  python tests/golden/make_golden.py

  c1_trajectory.txt   F_n, theta_n, n = 0..20 and the iteration count to theta < 1e-15 for config C1
                      (8^4, eps = 0.2, seed 1001, alpha = 0.08).  The paper prints no F/theta values for
                      any input (PAPER.md has none), so these are regression values of the pinned oracle,
                      not paper values.
  c2pg_trajectory.txt same for the 16^4 pure-gauge configuration (closed form: F -> 1).
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
from paper_1206_0675_b200 import inputs  # noqa: E402


def write(name, cfg):
    c = inputs.CONFIGS[cfg]
    U = inputs.make_config(cfg)
    _, it, Fh, Th = oracle.fix(c["dims"], U, c["alpha"], 1e-15, 2000)
    P = oracle.plaquette(c["dims"], U)
    with open(os.path.join(HERE, name), "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/lgf_oracle.c (regression values, not paper values)\n")
        f.write("# config %s dims %s eps %s seed %d alpha %g tol 1e-15\n" % (cfg, c["dims"], c["eps"], c["seed"], c["alpha"]))
        f.write("iterations %d\n" % it)
        f.write("plaquette %.17g\n" % P)
        for n in range(min(21, it + 1)):
            f.write("%d %.17g %.17g\n" % (n, Fh[n], Th[n]))
        f.write("final %d %.17g %.17g\n" % (it, Fh[it], Th[it]))


if __name__ == "__main__":
    write("c1_trajectory.txt", "C1")
    write("c2pg_trajectory.txt", "C2pg")

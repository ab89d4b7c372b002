"""Writes tests/golden/*.txt.  Calls ONLY oracle/ (and the seeded input generators); never the
CUDA path.  The paper prints no worked numeric example (PAPER.md:67-73 name the method only), so
these are not the paper's values: they are the pinned oracle's, stored so that (a) a change to the
oracle's arithmetic shows up as a diff that its commit message must justify, and (b) the GPU can
be checked on a box where only the stored numbers are consulted.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
from paper_2009_06635_b200 import workloads as W  # noqa: E402


def golden_points(grid):
    """64 in-range points of config 2 + 64 points of the config-4 mix (all regions occur)."""
    x1, q1 = W.queries_in_range(grid, 64, 2)
    x2, q2 = W.queries_extrapolation_mix(grid, 64, 4)
    return np.concatenate([x1, x2]), np.concatenate([q1, q2])


def main():
    grid = W.grid_nnpdf_shaped()
    x, q2 = golden_points(grid)
    out = oracle.OraclePdfGrid.from_spec(grid).xfxq2(grid.pids, x, q2)
    hdr = ("oracle xf for workloads.grid_nnpdf_shaped(); columns: x, Q2, then PIDs "
           + " ".join(str(int(p)) for p in grid.pids) + "; floats as C99 hex")
    with open(os.path.join(HERE, "xfxq2_nnpdf_shaped.txt"), "w") as f:
        f.write("# " + hdr + "\n")
        for p in range(len(x)):
            f.write(" ".join(float(v).hex() for v in [x[p], q2[p]] + list(out[:, p])) + "\n")
    aspec = W.make_alphas_grid()
    qq = np.exp(np.random.default_rng(2009).uniform(np.log(0.5), np.log(4e10), 64))
    al = oracle.OracleAlphas.from_spec(aspec).q2(qq)
    with open(os.path.join(HERE, "alphas_one_loop_grid.txt"), "w") as f:
        f.write("# oracle alpha_s(Q2) on workloads.make_alphas_grid(); columns: Q2, alpha_s; C99 hex\n")
        for a, b in zip(qq, al):
            f.write(f"{float(a).hex()} {float(b).hex()}\n")


if __name__ == "__main__":
    main()

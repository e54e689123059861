"""Writes tests/golden/config1_oracle.txt from the CPU oracle ONLY (never from the CUDA path).

Run from the repo root:  python tests/golden/make_golden.py
The file is a regression lock on the oracle's arithmetic: a later change that moves any of these
values must name, in its commit message, the PAPER.md passage or DESIGN.md reading behind it.
The paper prints no worked example, so there is no paper-value fixture.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle.vrc_oracle import Oracle  # noqa: E402
from workloads import make_problem, make_rays  # noqa: E402


def main():
    prob = make_problem(1)
    rays = make_rays(prob, 10_000)
    res = Oracle(prob).cast(rays, per_ray=True)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_oracle.txt")
    with open(out, "w") as f:
        f.write("# config 1 (BASELINE.json configs[0]), 10000 rays, oracle/vrc_oracle.c, IEEE double\n")
        f.write("# written by tests/golden/make_golden.py; values are C99 hex floats\n")
        f.write(f"segments {res.segments}\n")
        f.write(f"rays_accepted {res.rays_accepted}\n")
        f.write(f"tally_sum {float(res.tally.sum()).hex()}\n")
        f.write(f"tally_max {float(res.tally.max()).hex()}\n")
        f.write(f"hash_xor {int(np.bitwise_xor.reduce(res.hash)):#018x}\n")
        for r in range(0, 10_000, 625):
            f.write(f"ray {r} nseg {int(res.nseg[r])} hash {int(res.hash[r]):#018x} "
                    f"sum_score {float(res.sum_score[r]).hex()} tau_exit {float(res.tau_exit[r]).hex()}\n")
        for c in range(0, 1000, 111):
            f.write(f"cell {c} tally {float(res.tally[c]).hex()}\n")
    print("wrote", out)


if __name__ == "__main__":
    main()

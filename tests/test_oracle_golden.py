"""Regression lock: the oracle still reproduces tests/golden/config1_oracle.txt (written by
tests/golden/make_golden.py from the oracle alone)."""
import os

import numpy as np

from oracle.vrc_oracle import Oracle
from workloads import make_problem, make_rays


def _close(a, b):
    # libm exp/expm1 are faithfully, not correctly, rounded: allow a few ulp between glibc builds
    return abs(a - b) <= 1e-14 * abs(b)


def test_oracle_reproduces_golden_config1():
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config1_oracle.txt")
    prob = make_problem(1)
    rays = make_rays(prob, 10_000)
    res = Oracle(prob).cast(rays, per_ray=True)
    seen = 0
    for line in open(path):
        if line.startswith("#"):
            continue
        w = line.split()
        seen += 1
        if w[0] == "segments":
            assert res.segments == int(w[1])
        elif w[0] == "rays_accepted":
            assert res.rays_accepted == int(w[1])
        elif w[0] == "tally_sum":
            assert abs(res.tally.sum() - float.fromhex(w[1])) <= 1e-12 * abs(float.fromhex(w[1]))
        elif w[0] == "tally_max":
            assert _close(res.tally.max(), float.fromhex(w[1]))
        elif w[0] == "hash_xor":
            assert int(np.bitwise_xor.reduce(res.hash)) == int(w[1], 16)
        elif w[0] == "ray":
            r = int(w[1])
            assert int(res.nseg[r]) == int(w[3]) and int(res.hash[r]) == int(w[5], 16)
            assert _close(res.sum_score[r], float.fromhex(w[7])) and _close(res.tau_exit[r], float.fromhex(w[9]))
        elif w[0] == "cell":
            assert _close(res.tally[int(w[1])], float.fromhex(w[3]))
    assert seen >= 30

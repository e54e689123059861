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
    write_extensions()


def write_extensions():
    """tests/golden/extensions_oracle.txt: regression lock on the oracle's next-event, nuclide-mixture, R-Z and
    spherical paths; same rule: written from the oracle alone."""
    from tests.tiny import tiny_rz_problem, tiny_rz_rays, tiny_sphere_problem, tiny_sphere_rays
    from workloads import add_nuclides

    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "extensions_oracle.txt")
    with open(out, "w") as f:
        f.write("# oracle/vrc_oracle.c, IEEE double; written by tests/golden/make_golden.py; C99 hex floats\n")
        prob = make_problem(1)
        rays = make_rays(prob, 2000)
        ne = Oracle(prob).next_event(rays, [5.0, 5.0, 5.0])
        f.write(f"next_event config1 2000 det 5,5,5 segments {ne.segments} hash_xor {int(np.bitwise_xor.reduce(ne.hash)):#018x} "
                f"det_sum {ne.det_sum.hex()} tau17 {float(ne.tau[17]).hex()}\n")
        mix = add_nuclides(prob, n_nuclides=5)
        rm = Oracle(mix).cast(rays, per_ray=True)
        f.write(f"nuclides config1 2000 segments {rm.segments} tally_sum {float(rm.tally.sum()).hex()} "
                f"sum_score17 {float(rm.sum_score[17]).hex()}\n")
        rz = tiny_rz_problem(7, nr=6, nz=5, K=2, M=3)
        rr = tiny_rz_rays(rz, 7, 500)
        zr = Oracle(rz).cast_rz(rr, rz.re, rz.ze)
        f.write(f"rz tiny7 500 segments {zr.segments} hash_xor {int(np.bitwise_xor.reduce(zr.hash)):#018x} "
                f"tally_sum {float(zr.tally.sum()).hex()} t_exit3 {float(zr.t_exit[3]).hex()}\n")
        sp = tiny_sphere_problem(14, nr=6, K=2, M=3)
        sr = tiny_sphere_rays(sp, 14, 500)
        ss = Oracle(sp).cast_sphere(sr, sp.re)
        f.write(f"sphere tiny14 500 segments {ss.segments} hash_xor {int(np.bitwise_xor.reduce(ss.hash)):#018x} "
                f"tally_sum {float(ss.tally.sum()).hex()} t_exit3 {float(ss.t_exit[3]).hex()}\n")
    print("wrote", out)


if __name__ == "__main__":
    main()

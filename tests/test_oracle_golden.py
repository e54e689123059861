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


def test_oracle_reproduces_golden_extensions():
    """Next-event, nuclide mixtures, R-Z and spherical meshes: tests/golden/extensions_oracle.txt."""
    from tests.tiny import tiny_rz_problem, tiny_rz_rays, tiny_sphere_problem, tiny_sphere_rays
    from workloads import add_nuclides

    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "extensions_oracle.txt")
    lines = {ln.split()[0]: ln.split() for ln in open(path) if not ln.startswith("#")}
    field = lambda w, k: w[w.index(k) + 1]
    prob = make_problem(1)
    rays = make_rays(prob, 2000)
    ne = Oracle(prob).next_event(rays, [5.0, 5.0, 5.0])
    w = lines["next_event"]
    assert ne.segments == int(field(w, "segments")) and int(np.bitwise_xor.reduce(ne.hash)) == int(field(w, "hash_xor"), 16)
    assert abs(ne.det_sum - float.fromhex(field(w, "det_sum"))) <= 1e-12 * ne.det_sum and _close(ne.tau[17], float.fromhex(field(w, "tau17")))
    rm = Oracle(add_nuclides(prob, n_nuclides=5)).cast(rays, per_ray=True)
    w = lines["nuclides"]
    assert rm.segments == int(field(w, "segments")) and _close(rm.sum_score[17], float.fromhex(field(w, "sum_score17")))
    assert abs(rm.tally.sum() - float.fromhex(field(w, "tally_sum"))) <= 1e-12 * rm.tally.sum()
    rz = tiny_rz_problem(7, nr=6, nz=5, K=2, M=3)
    zr = Oracle(rz).cast_rz(tiny_rz_rays(rz, 7, 500), rz.re, rz.ze)
    w = lines["rz"]
    assert zr.segments == int(field(w, "segments")) and int(np.bitwise_xor.reduce(zr.hash)) == int(field(w, "hash_xor"), 16)
    assert zr.t_exit[3] == float.fromhex(field(w, "t_exit3")) and abs(zr.tally.sum() - float.fromhex(field(w, "tally_sum"))) <= 1e-12 * zr.tally.sum()
    sp = tiny_sphere_problem(14, nr=6, K=2, M=3)
    ss = Oracle(sp).cast_sphere(tiny_sphere_rays(sp, 14, 500), sp.re)
    w = lines["sphere"]
    assert ss.segments == int(field(w, "segments")) and int(np.bitwise_xor.reduce(ss.hash)) == int(field(w, "hash_xor"), 16)
    assert ss.t_exit[3] == float.fromhex(field(w, "t_exit3")) and abs(ss.tally.sum() - float.fromhex(field(w, "tally_sum"))) <= 1e-12 * ss.tally.sum()


def test_reference_arm_of_bench_runs_on_the_host(repo_root):
    """bench.py --impl reference (the oracle on the host cores) prints the contract's JSON line without a GPU."""
    import json
    import subprocess
    import sys

    out = subprocess.run([sys.executable, os.path.join(repo_root, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "1", "--config", "1", "--ref-rays", "2000"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-500:]
    d = json.loads(out.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["metric"] == "ray_cell_segments_per_sec" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0

"""Pins for the R-Z (cylindrical) mesh walk of the oracle (vrc_cast_rz, steps Z1..Z5; SURVEY.md §8(f) NEXT-4,
PAPER.md:358) against things other than itself: brute-force crossing lists from numpy polynomial roots, point
membership of segment mid-points, the exit distance from an independent ray/cylinder/slab intersection, the
homogeneous closed form, the collision-probability invariant, rotation invariance about the axis, quadrature
of the plain definition  score_i = W int_{cell i} exp(-tau(s)) ds.
"""
import numpy as np
import pytest

from oracle.vrc_oracle import Oracle, fnv1a_cells
from tests.test_oracle_pins import np_sigma_cell
from tests.tiny import tiny_rz_problem, tiny_rz_rays


def rz_cell_of(prob, pts):
    """Cell of 3-D points by numpy.searchsorted on (rho, z); -1 outside."""
    rho = np.hypot(pts[:, 0], pts[:, 1])
    ir = np.searchsorted(prob.re, rho, side="right") - 1
    iz = np.searchsorted(prob.ze, pts[:, 2], side="right") - 1
    ok = (ir >= 0) & (ir < prob.nr) & (iz >= 0) & (iz < prob.nz)
    return np.where(ok, ir + prob.nr * iz, -1)


def brute_crossings(prob, o, d):
    """Every positive parameter at which the line meets a cylinder r_p (roots of a quadratic, numpy.roots) or a plane
    z_p, sorted; cut at the first one that leaves the mesh (outer cylinder or end planes)."""
    ts = []
    a = d[0] ** 2 + d[1] ** 2
    for p in range(1, prob.nr + 1):
        if a > 0:
            roots = np.roots([a, 2 * (o[0] * d[0] + o[1] * d[1]), o[0] ** 2 + o[1] ** 2 - prob.re[p] ** 2])
            ts += [float(t.real) for t in roots if abs(t.imag) < 1e-12 and t.real > 0]
    if d[2] != 0:
        ts += [float((z - o[2]) / d[2]) for z in prob.ze if (z - o[2]) / d[2] > 0]
    ts = sorted(ts)
    # exit: the first crossing after which the point is outside
    out = []
    for i, t in enumerate(ts):
        out.append(t)
        nxt = ts[i + 1] if i + 1 < len(ts) else t + 1.0
        mid = o + 0.5 * (t + nxt) * d
        if rz_cell_of(prob, mid[None, :])[0] < 0:
            break
    return np.array(out)


def test_trace_equals_brute_force_roots_and_midpoint_membership():
    for seed, uniform in ((1, False), (2, True), (3, False)):
        prob = tiny_rz_problem(seed, nr=6, nz=5, uniform=uniform)
        rays = tiny_rz_rays(prob, seed, 300).astype(np.float64)
        res = Oracle(prob).cast_rz(rays, prob.re, prob.ze, cap=40)
        for r in range(len(rays)):
            o, d = rays[r, :3], rays[r, 3:6]
            ts = brute_crossings(prob, o, d)
            n = int(res.nseg[r])
            assert n == len(ts), (seed, r, n, len(ts))
            bounds = np.concatenate([[0.0], ts])
            np.testing.assert_allclose(res.lens[r, :n], np.diff(bounds), rtol=1e-9, atol=1e-12)
            mids = o[None, :] + (0.5 * (bounds[1:] + bounds[:-1]))[:, None] * d[None, :]
            cells = rz_cell_of(prob, mids)
            assert np.array_equal(res.cells[r, :n], cells), (seed, r)
            assert int(res.hash[r]) == fnv1a_cells(cells)
            assert res.t_exit[r] == pytest.approx(ts[-1], rel=1e-12)
            assert res.sum_l[r] == pytest.approx(ts[-1], rel=1e-13)


def test_axis_parallel_and_through_axis_rays():
    prob = tiny_rz_problem(4, nr=5, nz=6, uniform=True)      # radii 0.5 k, planes -1 + 0.75 k
    orc = Oracle(prob)
    # parallel to the axis at rho = 0.6 (shell 1), from z = -0.9 upward: 6 slabs, length 0.65 then 0.75 each
    res = orc.cast_rz(np.array([[0.6, 0.0, -0.9, 0, 0, 1, 1.0, 1.0]]), prob.re, prob.ze, cap=8)
    assert res.nseg[0] == 6 and np.array_equal(res.cells[0, :6], 1 + 5 * np.arange(6))
    np.testing.assert_allclose(res.lens[0, :6], [0.65] + [0.75] * 5, rtol=1e-14)
    # through the axis in the plane z = -0.9: shells 3,2,1,0 inward, then 1,2,3,4 outward (the axis is not a surface)
    res = orc.cast_rz(np.array([[1.7, 0.0, -0.9, -1, 0, 0, 1.0, 1.0]]), prob.re, prob.ze, cap=12)
    assert res.nseg[0] == 8 and list(res.cells[0, :8]) == [3, 2, 1, 0, 1, 2, 3, 4]
    np.testing.assert_allclose(res.lens[0, :8], [0.2, 0.5, 0.5, 1.0, 0.5, 0.5, 0.5, 0.5], rtol=1e-13, atol=1e-15)
    # tangent-ish chord inside shell 2 that misses cylinder r = 1.0: stays in shell 2 then leaves outward
    res = orc.cast_rz(np.array([[1.2, -0.5, 0.0, 0, 1, 0, 1.0, 1.0]]), prob.re, prob.ze, cap=12)
    assert list(res.cells[0, : res.nseg[0]]) == [2 + 5, 3 + 5, 4 + 5]


def test_exit_distance_homogeneous_closed_form_and_collision_invariant():
    prob = tiny_rz_problem(5, nr=7, nz=4, homogeneous=True)
    rays = tiny_rz_rays(prob, 5, 400, axis_parallel_share=0.05, through_axis_share=0.05)
    res = Oracle(prob).cast_rz(rays, prob.re, prob.ze)
    R, z0, z1 = prob.re[-1], prob.ze[0], prob.ze[-1]
    for r in range(len(rays)):
        o, d = rays[r, :3].astype(np.float64), rays[r, 3:6].astype(np.float64)
        t = np.inf                                               # independent exit: outer cylinder and the two end planes
        a = d[0] ** 2 + d[1] ** 2
        if a > 0:
            b = o[0] * d[0] + o[1] * d[1]
            t = min(t, (-b + np.sqrt(b * b - a * (o[0] ** 2 + o[1] ** 2 - R * R))) / a)
        if d[2] > 0:
            t = min(t, (z1 - o[2]) / d[2])
        elif d[2] < 0:
            t = min(t, (z0 - o[2]) / d[2])
        assert res.t_exit[r] == pytest.approx(t, rel=1e-12)
        S = prob.density[0] * np.interp(float(rays[r, 6]), *prob.xs[0])
        want = float(rays[r, 7]) / S * -np.expm1(-S * t)
        assert res.sum_score[r] == pytest.approx(want, rel=1e-11)
    prob2 = tiny_rz_problem(6, nr=6, nz=5, K=3, M=4)
    rays2 = tiny_rz_rays(prob2, 6, 300)
    res2 = Oracle(prob2).cast_rz(rays2, prob2.re, prob2.ze)
    np.testing.assert_allclose(res2.sum_sig_score, rays2[:, 7] * -np.expm1(-res2.tau_exit), rtol=1e-12)


def test_rotation_about_the_axis_leaves_the_tally_unchanged():
    prob = tiny_rz_problem(7, nr=6, nz=5, K=2, M=3)
    rays = tiny_rz_rays(prob, 7, 500).astype(np.float64)
    a = Oracle(prob).cast_rz(rays, prob.re, prob.ze).tally
    th = 0.7312
    c, s = np.cos(th), np.sin(th)
    rot = rays.copy()
    rot[:, 0], rot[:, 1] = c * rays[:, 0] - s * rays[:, 1], s * rays[:, 0] + c * rays[:, 1]
    rot[:, 3], rot[:, 4] = c * rays[:, 3] - s * rays[:, 4], s * rays[:, 3] + c * rays[:, 4]
    b = Oracle(prob).cast_rz(rot, prob.re, prob.ze).tally
    np.testing.assert_allclose(a, b, rtol=1e-9, atol=1e-12 * a.max())


def test_quadrature_of_the_plain_definition():
    prob = tiny_rz_problem(8, nr=4, nz=3, K=2, M=3)
    rays = tiny_rz_rays(prob, 8, 6).astype(np.float64)
    res = Oracle(prob).cast_rz(rays, prob.re, prob.ze)
    steps = 400_000
    want = np.zeros(prob.ncell)
    for r in range(len(rays)):
        o, d, E, W = rays[r, :3], rays[r, 3:6], float(rays[r, 6]), float(rays[r, 7])
        S = np_sigma_cell(prob, E)
        ds = res.t_exit[r] / steps
        smid = (np.arange(steps) + 0.5) * ds
        cells = rz_cell_of(prob, o[None, :] + smid[:, None] * d[None, :])
        sig = S[cells]
        tau_mid = np.cumsum(sig * ds) - 0.5 * sig * ds
        np.add.at(want, cells, W * np.exp(-tau_mid) * ds)
    np.testing.assert_allclose(res.tally, want, rtol=2e-4, atol=1e-6 * want.max())


def test_rejections():
    prob = tiny_rz_problem(9, nr=4, nz=3, uniform=True)       # R = 2.0, z in [-1, 1.25)
    ok = [0.3, 0.2, 0.0, 0.6, 0.0, 0.8, 1.0, 1.0]
    rows = [ok]
    for f, v in ((0, np.nan), (6, 0.0), (7, np.inf), (0, 2.0), (2, 1.25), (2, -1.0000001)):
        b = list(ok)
        b[f] = v
        rows.append(b)
    rows.append([0.3, 0.2, 0.0, 0.0, 0.0, -0.0, 1.0, 1.0])   # zero direction
    rows.append([0.0, 0.0, -1.0, 0.0, 0.0, 1.0, 1.0, 1.0])   # on the axis, on the lower plane: accepted
    res = Oracle(prob).cast_rz(np.array(rows), prob.re, prob.ze)
    assert res.rays_accepted == 2 and res.rays_rejected == 7
    assert res.nseg[-1] == 3 and not res.nseg[1:-1].any()


# ----------------------------------------------------------------------------- 1-D spherical shells
def test_sphere_trace_equals_brute_force_roots_and_closed_forms():
    """Spherical shells ("1-D spherical meshes"): crossings from numpy.roots of |o + t d|^2 = r_p^2,
    shell of each segment mid-point by searchsorted on |x|, exit = outer sphere; homogeneous closed form."""
    from tests.tiny import tiny_sphere_problem, tiny_sphere_rays

    for seed, uniform in ((11, False), (12, True)):
        prob = tiny_sphere_problem(seed, nr=7, uniform=uniform, homogeneous=True)
        rays = tiny_sphere_rays(prob, seed, 300, through_centre_share=0.05).astype(np.float64)
        res = Oracle(prob).cast_sphere(rays, prob.re, cap=20)
        assert res.rays_accepted == 300
        for r in range(len(rays)):
            o, d = rays[r, :3], rays[r, 3:6]
            ts = []
            for p in range(1, prob.nr + 1):
                for t in np.roots([d @ d, 2 * (o @ d), o @ o - prob.re[p] ** 2]):
                    if abs(t.imag) < 1e-9 and t.real > 1e-12:
                        ts.append(float(t.real))
            ts = np.array(sorted(ts))
            t_out = (-(o @ d) + np.sqrt((o @ d) ** 2 - (d @ d) * (o @ o - prob.re[-1] ** 2))) / (d @ d)
            ts = ts[ts <= t_out * (1 + 1e-12)]
            n = int(res.nseg[r])
            if r >= 15:                                   # (the rays aimed exactly at the centre have double roots)
                assert n == len(ts), (seed, r, n, len(ts))
                bounds = np.concatenate([[0.0], ts])
                np.testing.assert_allclose(res.lens[r, :n], np.diff(bounds), rtol=1e-8, atol=1e-11)
                mids = o[None, :] + (0.5 * (bounds[1:] + bounds[:-1]))[:, None] * d[None, :]
                shells = np.searchsorted(prob.re, np.linalg.norm(mids, axis=1), side="right") - 1
                assert np.array_equal(res.cells[r, :n], shells)
            assert res.t_exit[r] == pytest.approx(t_out, rel=1e-12)
            S = prob.density[0] * np.interp(float(rays[r, 6]), *prob.xs[0])
            assert res.sum_score[r] == pytest.approx(float(rays[r, 7]) / S * -np.expm1(-S * t_out), rel=1e-11)
    # through the centre from shell 3 of uniform shells 0.5 k: 3,2,1,0,1,2,...,6 with lengths 0.2, 0.5, 0.5, 1.0, 0.5...
    prob = tiny_sphere_problem(13, nr=7, uniform=True)
    res = Oracle(prob).cast_sphere(np.array([[0.0, 1.7, 0.0, 0, -1, 0, 1.0, 1.0]]), prob.re, cap=12)
    assert list(res.cells[0, : res.nseg[0]]) == [3, 2, 1, 0, 1, 2, 3, 4, 5, 6]
    np.testing.assert_allclose(res.lens[0, :10], [0.2, 0.5, 0.5, 1.0] + [0.5] * 6, rtol=1e-13, atol=1e-15)


def test_sphere_rotation_invariance_and_rejections():
    from tests.tiny import tiny_sphere_problem, tiny_sphere_rays

    prob = tiny_sphere_problem(14, nr=6, K=2, M=3)
    rays = tiny_sphere_rays(prob, 14, 400).astype(np.float64)
    a = Oracle(prob).cast_sphere(rays, prob.re).tally
    q, _ = np.linalg.qr(np.random.default_rng(1).normal(size=(3, 3)))     # any orthogonal map leaves shells invariant
    rot = rays.copy()
    rot[:, :3] = rays[:, :3] @ q.T
    rot[:, 3:6] = rays[:, 3:6] @ q.T
    np.testing.assert_allclose(Oracle(prob).cast_sphere(rot, prob.re).tally, a, rtol=1e-9, atol=1e-12 * a.max())
    R = prob.re[-1]
    rows = [[0.1, 0.1, 0.1, 0, 0, 1, 1.0, 1.0], [R, 0, 0, 1, 0, 0, 1.0, 1.0], [0.1, 0, 0, 0, 0, 0, 1.0, 1.0],
            [0.1, 0, 0, 0, 0, 1, -1.0, 1.0], [0.0, 0.0, 0.0, 0, 0, 1, 1.0, 1.0]]
    res = Oracle(prob).cast_sphere(np.array(rows), prob.re)
    assert res.rays_accepted == 2 and res.rays_rejected == 3 and res.nseg[4] == prob.nr

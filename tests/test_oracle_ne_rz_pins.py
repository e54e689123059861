"""Pins for the next-event (point-detector) walk on R-Z and spherical meshes (vrc_next_event_rz, steps NZ1..NZ6;
SURVEY.md §8(f) NEXT-3 x NEXT-4) against things other than the oracle:

  * homogeneous medium, detector inside: the closed form  W exp(-S R) / R^2  (Kalos 1963: the plain definition);
  * void: the inverse-square law  W / R^2;
  * cell sequence: every root of the cylinder / sphere quadratics (numpy.roots) and every plane crossing with
    0 < t < 1, sorted; mid-point membership by numpy.searchsorted; cut where the line leaves the mesh;
  * tau: mid-point quadrature of Sigma_t along the straight line (detectors inside and outside the mesh);
  * reciprocity tau(a -> b) = tau(b -> a); rotation about the axis (R-Z) / any orthogonal map (sphere);
  * detectors on a cylinder, on a plane, on the axis / at the centre; an event AT the detector; every rejection rule.
"""
import numpy as np
import pytest

from oracle.vrc_oracle import Oracle, fnv1a_cells
from tests.test_oracle_pins import np_sigma_cell
from tests.tiny import tiny_rz_problem, tiny_rz_rays, tiny_sphere_problem, tiny_sphere_rays


def cell_of(prob, pts, sphere):
    """Cell of 3-D points by numpy.searchsorted; -1 outside the mesh."""
    if sphere:
        ir = np.searchsorted(prob.re, np.sqrt((pts * pts).sum(axis=1)), side="right") - 1
        return np.where((ir >= 0) & (ir < prob.nr), ir, -1)
    rho = np.hypot(pts[:, 0], pts[:, 1])
    ir = np.searchsorted(prob.re, rho, side="right") - 1
    iz = np.searchsorted(prob.ze, pts[:, 2], side="right") - 1
    ok = (ir >= 0) & (ir < prob.nr) & (iz >= 0) & (iz < prob.nz)
    return np.where(ok, ir + prob.nr * iz, -1)


def brute_cells_to_detector(prob, o, det, sphere):
    """Cells between o and det: all surface crossings with 0 < t < 1 (numpy.roots for the quadratics), sorted; the cell
    of every interval's mid-point; cut at the first interval that lies outside the mesh."""
    d = det - o
    ts = []
    if sphere:
        a, b2, c0 = d @ d, 2 * (o @ d), o @ o
    else:
        a, b2, c0 = d[0] ** 2 + d[1] ** 2, 2 * (o[0] * d[0] + o[1] * d[1]), o[0] ** 2 + o[1] ** 2
    if a > 0:
        for p in range(1, prob.nr + 1):
            for t in np.roots([a, b2, c0 - prob.re[p] ** 2]):
                if abs(t.imag) < 1e-12 and 0 < t.real < 1:
                    ts.append(float(t.real))
    if not sphere and d[2] != 0:
        ts += [float((z - o[2]) / d[2]) for z in prob.ze if 0 < (z - o[2]) / d[2] < 1]
    bounds = np.array([0.0] + sorted(ts) + [1.0])
    mids = o[None, :] + (0.5 * (bounds[1:] + bounds[:-1]))[:, None] * d[None, :]
    cells = cell_of(prob, mids, sphere)
    out = np.flatnonzero(cells < 0)
    n = out[0] if len(out) else len(cells)
    return cells[:n], np.diff(bounds)[:n]


def quad_tau(prob, o, det, E, sphere, n=200_000):
    """Mid-point quadrature of Sigma_t along the line from o to det (outside the mesh: void)."""
    S = np_sigma_cell(prob, E)
    s = (np.arange(n) + 0.5) / n
    pts = o[None, :] + s[:, None] * (det - o)[None, :]
    c = cell_of(prob, pts, sphere)
    inside = np.cumsum(c < 0) == 0                       # the walk stops where the line first leaves the mesh
    return np.where(inside, S[np.maximum(c, 0)], 0.0).sum() * np.linalg.norm(det - o) / n


def events_inside(prob, seed, n, sphere):
    rays = (tiny_sphere_rays if sphere else tiny_rz_rays)(prob, seed, n).astype(np.float64)
    rays[:, 3:6] = np.nan                                # the direction fields are ignored, even non-finite ones
    return rays


def ne(orc, prob, rays, det, sphere):
    return orc.next_event_sphere(rays, det, prob.re) if sphere else orc.next_event_rz(rays, det, prob.re, prob.ze)


@pytest.mark.parametrize("sphere", [False, True])
def test_homogeneous_closed_form_and_void_inverse_square(sphere):
    mk = tiny_sphere_problem if sphere else tiny_rz_problem
    prob = mk(51, nr=7, homogeneous=True) if sphere else mk(51, nr=7, nz=5, homogeneous=True)
    rays = events_inside(prob, 51, 300, sphere)
    det = np.array([0.31, -0.22, 0.4 if not sphere else 0.17])
    assert cell_of(prob, det[None, :], sphere)[0] >= 0
    res = ne(Oracle(prob), prob, rays, det, sphere)
    assert res.rays_rejected == 0
    R = np.linalg.norm(det[None, :] - rays[:, :3], axis=1)
    for r in range(len(rays)):
        S = prob.density[0] * np.interp(rays[r, 6], *prob.xs[0])
        assert res.tau[r] == pytest.approx(S * R[r], rel=1e-12)
        assert res.score[r] == pytest.approx(rays[r, 7] * np.exp(-S * R[r]) / R[r] ** 2, rel=1e-12)
    assert res.det_sum == pytest.approx(res.score.sum(), rel=1e-13)
    void = mk(52, nr=6, homogeneous=True) if sphere else mk(52, nr=6, nz=4, void=True)
    void.density[:] = 0.0
    rays = events_inside(void, 52, 200, sphere)
    for det in (np.array([0.2, 0.1, 0.3]), np.array([30.0, -12.0, 7.0])):      # inside and far outside
        res = ne(Oracle(void), void, rays, det, sphere)
        R2 = ((det[None, :] - rays[:, :3]) ** 2).sum(axis=1)
        np.testing.assert_allclose(res.score, rays[:, 7] / R2, rtol=1e-14)
        assert not res.tau.any()


@pytest.mark.parametrize("sphere", [False, True])
@pytest.mark.parametrize("seed", [61, 62])
def test_cell_sequence_equals_brute_force_roots_cut_at_the_detector(seed, sphere):
    prob = tiny_sphere_problem(seed, nr=8, K=2, M=3) if sphere else tiny_rz_problem(seed, nr=6, nz=5, K=2, M=3)
    rays = events_inside(prob, seed, 250, sphere)
    orc = Oracle(prob)
    top = prob.re[-1]
    dets = [np.array([0.13 * top, -0.21 * top, 0.3]), np.array([0.0, 0.0, 0.35]), np.array([2.5 * top, 0.3, 9.0]),
            np.array([-0.45 * top, 0.4 * top, -0.6])]
    for det in dets:
        res = ne(orc, prob, rays, det, sphere)
        assert res.rays_rejected == 0
        for r in range(len(rays)):
            cells, frac = brute_cells_to_detector(prob, rays[r, :3], det, sphere)
            assert res.nseg[r] == len(cells), (det, r, res.nseg[r], len(cells))
            assert int(res.hash[r]) == fnv1a_cells(cells)
            # tau = sum_i Sigma_i (l_i R) with the brute-force lengths
            S = np_sigma_cell(prob, rays[r, 6])
            tau = (S[cells] * frac).sum() * np.linalg.norm(det - rays[r, :3])
            assert res.tau[r] == pytest.approx(tau, rel=1e-9, abs=1e-13)


@pytest.mark.parametrize("sphere", [False, True])
def test_tau_equals_quadrature_along_the_line(sphere):
    prob = tiny_sphere_problem(71, nr=5, K=3, M=4) if sphere else tiny_rz_problem(71, nr=5, nz=4, K=3, M=4)
    rays = events_inside(prob, 71, 12, sphere)
    orc = Oracle(prob)
    top = prob.re[-1]
    for det in (np.array([0.2 * top, 0.1 * top, 0.25]), np.array([1.7 * top, -0.4 * top, 4.0])):
        res = ne(orc, prob, rays, det, sphere)
        for r in range(len(rays)):
            want = quad_tau(prob, rays[r, :3], det, rays[r, 6], sphere)
            assert res.tau[r] == pytest.approx(want, rel=2e-4, abs=1e-7)
            R2 = ((det - rays[r, :3]) ** 2).sum()
            assert res.score[r] == pytest.approx(rays[r, 7] * np.exp(-res.tau[r]) / R2, rel=1e-13)


@pytest.mark.parametrize("sphere", [False, True])
def test_reciprocity_and_rotation(sphere):
    prob = tiny_sphere_problem(81, nr=7, K=2, M=3) if sphere else tiny_rz_problem(81, nr=6, nz=5, K=2, M=3)
    a = events_inside(prob, 81, 40, sphere)
    b = events_inside(prob, 82, 40, sphere)
    b[:, 6] = a[:, 6]                                    # same energy both ways
    orc = Oracle(prob)
    for r in range(len(a)):
        ab = ne(orc, prob, a[r:r + 1], b[r, :3], sphere)
        ba = ne(orc, prob, b[r:r + 1], a[r, :3], sphere)
        assert ab.tau[0] == pytest.approx(ba.tau[0], rel=1e-11)
        assert ab.nseg[0] == ba.nseg[0]
    det = np.array([0.3, -0.2, 0.1])
    base = ne(orc, prob, a, det, sphere)
    th = 1.234
    c, s = np.cos(th), np.sin(th)
    Q = np.array([[c, -s, 0.0], [s, c, 0.0], [0.0, 0.0, 1.0]])
    if sphere:                                           # any orthogonal map leaves spherical shells alone
        Q = np.linalg.qr(np.random.default_rng(5).normal(size=(3, 3)))[0]
    rot = a.copy()
    rot[:, :3] = a[:, :3] @ Q.T
    res = ne(orc, prob, rot, Q @ det, sphere)
    np.testing.assert_allclose(res.tau, base.tau, rtol=1e-9, atol=1e-13)
    assert np.array_equal(res.nseg, base.nseg)


def test_detectors_on_surfaces_and_exact_geometry():
    prob = tiny_rz_problem(91, nr=4, nz=3, uniform=True)      # radii 0.5 k (R = 2), planes -1 + 0.75 k
    orc = Oracle(prob)
    ev = np.array([[1.75, 0.0, -0.875, 0, 0, 0, 1.0, 1.0]])   # dyadic coordinates: every crossing parameter below is exact
    # through the axis to the far side, inside slab 0: shells 3,2,1,0,1,2,3; the detector at rho = 1.625 is in shell 3
    res = orc.next_event_rz(ev, [-1.625, 0.0, -0.875], prob.re, prob.ze)
    assert res.nseg[0] == 7 and int(res.hash[0]) == fnv1a_cells([3, 2, 1, 0, 1, 2, 3])
    # a detector ON the cylinder r = 1.0 reached from outside: the crossing at t = 1 ends the walk in shell 2 (N-Q5)
    res = orc.next_event_rz(ev, [1.0, 0.0, -0.875], prob.re, prob.ze)
    assert res.nseg[0] == 2 and int(res.hash[0]) == fnv1a_cells([3, 2])
    # a detector on the plane z = -0.25 straight above: ends in slab 0
    res = orc.next_event_rz(ev, [1.75, 0.0, -0.25], prob.re, prob.ze)
    assert res.nseg[0] == 1 and int(res.hash[0]) == fnv1a_cells([3])
    # a detector ON the axis: shells 3,2,1,0
    res = orc.next_event_rz(ev, [0.0, 0.0, -0.875], prob.re, prob.ze)
    assert res.nseg[0] == 4 and int(res.hash[0]) == fnv1a_cells([3, 2, 1, 0])
    # straight up out of the mesh to a detector above it: slabs 0, 1, 2 then void
    res = orc.next_event_rz(ev, [1.75, 0.0, 50.0], prob.re, prob.ze)
    assert res.nseg[0] == 3 and int(res.hash[0]) == fnv1a_cells([3, 3 + 4, 3 + 8])
    S = np_sigma_cell(prob, 1.0)
    want = S[3] * 0.625 + S[7] * 0.75 + S[11] * 0.75
    assert res.tau[0] == pytest.approx(want, rel=1e-13)
    sph = tiny_sphere_problem(92, nr=4, uniform=True)          # radii 0.5 k
    res = Oracle(sph).next_event_sphere(np.array([[0.0, 1.25, 0.0, 0, 0, 0, 1.0, 1.0]]), [0.0, -1.75, 0.0], sph.re)
    assert res.nseg[0] == 6 and int(res.hash[0]) == fnv1a_cells([2, 1, 0, 1, 2, 3])
    res = Oracle(sph).next_event_sphere(np.array([[0.0, 1.25, 0.0, 0, 0, 0, 1.0, 1.0]]), [0.0, 0.0, 0.0], sph.re)
    assert res.nseg[0] == 3 and int(res.hash[0]) == fnv1a_cells([2, 1, 0])


@pytest.mark.parametrize("sphere", [False, True])
def test_rejection_rules(sphere):
    prob = tiny_sphere_problem(95, nr=4, uniform=True) if sphere else tiny_rz_problem(95, nr=4, nz=3, uniform=True)
    ok = [0.3, 0.2, 0.0, np.nan, np.inf, 0.0, 1.0, 1.0]
    rows = [ok]
    bad = [(0, np.nan), (2, np.inf), (6, 0.0), (6, -2.0), (6, np.nan), (7, np.inf), (0, 2.0), (1, -2.5)]
    if not sphere:
        bad += [(2, 1.25), (2, -1.0000001)]
    for f, v in bad:
        b = list(ok)
        b[f] = v
        rows.append(b)
    rows.append([0.5, 0.5, 0.5, 0, 0, 0, 1.0, 1.0])           # AT the detector: R2 == 0
    rays = np.array(rows, dtype=np.float64)
    res = ne(Oracle(prob), prob, rays, np.array([0.5, 0.5, 0.5]), sphere)
    assert res.rays_accepted == 1 and res.rays_rejected == len(rows) - 1
    assert not res.nseg[1:].any() and not res.score[1:].any() and res.nseg[0] > 0
    # linear in W, negative weights accepted
    two = np.array([ok, ok], dtype=np.float64)
    two[1, 7] = -2.5
    res = ne(Oracle(prob), prob, two, np.array([0.5, 0.5, 0.5]), sphere)
    assert res.score[1] == pytest.approx(-2.5 * res.score[0], rel=1e-15)

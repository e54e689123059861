"""Pins for the next-event (point-detector) oracle and the batch-moment oracle, against things OTHER
than themselves (Eq. 5).

Next-event plain definition (Kalos 1963, the estimator PAPER.md:354 names):
    score = W exp(-tau) / R^2,   tau = int_0^R Sigma_t(o + s Omega, E) ds,   Omega = (det - o)/R
with Sigma_t = 0 outside the mesh.  The paper prints no worked example for it.
"""
import numpy as np
import pytest

from oracle.vrc_oracle import (Oracle, batch_moments, figure_of_merit, fnv1a_cells, fom_ratio, fractional_difference, mean_and_sigma,
                               relative_difference)
from tests.test_oracle_pins import np_sigma_cell
from tests.tiny import tiny_problem, tiny_rays


def cell_of(prob, pts):
    """Cell index of points (numpy.searchsorted, side='right'), -1 outside the mesh."""
    ix = np.searchsorted(prob.xe, pts[:, 0], side="right") - 1
    iy = np.searchsorted(prob.ye, pts[:, 1], side="right") - 1
    iz = np.searchsorted(prob.ze, pts[:, 2], side="right") - 1
    ok = (ix >= 0) & (ix < prob.nx) & (iy >= 0) & (iy < prob.ny) & (iz >= 0) & (iz < prob.nz)
    return np.where(ok, ix + prob.nx * (iy + prob.ny * iz), -1)


def quadrature_tau(prob, o, det, E, steps=200_000):
    """Mid-point quadrature of Sigma_t along the straight line o -> det (void outside the mesh)."""
    S = np_sigma_cell(prob, E)
    s = (np.arange(steps) + 0.5) / steps
    pts = o[None, :] + s[:, None] * (det - o)[None, :]
    c = cell_of(prob, pts)
    R = np.linalg.norm(det - o)
    return np.where(c >= 0, S[np.maximum(c, 0)], 0.0).sum() * R / steps


def brute_cells_to_detector(prob, o, det):
    """Cells between o and det: every plane crossing with parameter t < 1 (t = 1 is the detector),
    stable-sorted by (t, axis), cut where the line leaves the mesh."""
    edges = (prob.xe, prob.ye, prob.ze)
    n = (prob.nx, prob.ny, prob.nz)
    d = det - o
    idx = [int(np.searchsorted(edges[a], o[a], side="right")) - 1 for a in range(3)]
    ev = []
    for a in range(3):
        if d[a] == 0:
            continue
        inv = 1.0 / d[a]
        planes = range(idx[a] + 1, n[a] + 1) if d[a] > 0 else range(idx[a], -1, -1)
        for seq, p in enumerate(planes):
            t = (edges[a][p] - o[a]) * inv
            if t < 1.0:
                ev.append((t, a, seq))
    ev.sort()
    cells = [idx[0] + n[0] * (idx[1] + n[1] * idx[2])]
    for t, a, _ in ev:
        idx[a] += 1 if d[a] > 0 else -1
        if idx[a] < 0 or idx[a] >= n[a]:
            break
        cells.append(idx[0] + n[0] * (idx[1] + n[1] * idx[2]))
    return np.array(cells)


# ----------------------------------------------------------------------------- closed forms
def test_homogeneous_closed_form_detector_inside():
    """One material everywhere: score = W exp(-Sigma R) / R^2 with Sigma from numpy.interp."""
    prob = tiny_problem(11, homogeneous=True)
    rays = tiny_rays(prob, 11, 300)
    det = np.array([0.37, 0.11, 0.93])
    res = Oracle(prob).next_event(rays, det)
    R = np.linalg.norm(det[None, :] - rays[:, :3].astype(np.float64), axis=1)
    Sig = np.array([prob.density[0] * np.interp(float(e), *prob.xs[0]) for e in rays[:, 6]])
    want = rays[:, 7].astype(np.float64) * np.exp(-Sig * R) / R**2
    np.testing.assert_allclose(res.score, want, rtol=2e-13)
    np.testing.assert_allclose(res.tau, Sig * R, rtol=2e-13)
    np.testing.assert_allclose(res.det_sum, want.sum(), rtol=1e-12)
    assert res.rays_accepted == 300 and res.segments == int(res.nseg.sum())


def test_void_is_inverse_square():
    prob = tiny_problem(12, void=True)
    rays = tiny_rays(prob, 12, 100)
    det = np.array([5.0, -3.0, 9.0])          # outside the mesh: the way there is void anyway
    res = Oracle(prob).next_event(rays, det)
    R2 = ((det[None, :] - rays[:, :3].astype(np.float64)) ** 2).sum(axis=1)
    np.testing.assert_allclose(res.score, rays[:, 7] / R2, rtol=1e-15)
    assert not res.tau.any()


# ----------------------------------------------------------------------------- quadrature of the plain definition
@pytest.mark.parametrize("seed,det", [(21, (0.4, 0.3, 1.1)), (22, (-0.9, 1.0, 2.0)), (23, (7.0, 4.0, -6.0)),
                                      (24, (0.0, -4.0, 0.5))])
def test_tau_equals_quadrature_of_sigma_along_the_line(seed, det):
    """Detectors inside and outside the mesh (outside: void beyond the boundary, reading N-Q2)."""
    prob = tiny_problem(seed, K=3, M=4)
    rays = tiny_rays(prob, seed, 12)
    det = np.array(det, dtype=np.float64)
    res = Oracle(prob).next_event(rays, det)
    for r in range(len(rays)):
        o = rays[r, :3].astype(np.float64)
        q = quadrature_tau(prob, o, det, float(rays[r, 6]))
        assert abs(res.tau[r] - q) <= 2e-4 * max(q, 1e-3), (r, res.tau[r], q)
        R2 = ((det - o) ** 2).sum()
        assert res.score[r] == pytest.approx(float(rays[r, 7]) * np.exp(-res.tau[r]) / R2, rel=1e-14)


# ----------------------------------------------------------------------------- trace
@pytest.mark.parametrize("seed,uniform", [(31, True), (32, False), (33, False)])
def test_cell_sequence_equals_brute_force_crossing_list(seed, uniform):
    prob = tiny_problem(seed, uniform=uniform)
    rays = tiny_rays(prob, seed, 200, axis_aligned_share=0.2)
    g = np.random.default_rng(seed)
    for det in (np.array([0.31, 0.17, 0.77]), np.array([3.5, -2.0, 1.0]), g.normal(size=3) * 3):
        res = Oracle(prob).next_event(rays, det)
        for r in range(len(rays)):
            cells = brute_cells_to_detector(prob, rays[r, :3].astype(np.float64), det)
            assert res.nseg[r] == len(cells)
            assert int(res.hash[r]) == fnv1a_cells(cells)


def test_detector_on_planes_and_lattice_points_ends_the_walk_there():
    """t = 1 exactly at a plane: the segment ends AT the detector and the cell beyond is not entered."""
    prob = tiny_problem(41, nx=4, ny=4, nz=4, uniform=True)     # planes at -1 + 0.75 k
    o = [-0.625, -0.625, -0.625]                                # centre of cell (0,0,0)
    rays = np.array([o + [0, 0, 0] + [1.0, 1.0]], dtype=np.float64)
    orc = Oracle(prob)
    res = orc.next_event(rays, [0.5, -0.625, -0.625])           # on the x plane p=2 (x = 0.5): cells ix = 0, 1
    assert res.nseg[0] == 2 and int(res.hash[0]) == fnv1a_cells([0, 1])
    res = orc.next_event(rays, [0.5, 0.5, 0.5])                 # lattice point along the diagonal
    cells = brute_cells_to_detector(prob, np.array(o), np.array([0.5, 0.5, 0.5]))
    assert res.nseg[0] == len(cells) and int(res.hash[0]) == fnv1a_cells(cells)
    res = orc.next_event(rays, [-0.625, -0.625, -0.5])          # same cell: one segment
    assert res.nseg[0] == 1


# ----------------------------------------------------------------------------- symmetries
def test_reciprocity_and_linearity():
    """tau(o -> d) == tau(d -> o) for points inside the mesh; the score is linear in W."""
    prob = tiny_problem(51, K=2, M=3)
    rays = tiny_rays(prob, 51, 50)
    rays[:, 6] = rays[0, 6]                                     # one energy
    orc = Oracle(prob)
    det = rays[7, :3].astype(np.float64)
    fwd = orc.next_event(rays, det)
    for r in (0, 3, 11, 29):
        back = rays[7:8].copy()
        bres = orc.next_event(back, rays[r, :3].astype(np.float64))
        assert bres.tau[0] == pytest.approx(fwd.tau[r], rel=1e-12)
    r2 = rays.copy()
    r2[:, 7] *= 2.0
    np.testing.assert_array_equal(orc.next_event(r2, det).score, 2.0 * fwd.score)
    assert fwd.rays_rejected == 1 and fwd.score[7] == 0.0      # the event AT the detector (R = 0) is rejected


def test_rejection_rules():
    prob = tiny_problem(61, uniform=True)
    ok = [0.0, 0.0, 0.0, np.nan, np.inf, 0.0, 1.0, 1.0]         # direction fields are ignored, even non-finite
    rows = [ok]
    for f, v in ((0, np.nan), (6, 0.0), (6, -2.0), (7, np.inf), (2, 1e9), (1, -1.0000001)):
        b = list(ok)
        b[f] = v
        rows.append(b)
    res = Oracle(prob).next_event(np.array(rows), [0.5, 0.5, 0.5])
    assert res.rays_accepted == 1 and res.rays_rejected == 6
    assert res.score[0] > 0 and not res.score[1:].any() and not res.nseg[1:].any()
    assert Oracle(prob).next_event(np.array([ok]), [np.nan, 0, 0]).rays_rejected == 1


# ----------------------------------------------------------------------------- batch moments (NEXT-2)
def test_batch_moments_against_numpy_statistics():
    """mean == numpy.mean over batches; sigma == numpy.std(ddof=1)/sqrt(B) (the standard error of the mean)."""
    g = np.random.default_rng(5)
    x = g.random((7, 50)) * g.random(50) * 10
    s1, s2 = batch_moments(x)
    mean, sigma = mean_and_sigma(s1, s2, 7)
    np.testing.assert_allclose(mean, x.mean(axis=0), rtol=1e-14)
    np.testing.assert_allclose(sigma, x.std(axis=0, ddof=1) / np.sqrt(7), rtol=1e-9)
    np.testing.assert_allclose(s1, x.sum(axis=0), rtol=1e-14)
    np.testing.assert_allclose(s2, (x * x).sum(axis=0), rtol=1e-14)
    # identical batches: zero variance (clamped, never NaN); Eq. (5) with sigma = 0.5, T = 4 is exactly 1
    s1, s2 = batch_moments(np.tile(x[:1], (4, 1)))
    _, sig0 = mean_and_sigma(s1, s2, 4)
    assert np.all(sig0 <= 1e-7 * x[0]) and np.all(np.isfinite(sig0))
    assert figure_of_merit(0.5, 4.0) == 1.0


def test_paper_comparison_metrics_eq6_eq7_eq8():
    """Eqs. (6)-(8) on hand-computed values, and the number the paper prints for Eq. (6): with equal
    variances the criticality-accident run's eta would be the time ratio alone."""
    assert fom_ratio(0.5, 2.0, 1.0, 3.0) == (1.0 / 0.25) * (3.0 / 2.0)
    assert fom_ratio(0.1, 600.0, 0.1, 5893.0) == pytest.approx(5893.0 / 600.0)          # PAPER.md:158, variance ratio 1
    ref = np.array([2.0, 4.0, 0.0, 0.0, -8.0])
    got = np.array([2.5, 3.0, 0.0, 1.0, -6.0])
    assert np.array_equal(relative_difference(ref, got), np.array([0.25, 0.25, 0.0, np.inf, 0.25]))
    sig = np.array([0.25, 2.0, 0.0, 0.0, 4.0])
    assert np.array_equal(fractional_difference(ref, got, sig), np.array([2.0, 0.5, 0.0, np.inf, 0.5]))
    assert np.array_equal(relative_difference(ref, ref), np.zeros(5))

"""Pin for the "1/d_a not finite" branch of O1 / O4 (reading Q10; oracle/vrc_oracle.c cast_one).

A direction component so small that its reciprocal overflows (|d_a| < 2^-1024: 5e-324, 1e-310, ...) cannot
carry the ray across a plane of that axis before the other axes take it out of the mesh: over a path of
length L the coordinate moves by |d_a| L < 1e-300 cm.  What fixes the expected values here is therefore the
ray WITH THAT AXIS REMOVED, evaluated by things other than the oracle:
  * trace: the brute-force crossing list (all plane crossings stable-sorted by (t, axis)) of the ray whose
    tiny component is replaced by an exact zero -- built without any reciprocal of the tiny component;
  * exit distance: the textbook slab method over the remaining axes;
  * score: the homogeneous closed form  sum_i score_i = W/S (1 - exp(-S L)) with L
    that slab-method distance;
  * O1: a ray whose three components are all of that kind cannot move at all and is rejected, like the zero vector.
A component that is subnormal but whose reciprocal is still finite (1e-308) keeps its axis: its crossings exist
(t ~ 1e308 or +inf) and simply come after the exit -- the same trace, by brute force with the axis kept.
"""
import numpy as np
import pytest

from oracle.vrc_oracle import Oracle
from tests.test_oracle_pins import brute_trace, np_sigma_cell, py_fnv1a, slab_exit
from tests.tiny import tiny_problem

TINY = (5e-324, 1e-310, -1e-310, -5e-324, 2.0 ** -1025)   # 1/d overflows to +-inf for every one of them


def subnormal_direction_rays(prob, seed=0):
    """Rays whose direction has one or two components from TINY beside normal ones; returns (rays, zeroed) where
    `zeroed` holds the same rays with the tiny components replaced by exact zeros."""
    g = np.random.default_rng(seed)
    lo = np.array([prob.xe[0], prob.ye[0], prob.ze[0]])
    hi = np.array([prob.xe[-1], prob.ye[-1], prob.ze[-1]])
    rows, zero = [], []
    for axes in ((0,), (1,), (2,), (0, 1), (0, 2), (1, 2)):
        for tiny in TINY:
            for _ in range(3):
                o = lo + (0.05 + 0.9 * g.random(3)) * (hi - lo)
                d = g.normal(size=3)
                d[list(axes)] = 0.0
                d /= np.linalg.norm(d)
                z = d.copy()
                d[list(axes)] = tiny
                E, W = 10.0 ** g.uniform(-2, 1), 0.5 + g.random()
                rows.append(np.concatenate([o, d, [E, W]]))
                zero.append(np.concatenate([o, z, [E, W]]))
    return np.array(rows), np.array(zero)


def test_reciprocals_are_what_the_docstring_says():
    with np.errstate(over="ignore", divide="ignore"):
        for t in TINY:
            assert t != 0.0 and np.isinf(1.0 / np.float64(t))
        assert np.isfinite(1.0 / np.float64(1e-308)) and 1e-308 < np.finfo(np.float64).tiny


@pytest.mark.parametrize("seed,uniform", [(31, True), (32, False)])
def test_axis_with_overflowing_reciprocal_never_steps(seed, uniform):
    prob = tiny_problem(seed, nx=5, ny=4, nz=6, uniform=uniform)
    rays, zeroed = subnormal_direction_rays(prob, seed)
    cap = prob.nx + prob.ny + prob.nz + 3
    res = Oracle(prob).cast(rays, cap=cap)
    assert res.rays_rejected == 0 and res.rays_accepted == len(rays)
    for r in range(len(rays)):
        cells, lens, t_exit = brute_trace(prob, zeroed[r, :3], zeroed[r, 3:6])     # no 1/tiny anywhere in here
        assert res.nseg[r] == len(cells)
        assert np.array_equal(res.cells[r, : len(cells)], cells)
        assert np.array_equal(res.lens[r, : len(cells)], lens)
        assert res.hash[r] == py_fnv1a(cells.astype("<u4").tobytes())
        assert res.t_exit[r] == t_exit == slab_exit(prob, zeroed[r, :3], zeroed[r, 3:6])
        assert abs(res.sum_l[r] - t_exit) <= len(cells) * 2.0 ** -52 * t_exit


def test_all_three_components_tiny_is_rejected_like_the_zero_vector():
    prob = tiny_problem(33, uniform=True)
    rows = []
    for d in ((5e-324, 1e-310, -1e-310), (1e-310, 0.0, 0.0), (0.0, -5e-324, 0.0), (-0.0, 0.0, 2.0 ** -1025), (0.0, 0.0, 0.0)):
        rows.append([0.1, 0.2, 0.3, *d, 1.0, 1.0])
    rows.append([0.1, 0.2, 0.3, 1e-310, 0.0, 1.0, 1.0, 1.0])       # one normal component: accepted
    res = Oracle(prob).cast(np.array(rows), per_ray=True)
    assert res.rays_rejected == 5 and res.rays_accepted == 1
    assert not res.nseg[:5].any() and res.nseg[5] > 0
    assert res.tally is not None and np.isfinite(res.tally).all()


def test_homogeneous_closed_form_with_a_tiny_component():
    """sum_i score_i = W/S (1 - exp(-S L)), L from the slab method over the axes that can move."""
    prob = tiny_problem(34, nx=6, ny=5, nz=4, homogeneous=True)
    rays, zeroed = subnormal_direction_rays(prob, 34)
    res = Oracle(prob).cast(rays, per_ray=True)
    for r in range(len(rays)):
        S = np_sigma_cell(prob, rays[r, 6])[0]
        L = slab_exit(prob, zeroed[r, :3], zeroed[r, 3:6])
        want = rays[r, 7] / S * -np.expm1(-S * L)
        assert abs(res.sum_score[r] - want) <= 1e-13 * want


def test_subnormal_component_with_a_finite_reciprocal_keeps_its_axis():
    """d_a = 1e-308 is subnormal but 1/d_a = 1e308 is finite: the axis steps in principle, its crossings lie at
    t ~ 1e308 (or overflow to +inf) -- after the exit through the normal axes.  Brute force with the axis KEPT."""
    prob = tiny_problem(35, nx=5, ny=4, nz=6, uniform=False)
    g = np.random.default_rng(35)
    lo = np.array([prob.xe[0], prob.ye[0], prob.ze[0]])
    hi = np.array([prob.xe[-1], prob.ye[-1], prob.ze[-1]])
    rows = []
    for a in range(3):
        for s in (1e-308, -1e-308, 6e-309):
            o = lo + (0.05 + 0.9 * g.random(3)) * (hi - lo)
            d = g.normal(size=3)
            d[a] = 0.0
            d /= np.linalg.norm(d)
            d[a] = s
            rows.append(np.concatenate([o, d, [1.0, 1.0]]))
    rays = np.array(rows)
    cap = prob.nx + prob.ny + prob.nz + 3
    res = Oracle(prob).cast(rays, cap=cap)
    assert res.rays_rejected == 0
    with np.errstate(over="ignore"):
        for r in range(len(rays)):
            cells, lens, t_exit = brute_trace(prob, rays[r, :3], rays[r, 3:6])
            assert res.nseg[r] == len(cells)
            assert np.array_equal(res.cells[r, : len(cells)], cells)
            assert np.array_equal(res.lens[r, : len(cells)], lens)
            assert np.isfinite(t_exit) and t_exit < 100.0

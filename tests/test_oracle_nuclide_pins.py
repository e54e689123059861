"""Pins for multi-nuclide materials in the oracle ("first calculating
all cross-sections"): sigma_m(E) = sum_j w_j sigma_nuclide_j(E), every nuclide table lin-lin interpolated."""
import copy

import numpy as np

from oracle.vrc_oracle import Oracle
from tests.tiny import tiny_problem, tiny_rays
from workloads import add_nuclides, make_problem, make_rays


def test_mixture_sigma_is_the_weighted_sum_of_numpy_interp():
    prob = add_nuclides(make_problem(1), n_nuclides=5)
    orc = Oracle(prob)
    g = np.random.default_rng(3)
    for E in np.concatenate([1e-11 * (2e12) ** g.random(200), [1e-12, 50.0]]):   # inside, below and above the grids
        for m in range(prob.M):
            if prob.mixtures[m] is None:
                want = np.interp(E, *prob.xs[m])
            else:
                ids, w = prob.mixtures[m]
                want = sum(float(wj) * np.interp(E, *prob.nuclide_xs[int(q)]) for q, wj in zip(ids, w))
            assert orc.sigma(m, float(E)) == np.float64(want) or abs(orc.sigma(m, float(E)) - want) <= 4e-16 * want


def test_single_nuclide_with_weight_one_equals_the_direct_table_exactly():
    prob = tiny_problem(71, K=2, M=3)
    rays = tiny_rays(prob, 71, 500)
    ref = Oracle(prob).cast(rays, per_ray=True)
    q = copy.copy(prob)
    q.nuclide_xs = [prob.xs[2], prob.xs[1]]
    q.mixtures = [None, (np.array([1], dtype=np.int32), np.array([1.0])), (np.array([0], dtype=np.int32), np.array([1.0]))]
    q.xs = [prob.xs[0], None, None]
    got = Oracle(q).cast(rays, per_ray=True)
    assert np.array_equal(got.tally, ref.tally) and np.array_equal(got.hash, ref.hash)
    # doubling every weight of a material doubles its cross section: same as doubling its density
    q2 = copy.copy(q)
    q2.mixtures = [None, (q.mixtures[1][0], np.array([2.0])), q.mixtures[2]]
    p2 = copy.copy(prob)
    p2.density = prob.density.copy()
    p2.density[1] *= 2.0
    np.testing.assert_allclose(Oracle(q2).cast(rays).tally, Oracle(p2).cast(rays).tally, rtol=1e-13)


def test_homogeneous_mixture_closed_form():
    """One mixture material everywhere: sum of a ray's scores = W/S (1 - exp(-S L)) with S from numpy.interp."""
    prob = tiny_problem(72, homogeneous=True, M=2)
    q = copy.copy(prob)
    q.nuclide_xs = [prob.xs[0], prob.xs[1]]
    q.mixtures = [(np.array([0, 1], dtype=np.int32), np.array([0.25, 0.75])), None]
    q.xs = [None, prob.xs[1]]
    rays = tiny_rays(prob, 72, 200)
    res = Oracle(q).cast(rays, per_ray=True)
    for r in range(len(rays)):
        E = float(rays[r, 6])
        S = prob.density[0] * (0.25 * np.interp(E, *prob.xs[0]) + 0.75 * np.interp(E, *prob.xs[1]))
        want = float(rays[r, 7]) / S * -np.expm1(-S * res.t_exit[r])
        assert abs(res.sum_score[r] - want) <= 1e-12 * want

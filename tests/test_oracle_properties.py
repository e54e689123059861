"""Property tests (hypothesis) of the oracle on random tiny meshes and rays: invariants that hold for ANY input
(SURVEY.md §4 "property tests on tiny random meshes"), each fixed by the mathematics, not by the oracle:
  * sum of segment lengths == the slab-method exit distance (north_star fixed point), per ray;
  * collision-probability invariant  sum_i Sigma_i score_i == W (1 - exp(-tau_exit));
  * every score has the sign of W, and 0 <= sum_i score_i <= W * L (attenuation never adds length);
  * the trace is a chain of face-neighbours that ends on a boundary cell;
  * next-event: tau to a detector ON the ray equals the cast's optical depth accumulated up to that point.
"""
import numpy as np
from hypothesis import HealthCheck, given, settings
from hypothesis import strategies as st

from oracle.vrc_oracle import Oracle
from tests.test_oracle_pins import np_sigma_cell, slab_exit
from tests.tiny import tiny_problem, tiny_rays

SET = dict(max_examples=40, deadline=None, suppress_health_check=[HealthCheck.too_slow])


@settings(**SET)
@given(seed=st.integers(0, 10_000), nx=st.integers(1, 6), ny=st.integers(1, 5), nz=st.integers(1, 6),
       K=st.integers(1, 4), uniform=st.booleans(), aligned=st.sampled_from([0.0, 0.3]))
def test_cast_invariants(seed, nx, ny, nz, K, uniform, aligned):
    prob = tiny_problem(seed, nx=nx, ny=ny, nz=nz, M=3, K=K, uniform=uniform)
    rays = tiny_rays(prob, seed, 40, axis_aligned_share=aligned)
    cap = nx + ny + nz + 2
    res = Oracle(prob).cast(rays, per_ray=True, cap=cap)
    assert res.rays_accepted == 40 and int(res.nseg.max()) <= cap
    n = (nx, ny, nz)
    for r in range(40):
        o, d = rays[r, :3].astype(np.float64), rays[r, 3:6].astype(np.float64)
        W, ns = float(rays[r, 7]), int(res.nseg[r])
        L = slab_exit(prob, o, d)
        assert res.t_exit[r] == L                                           # bitwise: same expression (edge - o) * inv
        assert abs(res.sum_l[r] - L) <= ns * 2.0**-52 * L
        assert abs(res.sum_sig_score[r] - W * -np.expm1(-res.tau_exit[r])) <= 1e-12 * W
        sc = res.scores[r, :ns]
        assert np.all(sc >= 0.0) and sc.sum() <= W * L * (1 + 1e-12)
        cells = res.cells[r, :ns].astype(np.int64)
        ijk = np.stack([cells % nx, (cells // nx) % ny, cells // (nx * ny)], axis=1)
        if ns > 1:
            assert np.all(np.abs(np.diff(ijk, axis=0)).sum(axis=1) == 1)    # one axis per step, one cell at a time
        last = ijk[-1]
        assert any(last[a] in (0, n[a] - 1) for a in range(3))             # the ray leaves through a boundary cell


@settings(**SET)
@given(seed=st.integers(0, 10_000), frac=st.floats(0.05, 0.95))
def test_next_event_tau_matches_the_cast_along_the_same_line(seed, frac):
    """A detector placed ON a ray at parameter s = frac * t_exit: tau(origin -> detector) == sum over the cast's
    segments of Sigma_i * (length inside [0, s])."""
    prob = tiny_problem(seed, nx=4, ny=4, nz=4, M=3, K=2)
    rays = tiny_rays(prob, seed, 6).astype(np.float64)
    orc = Oracle(prob)
    res = orc.cast(rays, per_ray=True, cap=16)
    for r in range(6):
        o, d = rays[r, :3], rays[r, 3:6]
        s = frac * res.t_exit[r]
        ne = orc.next_event(rays[r : r + 1], o + s * d)
        ns = int(res.nseg[r])
        ends = np.cumsum(res.lens[r, :ns])
        starts = ends - res.lens[r, :ns]
        inside = np.clip(np.minimum(ends, s) - starts, 0.0, None)
        # Sigma_i of the crossed cells from numpy.interp (independent of the oracle)
        S = np_sigma_cell(prob, float(rays[r, 6]))[res.cells[r, :ns]]
        want = float((S * inside).sum()) * np.linalg.norm(d)
        assert abs(ne.tau[0] - want) <= 1e-9 * max(want, 1e-3)

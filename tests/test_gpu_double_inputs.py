"""GPU parity in the ALL-DOUBLE mode on genuinely double inputs (north_star: "<= 1e-10 relative in an all-double mode").

Every other DOUBLE-mode test feeds values that happen to be fp32-representable (reading Q2 needs that for the MIXED
mode only).  Here nothing is: tables, densities, fractions, nuclide weights, mesh planes and every ray field carry
their full 53-bit mantissas, so a loader, packer or kernel that demoted anything to float on the DOUBLE path fails
(a float round-trip is a 6e-8 relative error against the 1e-10 bar, and flips start cells / traces).

Covers: the cast on every record layout (LAYOUT_DK3 for K <= 3, generic beyond), the next-event cast, nuclide
mixtures, R-Z and spherical meshes, the ray-ordering pre-pass, the producer ring and host staging, direction
components whose reciprocal overflows (the Q10 branch pinned in tests/test_oracle_subnormal_pins.py), a shaped
reduced config 3, and BASELINE.json's full sizes in the launch configuration `bench.py --double` times.
Bars as everywhere: traces bit-exact (cells AND lengths), counters exact, tallies |d| <= 1e-10 |oracle|.
"""
import numpy as np
import pytest

from tests.tiny import (tiny_problem, tiny_rays, tiny_rz_problem, tiny_rz_rays, tiny_sphere_problem,
                        tiny_sphere_rays)
from workloads import make_problem, make_rays

pytestmark = pytest.mark.gpu

DOUBLE = 1


def _oracle(prob):
    from oracle.vrc_oracle import Oracle

    return Oracle(prob)


def _threads():
    import os

    return max(1, min(32, len(os.sched_getaffinity(0))))


def not_fp32(*arrays):
    """True when every array holds values a float round-trip would change."""
    return all(not np.array_equal(np.asarray(a, dtype=np.float64), np.asarray(a, dtype=np.float64).astype(np.float32))
               for a in arrays)


def assert_tally_double(got, want):
    bad = np.flatnonzero(np.abs(got - want) > 1e-10 * np.abs(want) + 1e-290)
    assert bad.size == 0, f"{bad.size} cells out of the 1e-10 bar; first {bad[0]}: got {got[bad[0]]!r} want {want[bad[0]]!r}"


def check_double_case(prob, rays, cap=0, threads=1):
    from paper_1706_07476_b200 import MonteRay

    assert rays.dtype == np.float64 and not_fp32(rays[:, :3], rays[:, 3:6], rays[:, 6], rays[:, 7])
    ref = _oracle(prob).cast(rays, per_ray=True, cap=cap, threads=threads)
    with MonteRay(0, DOUBLE) as m:
        m.load_problem(prob)
        assert m.ray_dtype == np.float64
        assert m.cast_rays(rays) == len(rays)
        got = m.read_tally()
        st = m.get_stats()
        nseg, hsh, cells, lens = m.trace_rays(rays, cap=cap)
    assert np.array_equal(nseg, ref.nseg), "segment counts differ"
    assert np.array_equal(hsh, ref.hash), "cell-sequence hashes differ"
    if cap:
        assert np.array_equal(cells, ref.cells), "cell traces differ"
        assert np.array_equal(lens, ref.lens), "segment lengths differ (must be bitwise equal)"
    assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
    assert_tally_double(got, ref.tally)
    return ref


# ------------------------------------------------------------------------------------- the cast, every layout
@pytest.mark.parametrize("seed,K,M,uniform", [(701, 1, 2, False), (702, 2, 3, False), (703, 3, 4, True),
                                              (704, 4, 5, False), (705, 5, 6, False), (706, 8, 8, False),
                                              (707, 16, 9, True)])
def test_tiny_random_problems_true_double(seed, K, M, uniform):
    prob = tiny_problem(seed, nx=7, ny=5, nz=6, M=M, K=K, n_e=33, uniform=uniform, fp32_values=False)
    assert not_fp32(prob.density, prob.cell_frac[prob.cell_mat >= 0], *[e for e, _ in prob.xs], *[s for _, s in prob.xs])
    if not uniform:
        assert not_fp32(prob.xe, prob.ye, prob.ze)
    rays = tiny_rays(prob, seed, 3001, axis_aligned_share=0.1, dtype=np.float64)
    check_double_case(prob, rays, cap=24)


def test_dense8_true_double():
    prob = tiny_problem(710, nx=6, ny=6, nz=6, M=8, K=8, n_e=65, fp32_values=False)
    prob.cell_mat[:] = np.arange(8, dtype=np.int32)[None, :]
    prob.cell_frac[:] = np.random.default_rng(710).random(prob.cell_frac.shape)
    check_double_case(prob, tiny_rays(prob, 710, 5000, dtype=np.float64), cap=24)


def test_energy_bracket_next_to_grid_points_true_double():
    """Energies one ulp below / at / one ulp above grid points and at both grid ends: the bucket index is computed
    on (float)E, which must only narrow the search, never change the bracket the double comparison gives."""
    prob = tiny_problem(711, nx=4, ny=4, nz=4, M=3, K=2, n_e=400, fp32_values=False)
    rays = tiny_rays(prob, 711, 6 * 400, dtype=np.float64)
    e = prob.xs[1][0]
    k = np.arange(len(rays)) % len(e)
    pick = np.arange(len(rays)) // len(e)
    E = np.where(pick == 0, e[k], np.where(pick == 1, np.nextafter(e[k], 0.0), np.where(pick == 2, np.nextafter(e[k], np.inf),
                 np.where(pick == 3, e[k] * (1 + 2.0 ** -30), np.where(pick == 4, e[k] * (1 - 2.0 ** -30), e[k] * 1.0000001)))))
    rays[:, 6] = E
    rays[0, 6], rays[1, 6] = e[0] * 0.999999999, e[-1] * 1.000000001     # outside the grid: end values
    check_double_case(prob, rays)


def test_directions_whose_reciprocal_overflows_true_double():
    """The Q10 branch (d_a != 0 but 1/d_a not finite): pinned on the CPU in tests/test_oracle_subnormal_pins.py,
    the same rays here; all-tiny directions are rejected and counted.  Unreachable in MIXED mode (an fp32 subnormal
    promotes to a double whose reciprocal is finite), so DOUBLE mode only."""
    from tests.test_oracle_subnormal_pins import subnormal_direction_rays

    prob = tiny_problem(32, nx=5, ny=4, nz=6, uniform=False, fp32_values=False)
    rays, _ = subnormal_direction_rays(prob, 32)
    c = [0.5 * (e[0] + e[-1]) + 1e-9 for e in (prob.xe, prob.ye, prob.ze)]      # a point well inside the box
    extra = np.array([[*c, 5e-324, 1e-310, -1e-310, 1.0, 1.0], [*c, 1e-310, 0.0, -0.0, 1.0, 1.0],
                      [*c, 1e-308, 0.6, 0.8, 1.0, 1.0], [*c, 0.6, -6e-309, 0.8, 1.0, 1.0]])
    rays = np.ascontiguousarray(np.concatenate([rays, extra, rays[::-1]]))
    ref = check_double_case(prob, rays, cap=prob.nx + prob.ny + prob.nz + 3)
    assert ref.rays_rejected == 2


# ------------------------------------------------------------------------------------- pre-pass, ring, staging
def test_ordering_prepass_ring_and_staging_true_double():
    import torch

    from paper_1706_07476_b200 import MR_OPT_SORT_RAYS, MR_OPT_STAGE_RAYS, MonteRay

    prob = make_problem(3, double_inputs=True, nx=68, ny=68, nz=40, n_e=2000)
    rays = make_rays(prob, 70_001, dtype=np.float64)
    rays[::1000, 6] = -1.0
    assert not_fp32(prob.density, prob.xs[0][0], prob.xs[0][1], rays[:, 0], rays[:, 4], rays[:, 6])
    ref = _oracle(prob).cast(rays, threads=_threads())
    with MonteRay(0, DOUBLE) as m:
        m.load_problem(prob)
        for sort in (1, 0):
            m.set_option(MR_OPT_SORT_RAYS, sort)
            m.clear_tally()
            m.cast_rays(torch.from_numpy(rays).cuda())
            st = m.get_stats()
            assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
            assert_tally_double(m.read_tally(), ref.tally)
        m.set_option(MR_OPT_SORT_RAYS, 1)
        m.set_option(MR_OPT_STAGE_RAYS, 16384)
        m.clear_tally()
        m.cast_rays(rays[:30_000])                      # pageable host batch, staged in chunks on two lanes
        m.ring_open(2, 8192)
        m.ring_push(rays[30_000:])
        m.ring_close()
        st = m.get_stats()
        assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
        assert_tally_double(m.read_tally(), ref.tally)


# ------------------------------------------------------------------------------------- next-event, nuclides
@pytest.mark.parametrize("seed,K,M,uniform", [(721, 1, 2, False), (722, 3, 4, True), (723, 4, 5, False), (724, 8, 8, False)])
def test_next_event_true_double(seed, K, M, uniform):
    from paper_1706_07476_b200 import MonteRay

    prob = tiny_problem(seed, nx=7, ny=5, nz=6, M=M, K=K, n_e=33, uniform=uniform, fp32_values=False)
    rays = tiny_rays(prob, seed, 3001, dtype=np.float64)
    dets = np.array([[0.31 + 1e-9, 0.17 - 1e-11, 0.77 + 3e-10], [float(prob.xe[3]), float(prob.ye[2]), float(prob.ze[4])],
                     [9.0 + 1e-9, -7.0, 3.0], rays[5, :3]])
    orc = _oracle(prob)
    refs = [orc.next_event(rays, d) for d in dets]
    with MonteRay(0, DOUBLE) as m:
        m.load_problem(prob)
        m.load_detectors(dets)
        m.cast_next_event(rays)
        sums = m.read_detectors()
        st = m.get_stats()
        for j, ref in enumerate(refs):
            nseg, hsh, tau, score = m.trace_next_event(rays, j)
            assert np.array_equal(nseg, ref.nseg) and np.array_equal(hsh, ref.hash), f"detector {j}: traces differ"
            assert np.all(np.abs(tau - ref.tau) <= 1e-10 * np.abs(ref.tau) + 1e-290)
            assert np.all(np.abs(score - ref.score) <= 1e-10 * np.abs(ref.score) + 1e-290)
    want = np.array([r.det_sum for r in refs])
    assert np.all(np.abs(sums - want) <= 1e-10 * np.abs(want))
    assert st.ne_pairs_rejected == sum(r.rays_rejected for r in refs) >= 1
    assert st.ne_segments == sum(r.segments for r in refs)


def test_nuclide_mixtures_true_double():
    from workloads import add_nuclides

    prob = add_nuclides(make_problem(3, double_inputs=True, nx=34, ny=34, nz=20, n_e=3000), n_nuclides=6)
    for j, mix in enumerate(prob.mixtures):                # weights with full mantissas
        if mix is not None:
            ids, w = mix
            w = w * (1.0 + 1e-9 * (1 + np.arange(len(w))))
            prob.mixtures[j] = (ids, w)
            assert not_fp32(w)
    rays = make_rays(prob, 20_000, dtype=np.float64)
    check_double_case(prob, rays, threads=_threads())


# ------------------------------------------------------------------------------------- R-Z and spherical meshes
def _check_rz_double(prob, rays, cap, spherical=False):
    from paper_1706_07476_b200 import MonteRay

    assert rays.dtype == np.float64 and not_fp32(rays)
    orc = _oracle(prob)
    ref = orc.cast_sphere(rays, prob.re, cap=cap) if spherical else orc.cast_rz(rays, prob.re, prob.ze, cap=cap)
    with MonteRay(0, DOUBLE) as m:
        m.load_problem(prob)
        m.cast_rays(rays)
        got = m.read_tally()
        st = m.get_stats()
        nseg, hsh, cells, lens = m.trace_rays(rays, cap=cap)
    assert np.array_equal(nseg, ref.nseg) and np.array_equal(hsh, ref.hash)
    assert np.array_equal(cells, ref.cells) and np.array_equal(lens, ref.lens)
    assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
    assert_tally_double(got, ref.tally)


@pytest.mark.parametrize("seed,K,M,uniform", [(731, 1, 2, False), (732, 3, 4, False), (733, 4, 5, False), (734, 8, 8, False)])
def test_rz_true_double(seed, K, M, uniform):
    prob = tiny_rz_problem(seed, nr=7, nz=6, M=M, K=K, n_e=33, uniform=uniform, fp32_values=False)
    assert not_fp32(prob.re[1:], prob.ze, prob.density)
    rays = tiny_rz_rays(prob, seed, 4001, axis_parallel_share=0.05, through_axis_share=0.05, dtype=np.float64)
    _check_rz_double(prob, rays, cap=32)


@pytest.mark.parametrize("seed,K,M,nr", [(741, 1, 2, 9), (742, 3, 4, 40)])
def test_sphere_true_double(seed, K, M, nr):
    prob = tiny_sphere_problem(seed, nr=nr, M=M, K=K, n_e=65, fp32_values=False)
    rays = tiny_sphere_rays(prob, seed, 5003, through_centre_share=0.05, dtype=np.float64)
    _check_rz_double(prob, rays, cap=2 * nr + 1, spherical=True)


# ------------------------------------------------------------------------------------- shaped + full size
def test_config3_reduced_true_double():
    """A shaped case whose tables, densities and fractions are NOT passed through the fp32 rounding of reading Q2."""
    prob = make_problem(3, double_inputs=True, nx=85, ny=85, nz=60)
    rays = make_rays(prob, 50_000, dtype=np.float64)
    assert not_fp32(prob.density, prob.xs[0][0], prob.xs[0][1], prob.xs[3][1])
    check_double_case(prob, rays, threads=_threads())


@pytest.mark.slow
@pytest.mark.parametrize("cfg", [3, 5, 2, 4])
def test_full_size_all_double_in_bench_configuration(cfg):
    """BASELINE.json's full sizes in ALL-DOUBLE mode on genuinely double inputs, library defaults = the launch
    configuration `bench.py --double --config C` times (ordering pre-pass on, device-resident 64-byte ray records;
    config 4: one 10^6-ray batch on the full 512^3 mesh): every ray's segment count and cell-sequence hash, the
    counters and the WHOLE tally against the oracle, |d| <= 1e-10 |oracle|."""
    import torch

    from paper_1706_07476_b200 import MonteRay
    from workloads import FULL_RAYS

    prob = make_problem(cfg, double_inputs=True)
    rays = make_rays(prob, FULL_RAYS[cfg], dtype=np.float64)
    assert not_fp32(prob.density, prob.xs[0][0], prob.xs[0][1], rays[:, 0], rays[:, 3], rays[:, 6], rays[:, 7])
    ref = _oracle(prob).cast(rays, per_ray=True, threads=_threads())
    with MonteRay(0, DOUBLE) as m:
        m.load_problem(prob)
        d_rays = torch.from_numpy(rays).cuda()
        m.cast_rays(d_rays)
        got = m.read_tally()
        st = m.get_stats()
        nseg, hsh, _, _ = m.trace_rays(d_rays)
    assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
    assert np.array_equal(nseg, ref.nseg), "segment counts differ"
    assert np.array_equal(hsh, ref.hash), "cell-sequence hashes differ"
    assert_tally_double(got, ref.tally)


@pytest.mark.slow
def test_config4_all_double_batches_49_and_99_on_the_full_mesh():
    """Config 4 in ALL-DOUBLE mode beyond its first batch (test_full_size_all_double_in_bench_configuration[4] casts
    batch 0): two more of its 100 seeded batches, from the middle and the end of the run, on one context -- traces of
    every ray, counters, and each batch's tally increment against the oracle at 1e-10."""
    import torch

    from paper_1706_07476_b200 import MonteRay

    prob = make_problem(4, double_inputs=True)
    orc = _oracle(prob)
    with MonteRay(0, DOUBLE) as m:
        m.load_problem(prob)
        seg = 0
        for batch in (49, 99):
            rays = make_rays(prob, 1_000_000, batch=batch, dtype=np.float64)
            assert not_fp32(rays[:, 0], rays[:, 3], rays[:, 6], rays[:, 7])
            ref = orc.cast(rays, per_ray=True, threads=_threads())
            d_rays = torch.from_numpy(rays).cuda()
            before = m.read_tally()
            m.cast_rays(d_rays)
            got = m.read_tally()
            nseg, hsh, _, _ = m.trace_rays(d_rays)
            assert np.array_equal(nseg, ref.nseg) and np.array_equal(hsh, ref.hash), f"batch {batch}: traces differ"
            # the increment is a difference of running sums: the bar is taken on the running sum's scale
            d = np.abs((got - before) - ref.tally)
            assert np.all(d <= 1e-10 * np.abs(ref.tally) + 2e-15 * np.abs(got) + 1e-290), f"batch {batch}"
            seg += ref.segments
        st = m.get_stats()
        assert (st.rays_accepted, st.rays_rejected, st.segments) == (2_000_000, 0, seg)

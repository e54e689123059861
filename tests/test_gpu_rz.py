"""GPU parity on R-Z (cylindrical) meshes, through the C ABI against the
oracle's vrc_cast_rz on the same seeded inputs: traces (count, hash, full cell and length lists) bit-exact,
counters exact, tallies within the parity tolerances of DESIGN.md §5."""
import numpy as np
import pytest

from tests.tiny import tiny_rz_problem, tiny_rz_rays

pytestmark = pytest.mark.gpu


def _check(prob, rays32, precision, cap):
    from oracle.vrc_oracle import Oracle
    from paper_1706_07476_b200 import MonteRay

    ref = Oracle(prob).cast_rz(rays32, prob.re, prob.ze, cap=cap)
    with MonteRay(0, precision) as m:
        m.load_problem(prob)
        rays = rays32.astype(m.ray_dtype)
        assert m.cast_rays(rays) == len(rays32)
        got = m.read_tally()
        st = m.get_stats()
        nseg, hsh, cells, lens = m.trace_rays(rays, cap=cap)
    assert np.array_equal(nseg, ref.nseg), "segment counts differ"
    assert np.array_equal(hsh, ref.hash), "cell-sequence hashes differ"
    assert np.array_equal(cells, ref.cells), "cell traces differ"
    assert np.array_equal(lens, ref.lens), "segment lengths differ (must be bitwise equal)"
    assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
    d = np.abs(got - ref.tally)
    bound = (1e-4 * np.abs(ref.tally) + 1e-7 * ref.tally.max()) if precision == 0 else (1e-10 * np.abs(ref.tally) + 1e-290)
    assert np.all(d <= bound)
    return ref


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("seed,K,M,uniform", [(401, 1, 2, False), (402, 3, 4, True), (403, 4, 5, False), (404, 8, 8, False)])
def test_rz_tiny_problems(seed, K, M, uniform, precision):
    """Every record layout; rays parallel to the axis, aimed at the axis, chords that miss inner cylinders;
    4001 rays = several CTAs and a ragged last warp."""
    prob = tiny_rz_problem(seed, nr=7, nz=6, M=M, K=K, n_e=33, uniform=uniform)
    rays = tiny_rz_rays(prob, seed, 4001, axis_parallel_share=0.05, through_axis_share=0.05)
    ref = _check(prob, rays, precision, cap=32)
    assert ref.nseg.max() <= 32


def test_rz_exact_geometry_cases_and_rejections():
    prob = tiny_rz_problem(409, nr=4, nz=3, uniform=True)       # radii 0.5 k (R = 2), planes -1 + 0.75 k
    ok = [0.3, 0.2, 0.0, 0.6, 0.0, 0.8, 1.0, 1.0]
    rows = [ok, [0.0, 0.0, -1.0, 0.0, 0.0, 1.0, 1.0, 1.0],     # on the axis, on the lower plane
            [1.5, 0.0, 0.5, -1.0, 0.0, 0.0, 1.0, 1.0],          # on a cylinder, through the axis
            [1.0, 0.0, 0.5, 0.0, 1.0, 0.0, 1.0, 1.0],           # on a cylinder, tangent direction
            [0.5, 0.5, -1.0, 1.0, 1.0, 1.0, 1.0, 1.0]]
    for f, v in ((0, np.nan), (6, 0.0), (7, np.inf), (0, 2.0), (2, 1.25), (2, -1.0000001)):
        b = list(ok)
        b[f] = v
        rows.append(b)
    rows.append([0.3, 0.2, 0.0, 0.0, 0.0, -0.0, 1.0, 1.0])      # zero direction
    rays = np.array(rows * 30, dtype=np.float32)
    for precision in (0, 1):
        ref = _check(prob, rays, precision, cap=16)
        assert ref.rays_rejected == 30 * 7


@pytest.mark.parametrize("precision", [0, 1])
def test_rz_larger_mesh_with_batches_ring_and_moments(precision):
    """A 300 x 400 R-Z mesh (120 000 cells): host batch, producer ring and per-batch moments work unchanged."""
    from oracle.vrc_oracle import Oracle
    from paper_1706_07476_b200 import MonteRay

    prob = tiny_rz_problem(410, nr=300, nz=400, M=4, K=3, n_e=500)
    rays32 = tiny_rz_rays(prob, 410, 40_000)
    ref = Oracle(prob).cast_rz(rays32, prob.re, prob.ze)
    with MonteRay(0, precision) as m:
        m.load_problem(prob)
        rays = np.ascontiguousarray(rays32.astype(m.ray_dtype))
        m.cast_rays(rays[:15_000])
        m.end_batch()
        m.ring_open(2, 4096)
        m.ring_push(rays[15_000:])
        m.ring_close()
        m.end_batch()
        got = m.read_tally()
        st = m.get_stats()
        s1, s2, nb = m.read_moments()
    assert nb == 2 and np.array_equal(s1, got)
    assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
    d = np.abs(got - ref.tally)
    bound = (1e-4 * np.abs(ref.tally) + 1e-7 * ref.tally.max()) if precision == 0 else (1e-10 * np.abs(ref.tally) + 1e-290)
    assert np.all(d <= bound)


def test_rz_argument_errors_and_unsupported_paths():
    from paper_1706_07476_b200 import MonteRay, MonteRayError

    prob = tiny_rz_problem(411, nr=4, nz=3)
    with MonteRay(0, 0) as m:
        with pytest.raises(MonteRayError):
            m.load_mesh_rz([0.1, 1.0], [0.0, 1.0])               # first radius must be 0
        with pytest.raises(MonteRayError):
            m.load_mesh_rz([0.0, 1.0, 1.0], [0.0, 1.0])           # not strictly increasing
        m.load_problem(prob)
        # a Cartesian mesh loaded afterwards replaces the R-Z one
        m.load_mesh([0.0, 1.0], [0.0, 1.0], [0.0, 1.0])
        assert m.ncell == 1


def test_rz_pin_cell_workload_in_bench_configuration():
    """The R-Z row bench.py times (pin cell, 256 x 2048 shells x slabs) on a sample of its rays: every ray's
    trace hash, counters and the whole tally against the oracle."""
    import torch

    from oracle.vrc_oracle import Oracle
    from paper_1706_07476_b200 import MonteRay
    from workloads import make_rz_problem, make_rz_rays

    prob = make_rz_problem(256, 2048)
    rays = make_rz_rays(prob, 300_000)
    ref = Oracle(prob).cast_rz(rays, prob.re, prob.ze)
    with MonteRay(0, 0) as m:
        m.load_problem(prob)
        d = torch.from_numpy(rays).cuda()
        m.cast_rays(d)
        got = m.read_tally()
        st = m.get_stats()
        nseg, hsh, _, _ = m.trace_rays(d)
    assert np.array_equal(nseg, ref.nseg) and np.array_equal(hsh, ref.hash)
    assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
    assert np.all(np.abs(got - ref.tally) <= 1e-4 * np.abs(ref.tally) + 1e-7 * ref.tally.max())


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("seed,K,M,uniform,nr", [(421, 1, 2, False, 9), (422, 3, 4, True, 40), (423, 8, 8, False, 300)])
def test_spherical_shell_mesh(seed, K, M, uniform, nr, precision):
    """1-D spherical shells (mr_load_mesh_sphere): traces (cells and lengths) bit-exact, counters
    exact, tallies in tolerance; rays aimed at the centre, rejected rays (outside the sphere, zero direction)."""
    from oracle.vrc_oracle import Oracle
    from paper_1706_07476_b200 import MonteRay
    from tests.tiny import tiny_sphere_problem, tiny_sphere_rays

    prob = tiny_sphere_problem(seed, nr=nr, M=M, K=K, n_e=65, uniform=uniform)
    rays32 = tiny_sphere_rays(prob, seed, 5003, through_centre_share=0.05)
    rays32[7, :3] = [1.5 * prob.re[-1], 0.0, 0.0]    # outside the sphere: rejected
    rays32[9, 3:6] = 0.0                             # zero direction: rejected
    cap = 2 * nr + 1 if nr <= 40 else 0
    ref = Oracle(prob).cast_sphere(rays32, prob.re, cap=cap)
    assert ref.rays_rejected == 2
    with MonteRay(0, precision) as m:
        m.load_problem(prob)
        rays = rays32.astype(m.ray_dtype)
        m.cast_rays(rays)
        got = m.read_tally()
        st = m.get_stats()
        nseg, hsh, cells, lens = m.trace_rays(rays, cap=cap)
    assert np.array_equal(nseg, ref.nseg) and np.array_equal(hsh, ref.hash)
    if cap:
        assert np.array_equal(cells, ref.cells) and np.array_equal(lens, ref.lens)
    assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
    d = np.abs(got - ref.tally)
    bound = (1e-4 * np.abs(ref.tally) + 1e-7 * ref.tally.max()) if precision == 0 else (1e-10 * np.abs(ref.tally) + 1e-290)
    assert np.all(d <= bound)


# ------------------------------------------------------------------------------------- next-event on R-Z / spherical meshes
def _check_next_event_rz(prob, rays_in, dets, precision, sphere):
    """mr_cast_next_event / mr_trace_next_event on an R-Z or spherical mesh against the oracle's steps NZ1..NZ6: cell
    sequences (count + FNV-1a hash) bit-exact, counters exact, per-event tau and score and the detector sums within the
    tally tolerances."""
    from oracle.vrc_oracle import Oracle
    from paper_1706_07476_b200 import MonteRay

    orc = Oracle(prob)
    dets = np.asarray(dets, dtype=np.float64).reshape(-1, 3)
    refs = [orc.next_event_sphere(rays_in, d, prob.re) if sphere else orc.next_event_rz(rays_in, d, prob.re, prob.ze) for d in dets]

    def close(got, want, what):
        got, want = np.asarray(got, dtype=np.float64), np.asarray(want, dtype=np.float64)
        scale = np.abs(want).max() if want.size else 0.0
        bound = (1e-4 * np.abs(want) + 1e-7 * scale) if precision == 0 else (1e-10 * np.abs(want) + 1e-290)
        bad = np.flatnonzero(np.abs(got - want) > bound)
        assert bad.size == 0, f"{what}: {bad.size} out of tolerance, first {bad[0]}: got {got[bad[0]]!r} want {want[bad[0]]!r}"

    with MonteRay(0, precision) as m:
        m.load_problem(prob)
        rays = rays_in.astype(m.ray_dtype)
        m.load_detectors(dets)
        assert m.cast_next_event(rays) == len(rays)
        sums = m.read_detectors()
        st = m.get_stats()
        for j, ref in enumerate(refs):
            nseg, hsh, tau, score = m.trace_next_event(rays, j)
            assert np.array_equal(nseg, ref.nseg), f"detector {j}: segment counts differ"
            assert np.array_equal(hsh, ref.hash), f"detector {j}: cell-sequence hashes differ"
            close(tau, ref.tau, f"detector {j} tau")
            close(score, ref.score, f"detector {j} score")
        assert np.array_equal(m.read_detectors(), sums)          # the trace entry adds nothing
        # the cast still works beside it, and a second next-event cast doubles the sums
        m.cast_rays(rays)
        m.cast_next_event(rays)
        close(m.read_detectors(), 2.0 * np.array([r.det_sum for r in refs]), "doubled detector sums")
    close(sums, [r.det_sum for r in refs], "detector sums")
    assert st.ne_pairs_accepted == sum(r.rays_accepted for r in refs)
    assert st.ne_pairs_rejected == sum(r.rays_rejected for r in refs)
    assert st.ne_segments == sum(r.segments for r in refs)
    return refs


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("seed,K,M,uniform", [(451, 1, 2, False), (452, 3, 4, True), (453, 4, 5, False), (454, 8, 8, False)])
def test_next_event_on_rz_mesh(seed, K, M, uniform, precision):
    """Every record layout; detectors inside, on the axis, on a cylinder and a plane, outside the mesh (radially and
    axially), and AT an event (rejected pair); 4001 events = several CTAs and a ragged last warp; fp32-representable
    inputs (reading Q2) for MIXED, genuinely double ones for DOUBLE."""
    dbl = precision == 1
    prob = tiny_rz_problem(seed, nr=7, nz=6, M=M, K=K, n_e=33, uniform=uniform, fp32_values=not dbl)
    rays = tiny_rz_rays(prob, seed, 4001, axis_parallel_share=0.05, dtype=np.float64 if dbl else np.float32)
    top = float(prob.re[-1])
    dets = [[0.31 * top, 0.17 * top, 0.37], [0.0, 0.0, 0.2], [float(prob.re[3]), 0.0, float(prob.ze[2])],
            [2.5 * top, -0.3 * top, 0.1], [0.1 * top, 0.2 * top, 40.0], rays[5, :3].astype(np.float64)]
    refs = _check_next_event_rz(prob, rays, dets, precision, sphere=False)
    assert refs[5].rays_rejected >= 1


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("seed,K,M,nr", [(461, 1, 2, 9), (462, 3, 4, 40), (463, 8, 8, 300)])
def test_next_event_on_spherical_mesh(seed, K, M, nr, precision):
    from tests.tiny import tiny_sphere_problem, tiny_sphere_rays

    dbl = precision == 1
    prob = tiny_sphere_problem(seed, nr=nr, M=M, K=K, n_e=65, fp32_values=not dbl)
    rays = tiny_sphere_rays(prob, seed, 5003, dtype=np.float64 if dbl else np.float32)
    rays[7, :3] = [1.5 * prob.re[-1], 0.0, 0.0]                  # outside the sphere: rejected
    top = float(prob.re[-1])
    dets = [[0.2 * top, -0.3 * top, 0.1 * top], [0.0, 0.0, 0.0], [float(prob.re[nr // 2]), 0.0, 0.0], [3.0 * top, top, -2.0 * top]]
    refs = _check_next_event_rz(prob, rays, dets, precision, sphere=True)
    assert all(r.rays_rejected >= 1 for r in refs)


def test_next_event_rz_rejection_rules_and_pin_cell_workload():
    import torch

    from oracle.vrc_oracle import Oracle
    from paper_1706_07476_b200 import MonteRay
    from workloads import make_rz_problem, make_rz_rays

    prob = tiny_rz_problem(471, nr=4, nz=3, uniform=True)
    ok = [0.25, 0.125, 0.0, np.nan, np.inf, 0.0, 1.0, 1.0]       # direction fields ignored, even non-finite
    rows = [ok]
    for f, v in ((0, np.nan), (6, 0.0), (6, -2.0), (7, np.inf), (0, 2.0), (2, 1.25), (2, -1.0000001)):
        b = list(ok)
        b[f] = v
        rows.append(b)
    rays = np.array(rows * 40, dtype=np.float32)
    for precision in (0, 1):
        refs = _check_next_event_rz(prob, rays, [[0.5, 0.5, 0.5], [0.25, 0.125, 0.0]], precision, sphere=False)
        assert refs[0].rays_rejected == 7 * 40 and refs[1].rays_rejected == 8 * 40
    # the pin-cell workload of bench.py's R-Z rows: a sample of its events against two detectors, device-resident
    big = make_rz_problem(256, 2048)
    ev = make_rz_rays(big, 100_000)
    dets = np.array([[0.6, 0.1, 180.0], [0.0, 0.0, 400.0]])
    orc = Oracle(big)
    refs = [orc.next_event_rz(ev, d, big.re, big.ze) for d in dets]
    with MonteRay(0, 0) as m:
        m.load_problem(big)
        m.load_detectors(dets)
        m.cast_next_event(torch.from_numpy(ev).cuda())
        sums = m.read_detectors()
        st = m.get_stats()
        nseg, hsh, _, _ = m.trace_next_event(torch.from_numpy(ev).cuda(), 0)
    assert np.array_equal(nseg, refs[0].nseg) and np.array_equal(hsh, refs[0].hash)
    assert st.ne_segments == sum(r.segments for r in refs)
    want = np.array([r.det_sum for r in refs])
    assert np.all(np.abs(sums - want) <= 1e-4 * np.abs(want))

"""GPU parity for the two widened rows of SURVEY.md §8(f): NEXT-3 next-event (point-detector) ray cast
and NEXT-2 per-batch moments, through the C ABI, against the CPU oracle on the same seeded inputs.

Bars: cell sequences (count + FNV-1a hash) bit-exact; counters exact; per-event tau and score and the
detector sums within 1e-4 relative (+1e-7 of the largest) in MIXED mode and 1e-10 relative in DOUBLE
mode; batch moments within the tally tolerances (sum) and twice them (sum of squares).
"""
import numpy as np
import pytest

from tests.tiny import tiny_problem, tiny_rays
from workloads import make_problem, make_rays

pytestmark = pytest.mark.gpu


def _mr(prob, precision):
    from paper_1706_07476_b200 import MonteRay

    m = MonteRay(0, precision)
    m.load_problem(prob)
    return m


def _oracle(prob):
    from oracle.vrc_oracle import Oracle

    return Oracle(prob)


def _close(got, want, precision, what):
    got, want = np.asarray(got, dtype=np.float64), np.asarray(want, dtype=np.float64)
    scale = np.abs(want).max() if want.size else 0.0
    bound = (1e-4 * np.abs(want) + 1e-7 * scale) if precision == 0 else (1e-10 * np.abs(want) + 1e-290)
    bad = np.flatnonzero(np.abs(got - want) > bound)
    assert bad.size == 0, f"{what}: {bad.size} out of tolerance, first {bad[0]}: got {got[bad[0]]!r} want {want[bad[0]]!r}"


def check_next_event(prob, rays32, dets, precision):
    orc = _oracle(prob)
    dets = np.asarray(dets, dtype=np.float64).reshape(-1, 3)
    refs = [orc.next_event(rays32, d) for d in dets]
    with _mr(prob, precision) as m:
        rays = rays32.astype(m.ray_dtype)
        m.load_detectors(dets)
        assert m.cast_next_event(rays) == len(rays32)
        sums = m.read_detectors()
        st = m.get_stats()
        for j, ref in enumerate(refs):
            nseg, hsh, tau, score = m.trace_next_event(rays, j)
            assert np.array_equal(nseg, ref.nseg), f"detector {j}: segment counts differ"
            assert np.array_equal(hsh, ref.hash), f"detector {j}: cell-sequence hashes differ"
            _close(tau, ref.tau, precision, f"detector {j} tau")
            _close(score, ref.score, precision, f"detector {j} score")
        # the trace entry adds nothing
        assert np.array_equal(m.read_detectors(), sums)
        m.clear_detectors()
        assert not m.read_detectors().any() and m.get_stats().ne_segments == 0
    _close(sums, [r.det_sum for r in refs], precision, "detector sums")
    assert st.ne_pairs_accepted == sum(r.rays_accepted for r in refs)
    assert st.ne_pairs_rejected == sum(r.rays_rejected for r in refs)
    assert st.ne_segments == sum(r.segments for r in refs)
    return refs


# ------------------------------------------------------------------------------------- next-event
@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("seed,K,M,uniform", [(201, 1, 2, False), (202, 3, 4, True), (203, 4, 5, False), (204, 8, 8, False)])
def test_next_event_tiny_problems(seed, K, M, uniform, precision):
    """Every record layout, non-uniform planes, detectors inside, on planes / lattice points, outside the mesh,
    and AT an event's origin (R = 0: rejected pair); 3001 events = several CTAs and a ragged last warp."""
    prob = tiny_problem(seed, nx=7, ny=5, nz=6, M=M, K=K, n_e=33, uniform=uniform)
    rays = tiny_rays(prob, seed, 3001, axis_aligned_share=0.1)
    dets = [[0.31, 0.17, 0.77], [float(prob.xe[3]), float(prob.ye[2]), float(prob.ze[4])], [9.0, -7.0, 3.0],
            [float(prob.xe[2]), 0.1, 0.2], rays[5, :3].astype(np.float64), [-1.0, -1.0, -1.0]]
    refs = check_next_event(prob, rays, dets, precision)
    assert refs[4].rays_rejected >= 1


@pytest.mark.parametrize("seed,K,uniform,dims", [(211, 2, False, (13, 11, 5)), (212, 3, True, (17, 9, 4)), (213, 3, False, (8, 8, 3)),
                                                 (214, 2, True, (300, 9, 2)), (215, 3, False, (9, 300, 2))])   # more than 256 cells along x / y
def test_next_event_on_the_dictionary_path_with_few_records(seed, K, uniform, dims):
    """Meshes with at most 16 distinct cell records and K >= 2 take next_event_tiled_kernel (walk in tile coordinates, per-entry
    Sigma_t): same cell sequences (hash of the LINEAR cell indices, rebuilt from tile and entry), tau, scores and sums as the
    oracle; plane table in shared memory (non-uniform) and arithmetic planes (uniform), sides that are not multiples of the
    8 x 8 tile, detectors inside, on a lattice point, outside the mesh and at an event's origin."""
    prob = tiny_problem(seed, nx=dims[0], ny=dims[1], nz=dims[2], M=4, K=K, n_e=33, uniform=uniform)
    prob.cell_mat[:] = prob.cell_mat[np.arange(prob.ncell) % 11]         # a repeating pattern of 11 records
    prob.cell_frac[:] = prob.cell_frac[np.arange(prob.ncell) % 11]
    rays = tiny_rays(prob, seed, 3001, axis_aligned_share=0.1)
    dets = [[0.31, 0.17, 0.77], [float(prob.xe[3]), float(prob.ye[2]), float(prob.ze[1])], [9.0, -7.0, 3.0],
            rays[5, :3].astype(np.float64)]
    with _mr(prob, 0) as m:
        assert m.record_path() == "tiled4"
    refs = check_next_event(prob, rays, dets, 0)
    assert refs[3].rays_rejected >= 1


def test_next_event_rejection_rules():
    prob = tiny_problem(261, uniform=True)
    ok = [0.0, 0.0, 0.0, np.nan, np.inf, 0.0, 1.0, 1.0]          # direction fields ignored, even non-finite
    rows = [ok]
    for f, v in ((0, np.nan), (6, 0.0), (6, -2.0), (7, np.inf), (2, 1e9), (1, -1.0000001)):
        b = list(ok)
        b[f] = v
        rows.append(b)
    rays = np.array(rows * 50, dtype=np.float32)
    for precision in (0, 1):
        refs = check_next_event(prob, rays, [[0.5, 0.5, 0.5], [0.0, 0.0, 0.0]], precision)
        assert refs[0].rays_rejected == 300 and refs[1].rays_rejected == 350


@pytest.mark.parametrize("cfg,kw,n", [(1, {}, 10_000), (2, {}, 100_000), (3, {}, 100_000), (5, {}, 50_000)])
def test_next_event_shaped_workloads_mixed(cfg, kw, n):
    """Full-size meshes of configs 1, 2, 3, 5 with detectors inside (far and near) and outside the mesh."""
    prob = make_problem(cfg, **kw)
    rays = make_rays(prob, n)
    lo = np.array([prob.xe[0], prob.ye[0], prob.ze[0]])
    hi = np.array([prob.xe[-1], prob.ye[-1], prob.ze[-1]])
    dets = [lo + 0.5 * (hi - lo), lo + np.array([0.93, 0.11, 0.71]) * (hi - lo), hi + 0.25 * (hi - lo)]
    check_next_event(prob, rays, dets, 0)


def test_next_event_shaped_workload_double_and_device_and_host_batches():
    import torch

    from paper_1706_07476_b200 import MR_OPT_STAGE_RAYS

    prob = make_problem(3, nx=85, ny=85, nz=60)
    rays = make_rays(prob, 30_000)
    lo = np.array([prob.xe[0], prob.ye[0], prob.ze[0]])
    hi = np.array([prob.xe[-1], prob.ye[-1], prob.ze[-1]])
    dets = np.array([lo + 0.4 * (hi - lo), hi + 1.0])
    refs = check_next_event(prob, rays, dets, 1)
    with _mr(prob, 0) as m:
        m.load_detectors(dets)
        m.cast_next_event(torch.from_numpy(rays).cuda())
        a = m.read_detectors()
        m.clear_detectors()
        m.set_option(MR_OPT_STAGE_RAYS, 4096)                  # host batch in 8 staged chunks
        m.cast_next_event(rays)
        b = m.read_detectors()
        assert m.cast_next_event(rays[:0]) == 0
    _close(a, [r.det_sum for r in refs], 0, "device batch")
    np.testing.assert_allclose(a, b, rtol=1e-12)


def test_next_event_call_order_errors():
    from paper_1706_07476_b200 import MonteRayError

    prob = make_problem(1)
    rays = make_rays(prob, 64)
    with _mr(prob, 0) as m:
        with pytest.raises(MonteRayError) as e:
            m.cast_next_event(rays)
        assert e.value.status == 2                               # no detectors
        with pytest.raises(MonteRayError):
            m.load_detectors([[0.0, np.nan, 0.0]])
        m.load_detectors([[1.0, 2.0, 3.0]])
        with pytest.raises(MonteRayError):
            m.trace_next_event(rays, 1)                          # detector index out of range
        m.cast_next_event(rays)
        assert m.get_stats().ne_pairs_accepted == 64


# ------------------------------------------------------------------------------------- per-batch moments
@pytest.mark.parametrize("precision", [0, 1])
def test_batch_moments_against_oracle(precision):
    """B batches of different sizes; sum and sum of squares per cell against the oracle's per-batch tallies,
    mean and sigma (standard deviation of the mean) against the numpy-pinned oracle formulas."""
    from oracle.vrc_oracle import batch_moments, mean_and_sigma

    prob = make_problem(3, nx=68, ny=68, nz=40, n_e=2000) if precision == 0 else tiny_problem(301, nx=9, ny=8, nz=7, K=3, M=4)
    sizes = [30_000, 20_001, 45_000, 10_000, 25_000] if precision == 0 else [3000, 2001, 4500, 999]
    batches = [make_rays(prob, n, batch=b) if precision == 0 else tiny_rays(prob, 300 + b, n) for b, n in enumerate(sizes)]
    orc = _oracle(prob)
    per_batch = np.stack([orc.cast(r, threads=8).tally for r in batches])
    s1, s2 = batch_moments(per_batch)
    with _mr(prob, precision) as m:
        z1, z2, nb = m.read_moments()
        assert nb == 0 and not z1.any() and not z2.any()
        for r in batches:
            m.cast_rays(r.astype(m.ray_dtype))
            m.end_batch()
        g1, g2, nb = m.read_moments()
        mean, sigma, nb2 = m.read_mean_sigma()
        total = m.read_tally()
        # an open batch does not change the closed-batch moments
        m.cast_rays(batches[0].astype(m.ray_dtype))
        h1, h2, nb3 = m.read_moments()
        m.clear_tally()
        c1, c2, nb4 = m.read_moments()
    B = len(sizes)
    assert nb == nb2 == nb3 == B and nb4 == 0 and not c1.any() and not c2.any()
    assert np.array_equal(g1, total) and np.array_equal(h1, g1) and np.array_equal(h2, g2)
    d1 = np.abs(g1 - s1)
    d2 = np.abs(g2 - s2)
    if precision == 0:
        assert np.all(d1 <= 1e-4 * np.abs(s1) + 1e-7 * s1.max())
        assert np.all(d2 <= 2e-4 * np.abs(s2) + 1e-7 * s2.max())
    else:
        assert np.all(d1 <= 1e-10 * np.abs(s1) + 1e-290)
        assert np.all(d2 <= 1e-9 * np.abs(s2) + 1e-290)     # x_b = total - previous total: B ulps of the total
    # mean / sigma evaluated on the device from ITS moments == the oracle formulas applied to the same moments
    rm, rs = mean_and_sigma(g1, g2, B)
    np.testing.assert_allclose(mean, rm, rtol=1e-15)
    np.testing.assert_allclose(sigma, rs, rtol=1e-9, atol=1e-12 * rm.max())
    # and close to the oracle's own statistics (variance is a difference of nearly equal numbers: looser bar)
    om, os_ = mean_and_sigma(s1, s2, B)
    tol = 1e-3 if precision == 0 else 1e-6
    assert np.all(np.abs(sigma - os_) <= tol * os_ + tol * 1e-2 * om.max())


def test_mean_sigma_needs_a_closed_batch():
    from paper_1706_07476_b200 import MonteRayError

    prob = make_problem(1)
    with _mr(prob, 0) as m:
        with pytest.raises(MonteRayError) as e:
            m.read_mean_sigma()
        assert e.value.status == 2
        m.cast_rays(make_rays(prob, 1000))
        m.end_batch()
        mean, sigma, nb = m.read_mean_sigma()
        assert nb == 1 and np.all(np.isinf(sigma)) and np.array_equal(mean, m.read_tally())


# ------------------------------------------------------------------------------------- producer ring (NEXT-1)
@pytest.mark.parametrize("precision,producers,slots,cap", [(0, 1, 3, 5000), (0, 4, 3, 5000), (1, 3, 3, 5000), (0, 8, 2, 1024)])
def test_producer_ring_many_threads_equals_one_call(precision, producers, slots, cap):
    """PAPER.md:77-83 (Fig. 4): producers fill a buffer, full buffers go to the GPU while the producers go on.
    Several host threads push ragged pieces concurrently; after flush the tally and counters equal the oracle's
    for the union of all pushed rays (buffers of 5000 rays: many ships, pieces that straddle buffers, a partial
    last buffer)."""
    import threading

    prob = make_problem(3, nx=68, ny=68, nz=40, n_e=2000)
    rays32 = make_rays(prob, 60_007)
    ref = _oracle(prob).cast(rays32, threads=8)
    with _mr(prob, precision) as m:
        rays = np.ascontiguousarray(rays32.astype(m.ray_dtype))
        m.ring_open(slots, cap)
        bounds = np.linspace(0, len(rays), producers + 1).astype(int)

        def produce(lo, hi, piece):
            i = lo
            while i < hi:
                j = min(hi, i + piece)
                m.ring_push(rays[i:j])
                i = j

        ts = [threading.Thread(target=produce, args=(bounds[k], bounds[k + 1], 777 + 1300 * (k % 3))) for k in range(producers)]
        for t in ts:
            t.start()
        for t in ts:
            t.join()
        m.ring_flush()
        got = m.read_tally()
        st = m.get_stats()
        rs = m.ring_stats()
        m.ring_push(rays[:100])          # the ring stays usable after a flush
        m.ring_close()
        assert m.get_stats().rays_accepted == ref.rays_accepted + 100
    assert rs["rays_pushed"] == len(rays) and rs["slots_shipped"] == -(-len(rays) // cap)
    assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
    d = np.abs(got - ref.tally)
    bound = (1e-4 * np.abs(ref.tally) + 1e-7 * ref.tally.max()) if precision == 0 else (1e-10 * np.abs(ref.tally) + 1e-290)
    assert np.all(d <= bound)


@pytest.mark.parametrize("precision", [0, 1])
def test_producer_ring_merges_waiting_buffers_into_one_cast(precision):
    """MR_OPT_RING_MERGE: a buffer shipped while the GPU is still busy with an earlier cast of the ring is copied at once but
    cast together with the buffers that follow it -- one ordering pre-pass and one launch over consecutive device buffers.
    Forced (2: hold until flush or until the ring wraps): 3 full buffers and a partial one become ONE cast; 6.3 buffers
    through 4 slots become two casts (the wrap sends the first four off) plus the flush.  Off (0): one cast per buffer.
    Auto (1): anything in between.  Every mode: counters exact, tally within tolerance of the oracle; several producer
    threads (buffers shipped out of order) included."""
    import threading

    from paper_1706_07476_b200 import MR_OPT_RING_MERGE

    prob = make_problem(3, nx=68, ny=68, nz=40, n_e=2000)
    cap = 20_000                                             # above the ordering pre-pass threshold (2^14 rays)
    rays32 = make_rays(prob, 6 * cap + 6_007)
    refs = {n: _oracle(prob).cast(rays32[:n], threads=8) for n in (3 * cap + 8_001, len(rays32))}

    def check(m, ref):
        st = m.get_stats()
        assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
        d = np.abs(m.read_tally() - ref.tally)
        bound = (1e-4 * np.abs(ref.tally) + 1e-7 * ref.tally.max()) if precision == 0 else (1e-10 * np.abs(ref.tally) + 1e-290)
        assert np.all(d <= bound)

    with _mr(prob, precision) as m:
        rays = np.ascontiguousarray(rays32.astype(m.ray_dtype))
        for mode in (2, 0, 1):
            m.set_option(MR_OPT_RING_MERGE, mode)
            assert m.get_option(MR_OPT_RING_MERGE) == mode
            # 3 full buffers + a partial one, pushed by one thread in ragged pieces
            n = 3 * cap + 8_001
            m.clear_tally()
            m.ring_open(4, cap)
            for i in range(0, n, 7_777):
                m.ring_push(rays[i:min(n, i + 7_777)])
            m.ring_flush()
            rs = m.ring_stats()
            assert rs["slots_shipped"] == 4 and rs["rays_pushed"] == n
            assert rs["casts"] == (1 if mode == 2 else 4 if mode == 0 else rs["casts"]) and 1 <= rs["casts"] <= 4
            check(m, refs[n])
            m.ring_close()
            # 6.3 buffers through 4 slots: the ring wraps while buffers are held back
            m.clear_tally()
            m.ring_open(4, cap)
            m.ring_push(rays)
            m.ring_flush()
            rs = m.ring_stats()
            assert rs["slots_shipped"] == 7
            if mode == 2:
                assert rs["casts"] == 2                      # slots 0-3 when slot 0 comes round again, then 0-2 at the flush
            if mode == 0:
                assert rs["casts"] == 7
            assert 2 <= rs["casts"] <= 7
            check(m, refs[len(rays)])
            m.ring_close()
            # four producer threads: buffers are shipped by whoever filled them, not necessarily in ring order
            m.clear_tally()
            m.ring_open(3, cap)
            bounds = np.linspace(0, len(rays), 5).astype(int)

            def produce(lo, hi):
                for i in range(lo, hi, 3_001):
                    m.ring_push(rays[i:min(hi, i + 3_001)])

            ts = [threading.Thread(target=produce, args=(bounds[k], bounds[k + 1])) for k in range(4)]
            for t in ts:
                t.start()
            for t in ts:
                t.join()
            m.ring_flush()
            assert m.ring_stats()["slots_shipped"] == 7
            check(m, refs[len(rays)])
            m.ring_close()
        from paper_1706_07476_b200 import MonteRayError

        m.ring_open(2, 4096)
        with pytest.raises(MonteRayError):
            m.set_option(MR_OPT_RING_MERGE, 0)               # not while a ring is open
        m.ring_close()


def test_ring_library_side_producers():
    """mr_ring_bench_producers (the bench's producers: C threads inside the library): the union of what 1, 3 and 7 producer
    threads push in ragged pieces equals one mr_cast_rays call (counters exact, tally within tolerance of the oracle); the
    dry run touches nothing; without an open ring it is a call-order error."""
    from paper_1706_07476_b200 import MonteRayError

    prob = make_problem(1)
    rays = make_rays(prob, 30_011)
    ref = _oracle(prob).cast(rays)
    with _mr(prob, 0) as m:
        with pytest.raises(MonteRayError):
            m.ring_bench_producers(rays, 2, 100)
        assert m.ring_bench_producers(rays, 2, 100, dry_run=True) >= 0.0
        assert not m.read_tally().any()
        for producers, piece in ((1, 4096), (3, 777), (7, 50)):
            m.clear_tally()
            m.ring_open(3, 4096)
            assert m.ring_bench_producers(rays, producers, piece) > 0.0
            tally = m.read_tally()
            st = m.get_stats()
            assert m.ring_stats()["rays_pushed"] == len(rays)
            m.ring_close()
            assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
            d = np.abs(tally - ref.tally)
            assert np.all(d <= 1e-4 * np.abs(ref.tally) + 1e-7 * ref.tally.max())


def test_ring_call_order_errors():
    from paper_1706_07476_b200 import MonteRay, MonteRayError

    prob = make_problem(1)
    with MonteRay(0, 0) as m:
        with pytest.raises(MonteRayError):
            m.ring_open(2, 4096)                 # nothing loaded
        m.load_problem(prob)
        with pytest.raises(MonteRayError):
            m.ring_push(make_rays(prob, 10))     # ring not open
        with pytest.raises(MonteRayError):
            m.ring_open(1, 4096)
        m.ring_open(2, 4096)
        with pytest.raises(MonteRayError):
            m.ring_open(2, 4096)                 # already open
        # set-up calls would free buffers the ring's ship path uses: refused while the ring is open
        with pytest.raises(MonteRayError):
            m.load_mesh(prob.xe, prob.ye, prob.ze)
        with pytest.raises(MonteRayError):
            m.load_materials(prob.density, prob.cell_mat, prob.cell_frac)
        with pytest.raises(MonteRayError):
            m.load_xs(0, *prob.xs[0])
        m.ring_push(make_rays(prob, 10))         # the ring still works
        m.ring_close()
        m.ring_close()                           # idempotent
        m.load_xs(0, *prob.xs[0])                # and set-up works again


# ------------------------------------------------------------------------------------- multi-nuclide materials (NEXT-4)
@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("cfg,kw,n", [(1, {}, 10_000), (3, {"nx": 68, "ny": 68, "nz": 40, "n_e": 3000}, 60_000),
                                      (5, {"n": 24, "n_e": 4000, "n_res": 50}, 30_000)])
def test_nuclide_mixtures_against_oracle(cfg, kw, n, precision):
    """Materials that are mixtures of nuclides on grids of different sizes, beside materials with their own table:
    cast tally, counters, traces, and the next-event detector sum against the oracle."""
    from workloads import add_nuclides

    prob = add_nuclides(make_problem(cfg, **kw), n_nuclides=6)
    assert any(mx is not None for mx in prob.mixtures) and any(mx is None for mx in prob.mixtures)
    rays32 = make_rays(prob, n)
    orc = _oracle(prob)
    ref = orc.cast(rays32, per_ray=True, threads=8)
    det = np.array([prob.xe[0] + 0.37 * (prob.xe[-1] - prob.xe[0]), prob.ye[0] + 0.61 * (prob.ye[-1] - prob.ye[0]),
                    prob.ze[0] + 0.55 * (prob.ze[-1] - prob.ze[0])])
    ne = orc.next_event(rays32, det)
    with _mr(prob, precision) as m:
        rays = rays32.astype(m.ray_dtype)
        m.cast_rays(rays)
        got = m.read_tally()
        st = m.get_stats()
        nseg, hsh, _, _ = m.trace_rays(rays)
        m.load_detectors(det)
        m.cast_next_event(rays)
        dsum = m.read_detectors()
    assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
    assert np.array_equal(nseg, ref.nseg) and np.array_equal(hsh, ref.hash)
    _close(got, ref.tally, precision, "tally")
    _close(dsum, [ne.det_sum], precision, "detector sum")


def test_nuclide_call_order_and_replacement():
    from paper_1706_07476_b200 import MonteRay, MonteRayError
    from workloads import add_nuclides

    base = make_problem(1)
    prob = add_nuclides(base, n_nuclides=4)
    rays = make_rays(base, 5000)
    ref_mix = _oracle(prob).cast(rays)
    ref_own = _oracle(base).cast(rays)
    with MonteRay(0, 0) as m:
        m.load_mesh(base.xe, base.ye, base.ze)
        with pytest.raises(MonteRayError) as e:
            m.define_material(1, [0], [1.0])
        assert e.value.status == 2                                     # materials first
        m.load_materials(base.density, base.cell_mat, base.cell_frac)
        m.load_xs(0, *base.xs[0])
        ids, w = prob.mixtures[1]
        with pytest.raises(MonteRayError):
            m.define_material(1, [99], [1.0])                          # nuclide index out of range
        with pytest.raises(MonteRayError):
            m.define_material(1, ids, -w)                              # negative weight
        m.define_material(1, ids, w)
        with pytest.raises(MonteRayError) as e:
            m.cast_rays(rays)
        assert e.value.status == 2 and "nuclide" in str(e.value)      # a named nuclide has no table yet
        for q, (en, sg) in enumerate(prob.nuclide_xs):
            m.load_nuclide_xs(q, en, sg)
        m.cast_rays(rays)
        _close(m.read_tally(), ref_mix.tally, 0, "mixture")
        m.load_xs(1, *base.xs[1])                                      # a table of its own replaces the mixture
        m.clear_tally()
        m.cast_rays(rays)
        _close(m.read_tally(), ref_own.tally, 0, "own table again")

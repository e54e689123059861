"""GPU parity: the CUDA library (through its C ABI / thin binding) against the CPU oracle, element by
element, on the same seeded inputs.

Bars (BASELINE.json north_star):
  * traces (segment count, FNV-1a hash of the cell sequence, and for small cases the full cell and
    length lists) bit-exact;
  * per-cell tallies |d| <= 1e-4*|oracle| + 1e-7*max(tally) in MIXED mode,
    |d| <= 1e-10*|oracle| (+1e-290 against denormals) in DOUBLE mode;
  * the kernel's segment / accepted / rejected counters equal the oracle's exactly.
"""
import numpy as np
import pytest

from tests.tiny import tiny_problem, tiny_rays
from workloads import make_problem, make_rays

pytestmark = pytest.mark.gpu


def _mr(prob, precision, **kw):
    from paper_1706_07476_b200 import MonteRay

    m = MonteRay(0, precision, **kw)
    m.load_problem(prob)
    return m


def _oracle(prob):
    from oracle.vrc_oracle import Oracle

    return Oracle(prob)


def _threads():
    import os

    return max(1, min(32, len(os.sched_getaffinity(0))))


def assert_tally(got, want, precision):
    d = np.abs(got - want)
    if precision == 0:
        bound = 1e-4 * np.abs(want) + 1e-7 * np.abs(want).max()
    else:
        bound = 1e-10 * np.abs(want) + 1e-290
    bad = np.flatnonzero(d > bound)
    assert bad.size == 0, (f"{bad.size} cells out of tolerance; worst cell {bad[np.argmax((d - bound)[bad])]}: "
                           f"got {got[bad[0]]!r} want {want[bad[0]]!r}")


def check_case(prob, rays32, precision, cap=0, threads=None, full_trace=False):
    """Casts + traces `rays32` on the GPU and on the oracle and compares everything."""
    orc = _oracle(prob)
    ref = orc.cast(rays32, per_ray=True, cap=cap, threads=threads or _threads())
    with _mr(prob, precision) as m:
        rays = rays32.astype(m.ray_dtype)
        n = m.cast_rays(rays)
        assert n == len(rays32)
        got = m.read_tally()
        st = m.get_stats()
        nseg, hsh, cells, lens = m.trace_rays(rays, cap=cap)
    assert np.array_equal(nseg, ref.nseg), "segment counts differ"
    assert np.array_equal(hsh, ref.hash), "cell-sequence hashes differ"
    if cap:
        assert np.array_equal(cells, ref.cells), "cell traces differ"
        assert np.array_equal(lens, ref.lens), "segment lengths differ (must be bitwise equal)"
    assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
    assert_tally(got, ref.tally, precision)
    return got, ref


# ------------------------------------------------------------------------------------- config 1 (full)
@pytest.mark.parametrize("precision", [0, 1])
def test_config1_full_traces_and_tally(precision):
    prob = make_problem(1)
    rays = make_rays(prob, 10_000)
    got, ref = check_case(prob, rays, precision, cap=32)
    assert ref.nseg.max() <= 32
    assert ref.segments == 71239  # tests/golden/config1_oracle.txt


# ------------------------------------------------------------------------------------- tiny random problems
@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("seed,K,M,uniform", [(101, 1, 2, False), (102, 2, 3, False), (103, 3, 4, True),
                                              (104, 4, 5, False), (105, 5, 6, False), (106, 8, 8, False),
                                              (107, 16, 9, True)])
def test_tiny_random_problems(seed, K, M, uniform, precision):
    """Every cell layout (K1..K4 packed, generic K=5/8/16), non-uniform planes, empty slots, void cells,
    axis-aligned and -0.0 directions; 3000 rays = several CTAs and a ragged last warp."""
    prob = tiny_problem(seed, nx=7, ny=5, nz=6, M=M, K=K, n_e=33, uniform=uniform)
    rays = tiny_rays(prob, seed, 3001, axis_aligned_share=0.1)
    check_case(prob, rays, precision, cap=24, threads=1)


def test_dense8_layout():
    """K = M = 8 with ids 0..7 in every cell selects the dense 32-byte record (config 5's layout)."""
    prob = tiny_problem(110, nx=6, ny=6, nz=6, M=8, K=8, n_e=65)
    prob.cell_mat[:] = np.arange(8, dtype=np.int32)[None, :]
    prob.cell_frac[:] = np.random.default_rng(110).random(prob.cell_frac.shape).astype(np.float32)
    rays = tiny_rays(prob, 110, 5000)
    check_case(prob, rays, 0, cap=24, threads=1)
    check_case(prob, rays, 1, threads=1)


def test_lattice_points_corners_and_faces():
    prob = tiny_problem(21, nx=4, ny=4, nz=4, uniform=True)
    rays = []
    for o in ([-1.0, -1.0, -1.0], [-0.25, -0.25, 0.5], [0.5, -0.25, -0.25], [-1.0, 0.5, 1.25]):
        for d in ([1, 1, 1], [1, 1, 0], [-1, 1, 1], [1, -1, -1], [0, 0, 1], [-1, -1, -1], [2, 1, 1], [0.0, -0.0, -1]):
            rays.append(o + d + [1.0, 1.0])
    rays = np.array(rays, dtype=np.float32)
    for precision in (0, 1):
        check_case(prob, rays, precision, cap=16, threads=1)


def test_rejection_rules_and_counters():
    prob = tiny_problem(81, uniform=True)  # box [-1,2] x [-1,1.25] x [-1,2.75]
    ok = [0.0, 0.0, 0.0, 0.6, 0.0, 0.8, 1.0, 1.0]
    rows = [ok]
    for f, v in ((0, np.nan), (4, np.inf), (6, 0.0), (6, -1.0), (7, np.nan), (0, 2.0), (1, -1.0000001), (2, 2.75), (7, -np.inf)):
        b = list(ok)
        b[f] = v
        rows.append(b)
    rows.append([0.0, 0.0, 0.0, 0.0, -0.0, 0.0, 1.0, 1.0])
    rows.append([-1.0, -1.0, -1.0, 0.6, 0.0, 0.8, 1.0, -2.5])  # on the lower faces, negative weight: accepted
    rays = np.array(rows * 40, dtype=np.float32)  # 480 rays: rejected lanes interleaved with live ones
    for precision in (0, 1):
        got, ref = check_case(prob, rays, precision, cap=12, threads=1)
        assert ref.rays_rejected == 40 * 10 and ref.rays_accepted == 40 * 2


# ------------------------------------------------------------------------------------- shaped workloads
@pytest.mark.parametrize("cfg,n_rays,kw", [
    (2, 200_000, {}),
    (3, 200_000, {}),
    (4, 100_000, {"n": 128, "n_e": 20_000}),
    (5, 200_000, {}),
])
def test_shaped_workloads_mixed(cfg, n_rays, kw):
    prob = make_problem(cfg, **kw)
    rays = make_rays(prob, n_rays)
    check_case(prob, rays, 0)


@pytest.mark.parametrize("cfg,n_rays,kw", [
    (2, 50_000, {"nx": 100, "ny": 100, "nz": 50}),
    (3, 50_000, {"nx": 85, "ny": 85, "nz": 60}),
    (4, 30_000, {"n": 64, "n_e": 5_000}),
    (5, 50_000, {"n_e": 50_000, "n_res": 500}),
])
def test_shaped_workloads_double(cfg, n_rays, kw):
    prob = make_problem(cfg, **kw)
    rays = make_rays(prob, n_rays)
    check_case(prob, rays, 1)


# ------------------------------------------------------------------------------------- full sizes, bench launch configuration
@pytest.mark.parametrize("cfg", [2, 3, 5, 4])
def test_full_size_configs_in_bench_configuration(cfg):
    """BASELINE.json's full sizes (config 4: one of its 10^6-ray batches on the full 512^3 mesh), library
    defaults = the launch configuration bench.py times (ray-ordering pre-pass on, device-resident batch):
    every ray's segment count and cell-sequence hash, the counters and the WHOLE tally against the oracle."""
    import torch

    from workloads import FULL_RAYS

    prob = make_problem(cfg)
    rays = make_rays(prob, FULL_RAYS[cfg])
    ref = _oracle(prob).cast(rays, per_ray=True, threads=_threads())
    with _mr(prob, 0) as m:
        d_rays = torch.from_numpy(rays).cuda()
        m.cast_rays(d_rays)
        got = m.read_tally()
        st = m.get_stats()
        nseg, hsh, _, _ = m.trace_rays(d_rays)
    assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
    assert np.array_equal(nseg, ref.nseg), "segment counts differ"
    assert np.array_equal(hsh, ref.hash), "cell-sequence hashes differ"
    assert_tally(got, ref.tally, 0)


CONFIG4_BATCHES = (0, 1, 9, 19, 29, 39, 49, 59, 69, 79, 89, 99)


@pytest.mark.slow
def test_config4_twelve_spaced_batches_on_the_full_mesh():
    """BASELINE.json config 4 is 10^8 rays in 100 batches of 10^6 on the 512^3 mesh.  The oracle needs about
    3.4e8 segments per batch (a few seconds on the host cores), so parity covers 12 OF THE 100 BATCHES, spaced over the
    whole run -- every batch has its own seeded stream, SeedSequence([.., 4, 9, batch]) -- each against its own oracle
    tally (every ray's segment count and cell-sequence hash, every cell of the batch's tally increment), then the
    twelve together (the resident tally is the running sum over batches)."""
    import torch

    prob = make_problem(4)
    orc = _oracle(prob)
    total = np.zeros(prob.ncell)
    with _mr(prob, 0) as m:
        seg = 0
        for batch in CONFIG4_BATCHES:
            rays = make_rays(prob, 1_000_000, batch=batch)
            ref = orc.cast(rays, per_ray=True, threads=_threads())
            d_rays = torch.from_numpy(rays).cuda()
            before = m.read_tally()
            m.cast_rays(d_rays)
            got = m.read_tally()
            nseg, hsh, _, _ = m.trace_rays(d_rays)
            assert np.array_equal(nseg, ref.nseg) and np.array_equal(hsh, ref.hash), f"batch {batch}: traces differ"
            assert_tally(got - before, ref.tally, 0)
            total += ref.tally
            seg += ref.segments
        st = m.get_stats()
        assert (st.rays_accepted, st.rays_rejected, st.segments) == (len(CONFIG4_BATCHES) * 1_000_000, 0, seg)
        assert_tally(m.read_tally(), total, 0)


# ------------------------------------------------------------------------------------- API behaviour
def test_host_device_and_chunked_staging_agree():
    import torch

    from paper_1706_07476_b200 import MR_OPT_STAGE_RAYS

    prob = make_problem(1)
    rays = make_rays(prob, 10_000)
    ref = _oracle(prob).cast(rays)
    with _mr(prob, 0) as m:
        m.cast_rays(torch.from_numpy(rays).cuda())          # device buffer
        t_dev = m.read_tally()
        m.clear_tally()
        m.set_option(MR_OPT_STAGE_RAYS, 1024)                # 10 chunks, ragged last one
        m.cast_rays(rays)                                     # pageable host buffer
        t_host = m.read_tally()
        st = m.get_stats()
        m.clear_tally()
        m.cast_rays(torch.from_numpy(rays).pin_memory())     # pinned host buffer
        t_pin = m.read_tally()
        m.clear_tally()
        assert m.cast_rays(rays[:0]) == 0                    # empty batch: no-op
        assert not m.read_tally().any()
        # additivity across calls: A then B == A u B
        m.cast_rays(rays[:3333])
        m.cast_rays(rays[3333:])
        t_ab = m.read_tally()
    assert st.segments == ref.segments and st.rays_accepted == 10_000
    for t in (t_dev, t_host, t_pin, t_ab):
        assert_tally(t, ref.tally, 0)
    np.testing.assert_allclose(t_host, t_dev, rtol=1e-12, atol=1e-14)


@pytest.mark.parametrize("precision", [0, 1])
def test_whole_batch_staging_of_back_to_back_host_batches(precision):
    """MR_OPT_WHOLE_BATCH: a page-locked host batch is DMA'd in one piece into one of two device buffers and cast in one launch
    (auto: when the stream is still busy with the previous batch).  Batches of different sizes back to back without waiting,
    the caller's buffer overwritten right after each call returns (it is consumed by then), forced on, forced off and auto:
    same counters, tally within tolerance of the oracle over the union."""
    import torch

    from paper_1706_07476_b200 import MR_OPT_STAGE_RAYS, MR_OPT_WHOLE_BATCH

    prob = make_problem(3, nx=68, ny=68, nz=40, n_e=2000)
    rays = make_rays(prob, 90_000)
    cuts = [0, 30_000, 30_500, 70_001, 90_000]
    ref = _oracle(prob).cast(rays, threads=_threads())
    with _mr(prob, precision) as m:
        m.set_option(MR_OPT_STAGE_RAYS, 2048)               # batches larger than a chunk: eligible for the whole-batch path
        host = torch.empty((40_000, 8), dtype=torch.float64 if precision else torch.float32).pin_memory()
        for mode in (1, 2, 0):
            m.set_option(MR_OPT_WHOLE_BATCH, mode)
            m.clear_tally()
            for a, b in zip(cuts[:-1], cuts[1:]):
                host[: b - a] = torch.from_numpy(rays[a:b].astype(m.ray_dtype))
                m.cast_rays(host[: b - a])                   # returns once the buffer has been copied out of
                host.fill_(float("nan"))                     # scribbling over it must not matter
            st = m.get_stats()
            assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
            assert_tally(m.read_tally(), ref.tally, precision)


def test_block_size_option_and_torch_stream():
    import torch

    from paper_1706_07476_b200 import MR_OPT_BLOCK_THREADS

    prob = make_problem(1)
    rays = make_rays(prob, 10_000)
    ref = _oracle(prob).cast(rays)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        with _mr(prob, 0) as m:
            for bt in (64, 128, 256):
                m.set_option(MR_OPT_BLOCK_THREADS, bt)
                m.clear_tally()
                m.cast_rays(rays)
                assert_tally(m.read_tally(), ref.tally, 0)


def test_call_order_and_argument_errors():
    from paper_1706_07476_b200 import MonteRay, MonteRayError

    prob = make_problem(1)
    rays = make_rays(prob, 100)
    with MonteRay(0, 0) as m:
        with pytest.raises(MonteRayError) as e:
            m.cast_rays(rays)
        assert e.value.status == 2  # MR_ERR_STATE: no mesh
        with pytest.raises(MonteRayError):
            m.load_mesh([0.0, 1.0, 1.0], [0.0, 1.0], [0.0, 1.0])  # not strictly increasing
        m.load_mesh(prob.xe, prob.ye, prob.ze)
        with pytest.raises(MonteRayError) as e:
            m.load_xs(0, prob.xs[0][0], prob.xs[0][1])
        assert e.value.status == 2  # materials first
        bad = prob.cell_mat.copy()
        bad[17, 0] = 5
        with pytest.raises(MonteRayError) as e:
            m.load_materials(prob.density, bad, prob.cell_frac)
        assert e.value.status == 1
        m.load_materials(prob.density, prob.cell_mat, prob.cell_frac)
        m.load_xs(0, *prob.xs[0])
        with pytest.raises(MonteRayError) as e:
            m.cast_rays(rays)
        assert e.value.status == 2 and "material 1" in str(e.value)
        with pytest.raises(MonteRayError):
            m.load_xs(1, prob.xs[1][0][::-1], prob.xs[1][1])  # decreasing grid
        m.load_xs(1, *prob.xs[1])
        m.cast_rays(rays)
        assert m.get_stats().rays_accepted == 100
        # the trace needs only the mesh; the context stays usable after argument errors
        nseg, _, _, _ = m.trace_rays(rays)
        assert nseg.sum() == m.get_stats().segments


def test_tally_tensor_view_is_the_resident_tally():
    prob = make_problem(1)
    rays = make_rays(prob, 2000)
    with _mr(prob, 0) as m:
        m.cast_rays(rays)
        m.sync()
        t = m.tally_tensor()
        assert t.is_cuda and t.numel() == prob.ncell
        assert np.array_equal(t.cpu().numpy(), m.read_tally())


def test_tally_tensor_all_reduce_in_a_world_of_one():
    """The one collective of the multi-GPU row: an NCCL fp64 sum all-reduce of tally_tensor().  Only one
    GPU is available here, so the group has ONE rank: this checks that the borrowed view is a tensor NCCL accepts and
    that the reduced view is still the resident tally -- not that two replicas add up (that runs on gloo, on the CPU)."""
    import torch
    import torch.distributed as dist

    if not dist.is_nccl_available():
        pytest.skip("torch built without NCCL")
    prob = make_problem(1)
    rays = make_rays(prob, 5000)
    created = False
    if not dist.is_initialized():
        dist.init_process_group("nccl", init_method="tcp://127.0.0.1:29537", rank=0, world_size=1)
        created = True
    try:
        with _mr(prob, 0) as m:
            m.cast_rays(rays)
            before = m.read_tally()
            t = m.tally_tensor()
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
            torch.cuda.synchronize()
            assert np.array_equal(t.cpu().numpy(), before)
            assert np.array_equal(m.read_tally(), before)
            m.cast_rays(rays)                                  # the view keeps following the resident tally
            m.sync()
            np.testing.assert_allclose(t.cpu().numpy(), 2.0 * before, rtol=1e-12)
    finally:
        if created:
            dist.destroy_process_group()


@pytest.mark.parametrize("precision", [0, 1])
def test_ray_ordering_prepass_on_and_off(precision):
    """MR_OPT_SORT_RAYS only changes which thread walks which ray: same counters, tally within tolerance
    either way; includes rejected rays (they get the last key) and a batch that is not a multiple of 256."""
    from paper_1706_07476_b200 import MR_OPT_SORT_RAYS

    prob = make_problem(3, nx=68, ny=68, nz=40, n_e=2000)
    rays = make_rays(prob, 70_001)
    rays[::1000, 6] = -1.0        # E <= 0: rejected
    rays[5::1000, 0] = 1.0e6      # origin outside the box: rejected
    ref = _oracle(prob).cast(rays, threads=_threads())
    assert ref.rays_rejected == 141
    with _mr(prob, precision) as m:
        r = rays.astype(m.ray_dtype)
        for sort in (0, 1):
            m.set_option(MR_OPT_SORT_RAYS, sort)
            m.clear_tally()
            before = m.get_stats().kernel_launches
            m.cast_rays(r)
            st = m.get_stats()
            assert st.kernel_launches - before == (6 if sort else 1)   # five ordering kernels + the cast
            assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
            assert_tally(m.read_tally(), ref.tally, precision)


def test_order_modes_give_the_same_result():
    """MR_OPT_ORDER_MODE (slab-major / longest first / auto) only permutes the work: counters identical,
    tally within tolerance of the oracle in every mode."""
    from paper_1706_07476_b200 import MR_OPT_ORDER_MODE

    prob = make_problem(2, nx=60, ny=60, nz=30, n_e=2000)
    rays = make_rays(prob, 50_003)
    ref = _oracle(prob).cast(rays, threads=_threads())
    with _mr(prob, 0) as m:
        assert m.get_option(MR_OPT_ORDER_MODE) == 0
        for mode in (1, 2, 0):
            m.set_option(MR_OPT_ORDER_MODE, mode)
            m.clear_tally()
            m.cast_rays(rays)
            st = m.get_stats()
            assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
            assert_tally(m.read_tally(), ref.tally, 0)
        from paper_1706_07476_b200 import MonteRayError
        with pytest.raises(MonteRayError):
            m.set_option(MR_OPT_ORDER_MODE, 3)


@pytest.mark.parametrize("fused", [1, 0])
def test_fused_in_record_tally_for_k4(fused):
    """MR_OPT_FUSED_TALLY: K = 4 records carry the score accumulators; every call that looks at the tally
    (read, device pointer / tensor view, end_batch, clear) first moves the in-record sums into the contiguous
    tally, so nothing observable changes.  Includes a materials reload between two casts (the sums survive)."""
    from paper_1706_07476_b200 import MR_OPT_FUSED_TALLY, MonteRay

    prob = make_problem(4, n=48, n_e=3000)
    rays = make_rays(prob, 40_001)
    ref = _oracle(prob).cast(rays, threads=_threads())
    with MonteRay(0, 0) as m:
        m.set_option(MR_OPT_FUSED_TALLY, fused)
        m.load_problem(prob)
        m.cast_rays(rays[:10_000])
        m.end_batch()
        m.cast_rays(rays[10_000:25_000])
        t_view = m.tally_tensor().cpu().numpy().copy()          # device view is up to date
        part = _oracle(prob).cast(rays[:25_000], threads=_threads())
        assert_tally(t_view, part.tally, 0)
        m.load_materials(prob.density, prob.cell_mat, prob.cell_frac)   # new records: pending sums must not be lost
        for k, (e, s) in enumerate(prob.xs):
            m.load_xs(k, e, s)
        m.cast_rays(rays[25_000:])
        m.end_batch()
        got = m.read_tally()
        s1, s2, nb = m.read_moments()
        st = m.get_stats()
        m.clear_tally()
        assert not m.read_tally().any()
        view = m.tally_tensor()
        m.cast_rays(rays[:10_000])                              # a cast AFTER the pointer was borrowed lands in the view
        m.sync()
        assert_tally(view.cpu().numpy(), _oracle(prob).cast(rays[:10_000], threads=_threads()).tally, 0)
        assert m.read_tally().any()
    assert nb == 2 and np.array_equal(s1, got)
    assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
    assert_tally(got, ref.tally, 0)


def test_tiled_mixture_index_on_off_and_fallback():
    """MR_OPT_TILED_INDEX: the dictionary + tiled 2-byte index path and the plain-record path give the same counters
    and tallies within tolerance of the oracle; meshes whose sides are not multiples of the 4 x 4 tile; a mesh with
    more than 1024 distinct records falls back to the plain records by itself."""
    from paper_1706_07476_b200 import MR_OPT_TILED_INDEX, MonteRay

    for seed, dims, K in ((601, (7, 5, 6), 1), (602, (9, 6, 5), 2), (603, (13, 11, 4), 3), (604, (12, 10, 9), 2)):
        prob = tiny_problem(seed, nx=dims[0], ny=dims[1], nz=dims[2], M=4, K=K, n_e=33)
        if seed == 603:      # few distinct records: a repeating pattern, as in a lattice
            prob.cell_mat[:] = prob.cell_mat[np.arange(prob.ncell) % 7]
            prob.cell_frac[:] = prob.cell_frac[np.arange(prob.ncell) % 7]
        rays = tiny_rays(prob, seed, 20_000, axis_aligned_share=0.05)
        ref = _oracle(prob).cast(rays, threads=_threads())
        tallies = []
        for tiled in (1, 0):
            with MonteRay(0, 0) as m:
                m.set_option(MR_OPT_TILED_INDEX, tiled)
                m.load_problem(prob)
                m.cast_rays(rays)
                st = m.get_stats()
                assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
                tallies.append(m.read_tally())
                assert_tally(tallies[-1], ref.tally, 0)
                if tiled:            # switching the option off after the load goes back to the plain records
                    m.set_option(MR_OPT_TILED_INDEX, 0)
                    m.clear_tally()
                    m.cast_rays(rays)
                    assert_tally(m.read_tally(), ref.tally, 0)
        np.testing.assert_allclose(tallies[0], tallies[1], rtol=1e-9, atol=1e-12 * ref.tally.max())


def test_coarse_block_records_on_off_and_detection():
    """MR_OPT_COARSE_RECORDS: compositions constant on aligned 2^s-cell blocks are read from one record per block.
    Same counters and tallies (within tolerance of the oracle) with the option on and off; mesh sides that are not
    multiples of the block; the block size found is the largest that holds; one odd cell anywhere lowers it."""
    from paper_1706_07476_b200 import MR_INFO_COARSE_SHIFT, MR_OPT_COARSE_RECORDS, MR_OPT_TILED_INDEX, MonteRay

    def blocky(seed, dims, block, K, M=5):
        prob = tiny_problem(seed, nx=dims[0], ny=dims[1], nz=dims[2], M=M, K=K, n_e=33)
        ix, iy, iz = np.meshgrid(np.arange(dims[0]), np.arange(dims[1]), np.arange(dims[2]), indexing="ij")
        rep = ((ix // block) * block + dims[0] * ((iy // block) * block + dims[1] * ((iz // block) * block)))
        rep = rep.transpose(2, 1, 0).reshape(-1)              # cell order: x fastest
        prob.cell_mat[:] = prob.cell_mat[rep]
        prob.cell_frac[:] = prob.cell_frac[rep]
        return prob

    cases = [(611, (40, 36, 32), 8, 4, 3), (612, (37, 41, 29), 4, 3, 2), (613, (64, 32, 16), 2, 1, 1), (614, (33, 33, 33), 16, 4, 4)]
    for seed, dims, block, K, want_shift in cases:
        prob = blocky(seed, dims, block, K)
        rays = tiny_rays(prob, seed, 30_000, axis_aligned_share=0.05)
        ref = _oracle(prob).cast(rays, threads=_threads())
        for coarse in (1, 0):
            with MonteRay(0, 0) as m:
                m.set_option(MR_OPT_COARSE_RECORDS, coarse)
                m.set_option(MR_OPT_TILED_INDEX, 0)            # else few distinct records would take the dictionary path
                m.load_problem(prob)
                assert m.get_option(MR_INFO_COARSE_SHIFT) == (want_shift if coarse else 0)
                assert (m.record_path() == "coarse_blocks") == bool(coarse)
                m.cast_rays(rays)
                st = m.get_stats()
                assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
                assert_tally(m.read_tally(), ref.tally, 0)
                if coarse:                                     # option off after the load: back to the per-cell records
                    m.set_option(MR_OPT_COARSE_RECORDS, 0)
                    assert m.record_path() != "coarse_blocks"
                    m.clear_tally()
                    m.cast_rays(rays)
                    assert_tally(m.read_tally(), ref.tally, 0)
    # one odd cell inside an 8-block: blocks of 8 and 4 no longer hold, blocks of 2 still do unless the cell sits in one
    prob = blocky(615, (40, 40, 32), 8, 4)
    c = 5 + 40 * (6 + 40 * 7)
    prob.cell_mat[c, 0] = (max(prob.cell_mat[c, 0], 0) + 1) % 5      # another material in slot 0 of that one cell
    with MonteRay(0, 0) as m:
        m.load_problem(prob)
        assert m.get_option(MR_INFO_COARSE_SHIFT) == 0
        rays = tiny_rays(prob, 615, 20_000)
        m.cast_rays(rays)
        assert_tally(m.read_tally(), _oracle(prob).cast(rays, threads=_threads()).tally, 0)


def test_cooperative_transposed_tally_adds():
    """MR_OPT_COOP_FLUSH: lanes stage (cell, score) for 8 steps, the warp adds them transposed (8 consecutive segments of
    4 rays per instruction).  Same counters, tallies within tolerance of the oracle, on every record path the kernel is
    built for (dictionary 4/8/16-bit, K = 1, K = 3 pairs, dense 8) and unchanged behaviour on the others; rejected rays,
    rays shorter than a window, a ragged last warp."""
    from paper_1706_07476_b200 import MR_OPT_COOP_FLUSH, MR_OPT_TILED_INDEX, MonteRay

    cases = []
    p3 = make_problem(3, nx=68, ny=68, nz=40, n_e=2000)
    cases.append((p3, make_rays(p3, 50_001), 1, "tiled4"))
    cases.append((p3, make_rays(p3, 50_001), 0, "k3_pairs"))
    p2 = make_problem(2, nx=60, ny=60, nz=30, n_e=2000)
    cases.append((p2, make_rays(p2, 40_003), 0, "k1"))
    p5 = make_problem(5, n=24, n_e=4000, n_res=50)
    cases.append((p5, make_rays(p5, 40_000), 1, "dense8"))
    pt = tiny_problem(631, nx=9, ny=8, nz=7, M=4, K=2, n_e=33)             # some 500 distinct records: 16-bit tiles
    cases.append((pt, tiny_rays(pt, 631, 20_001, axis_aligned_share=0.1), 1, "tiled16"))
    pk4 = tiny_problem(632, nx=9, ny=8, nz=7, M=5, K=4, n_e=33)            # a path the kernel is not built for
    cases.append((pk4, tiny_rays(pk4, 632, 10_001), 1, "k4"))
    for prob, rays, tiled, path in cases:
        rays[::501, 6] = -1.0
        ref = _oracle(prob).cast(rays, threads=_threads())
        with MonteRay(0, 0) as m:
            m.set_option(MR_OPT_TILED_INDEX, tiled)
            m.load_problem(prob)
            assert m.record_path() == path
            for coop in (1, 0, 3):                                            # 3: pairs by shuffle
                m.set_option(MR_OPT_COOP_FLUSH, coop)
                m.clear_tally()
                m.cast_rays(rays)
                st = m.get_stats()
                assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
                assert_tally(m.read_tally(), ref.tally, 0)


def test_read_tally_async_snapshots_in_stream_order():
    """mr_read_tally_async: a device snapshot taken in stream order and copied out on its own stream.  Batch after batch is
    cast from host memory with an asynchronous read after each (two alternating page-locked buffers, as bench.py's e2e loop
    does); after mr_sync each buffer holds the running tally as of ITS batch -- not a later one -- and equals what the
    blocking mr_read_tally returned at the same point of a second, blocking pass.  Also on a mesh whose scores live in
    in-record accumulators (fused K = 4), and after a mesh reload (the snapshot buffer follows the mesh)."""
    import torch

    from paper_1706_07476_b200 import MR_OPT_FUSED_TALLY, MonteRay

    for cfg, kw, fused in ((3, dict(nx=68, ny=68, nz=40, n_e=2000), 0), (4, dict(n=48, n_e=3000), 1)):
        prob = make_problem(cfg, **kw)
        rays = make_rays(prob, 60_000)
        parts = [rays[:25_000], rays[25_000:40_000], rays[40_000:]]
        with MonteRay(0, 0) as m:
            m.set_option(MR_OPT_FUSED_TALLY, fused)
            m.load_problem(prob)
            blocking = []
            for part in parts:
                m.cast_rays(part)
                blocking.append(m.read_tally())
            m.clear_tally()
            bufs = [torch.zeros(prob.ncell, dtype=torch.float64).pin_memory() for _ in range(3)]
            for part, buf in zip(parts, bufs):
                m.cast_rays(part)
                m.read_tally_async_into(buf.data_ptr())
            m.sync()
            ref = _oracle(prob).cast(rays, threads=_threads())
            for k, (buf, want) in enumerate(zip(bufs, blocking)):
                got = buf.numpy()
                np.testing.assert_allclose(got, want, rtol=1e-9, atol=1e-9 * want.max(), err_msg=f"snapshot {k}")
                assert k == 2 or not np.array_equal(got, bufs[2].numpy())       # an earlier snapshot is not the final tally
            assert_tally(bufs[2].numpy(), ref.tally, 0)
            assert_tally(m.read_tally(), ref.tally, 0)
            # the same buffer twice in a row: the second read waits for the first to leave the snapshot
            m.read_tally_async_into(bufs[0].data_ptr())
            m.read_tally_async_into(bufs[1].data_ptr())
            assert_tally(m.read_tally(), ref.tally, 0)                           # a blocking read completes the pending ones too
            assert np.array_equal(bufs[0].numpy(), bufs[1].numpy())
            small = make_problem(1)
            m.load_problem(small)                                                # new mesh: new snapshot buffer
            m.cast_rays(make_rays(small, 5000))
            out = torch.zeros(small.ncell, dtype=torch.float64).pin_memory()
            m.read_tally_async_into(out.data_ptr())
            m.sync()
            assert np.array_equal(out.numpy(), m.read_tally())


def test_tile_ordered_accumulators_of_the_dictionary_path():
    """MR_OPT_TILED_TALLY: cast_tiled_kernel walks in tile coordinates and adds into tile-ordered accumulators that are moved
    into the linear tally whenever it is looked at.  Same counters, tallies within tolerance of the oracle for 4-, 8- and
    16-bit index tiles, with and without the transposed adds, on meshes whose sides are not multiples of the tile, with
    non-uniform planes (plane table in shared memory), rejected rays and a ragged last warp; read / end_batch / clear see
    everything; once the device pointer has been borrowed the casts add straight into it (the view follows the tally)."""
    from paper_1706_07476_b200 import MR_OPT_COOP_FLUSH, MR_OPT_TILED_TALLY, MonteRay

    cases = []
    p3 = make_problem(3, nx=68, ny=68, nz=41, n_e=2000)                      # 12 distinct records: 4-bit tiles of 8 x 8, arithmetic mesh
    cases.append((p3, make_rays(p3, 50_001), "tiled4"))
    p2 = make_problem(2, nx=61, ny=59, nz=30, n_e=2000)                      # ragged tile edges
    cases.append((p2, make_rays(p2, 40_003), "tiled4"))
    p8 = tiny_problem(641, nx=13, ny=11, nz=6, M=4, K=3, n_e=33)             # repeating pattern of 100 records: 8-bit tiles of 8 x 4
    p8.cell_mat[:] = p8.cell_mat[np.arange(p8.ncell) % 100]
    p8.cell_frac[:] = p8.cell_frac[np.arange(p8.ncell) % 100]
    cases.append((p8, tiny_rays(p8, 641, 20_001, axis_aligned_share=0.1), "tiled8"))
    p16 = tiny_problem(642, nx=9, ny=8, nz=7, M=4, K=2, n_e=33)              # some 500 distinct records: 16-bit tiles of 4 x 4
    cases.append((p16, tiny_rays(p16, 642, 20_001, axis_aligned_share=0.1), "tiled16"))
    for seed, dims in ((643, (300, 9, 2)), (644, (9, 300, 2))):              # more than 256 cells along an axis (entry-word fields are 8 bits apart)
        pw = tiny_problem(seed, nx=dims[0], ny=dims[1], nz=dims[2], M=4, K=2, n_e=33)
        pw.cell_mat[:] = pw.cell_mat[np.arange(pw.ncell) % 11]
        pw.cell_frac[:] = pw.cell_frac[np.arange(pw.ncell) % 11]
        cases.append((pw, tiny_rays(pw, seed, 20_001, axis_aligned_share=0.1), "tiled4"))
    for prob, rays, path in cases:
        rays[::501, 6] = -1.0
        ref = _oracle(prob).cast(rays, threads=_threads())
        with MonteRay(0, 0) as m:
            m.set_option(MR_OPT_TILED_TALLY, 1)
            m.load_problem(prob)
            assert m.record_path() == path
            for coop in (1, 0):
                m.set_option(MR_OPT_COOP_FLUSH, coop)
                m.clear_tally()
                m.cast_rays(rays)
                st = m.get_stats()
                assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
                assert_tally(m.read_tally(), ref.tally, 0)
            m.clear_tally()
            assert not m.read_tally().any()
            half = len(rays) // 2
            m.cast_rays(rays[:half])
            m.end_batch()
            m.cast_rays(rays[half:])
            m.end_batch()
            s1, s2, nb = m.read_moments()
            assert nb == 2
            assert_tally(s1, ref.tally, 0)
            view = m.tally_tensor()                                          # borrowed: later casts add straight into it
            before = view.cpu().numpy().copy()
            assert_tally(before, ref.tally, 0)
            m.cast_rays(rays)
            m.sync()
            assert_tally(view.cpu().numpy(), 2.0 * ref.tally, 0)
            assert_tally(m.read_tally(), 2.0 * ref.tally, 0)


@pytest.mark.parametrize("coarse", [1, 0])
def test_deferred_tally_on_off_small_pool_and_pieces(coarse):
    """MR_OPT_DEFERRED_TALLY: phase A bins (cell, score) pairs by tally region, phase B adds them bin after bin.  Forced
    on a small mesh (auto needs a tally beyond twice the L2): same counters, tally within tolerance of the oracle, on
    the coarse-record and on the K = 4 record path; rejected rays, ragged batch sizes, a batch smaller than a warp; a
    pool far too small (most pairs take the direct path, counted by MR_INFO_DEFER_DIRECT_PAIRS) and a pool that makes
    the library cast the batch in several pieces; moments and the producer ring on top."""
    from paper_1706_07476_b200 import (MR_INFO_DEFER_DIRECT_PAIRS, MR_INFO_DEFERRED, MR_OPT_COARSE_RECORDS,
                                       MR_OPT_DEFER_POOL_ENTRIES, MR_OPT_DEFER_REGION_SHIFT, MR_OPT_DEFERRED_TALLY,
                                       MonteRay)

    prob = make_problem(4, n=64, n_e=3000)
    rays = make_rays(prob, 60_013)
    rays[::997, 6] = -1.0
    ref = _oracle(prob).cast(rays, threads=_threads())
    with MonteRay(0, 0) as m:
        m.set_option(MR_OPT_COARSE_RECORDS, coarse)
        m.load_problem(prob)
        assert m.get_option(MR_INFO_DEFERRED) == 0                  # auto: the tally fits in L2 many times over
        assert m.record_path() == ("coarse_blocks" if coarse else "k4")
        m.set_option(MR_OPT_DEFERRED_TALLY, 1)
        assert m.get_option(MR_INFO_DEFERRED) == 1
        seen = 0
        # regions of 2^12 cells (64 bins) with the pool sized by the library, then far too small (most pairs take the
        # direct path); regions of 2^15 cells (8 bins) and a pool that makes the library cast the batch in pieces; one region
        for shift, pool in ((12, 0), (12, 4096), (15, 1_800_000), (0, 0)):
            m.set_option(MR_OPT_DEFER_REGION_SHIFT, shift)
            m.set_option(MR_OPT_DEFER_POOL_ENTRIES, pool)
            m.clear_tally()
            m.cast_rays(rays)
            st = m.get_stats()
            assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
            assert_tally(m.read_tally(), ref.tally, 0)
            direct = m.get_option(MR_INFO_DEFER_DIRECT_PAIRS)
            if pool == 0:
                assert direct == 0
            if pool == 4096:
                assert direct > ref.segments // 2
        m.set_option(MR_OPT_DEFER_REGION_SHIFT, 12)
        m.set_option(MR_OPT_DEFER_POOL_ENTRIES, 0)
        # tiny batches, additivity, moments, the ring
        m.clear_tally()
        m.cast_rays(rays[:7])
        m.cast_rays(rays[7:20_000])
        m.end_batch()
        m.ring_open(2, 16384)
        m.ring_push(rays[20_000:])
        m.ring_close()
        m.end_batch()
        got = m.read_tally()
        s1, s2, nb = m.read_moments()
        st = m.get_stats()
        assert nb == 2 and np.array_equal(s1, got)
        assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
        assert_tally(got, ref.tally, 0)
        m.set_option(MR_OPT_DEFERRED_TALLY, 0)
        m.clear_tally()
        m.cast_rays(rays)
        assert_tally(m.read_tally(), ref.tally, 0)


@pytest.mark.parametrize("precision", [0, 1])
def test_warp_aggregated_atomics_for_the_first_segments(precision):
    """MR_OPT_AGGREGATE_FIRST: lanes of a warp that score into the same cell during a ray's first segments add one
    sum instead of many atomics (config 5's shape: every ray starts in a 4 x 4 x 4-cell region).  Counters and
    tallies are unchanged for 0, the default and a value larger than any ray."""
    from paper_1706_07476_b200 import MR_OPT_AGGREGATE_FIRST, MonteRay

    prob = make_problem(5, n=24, n_e=4000, n_res=50)
    rays = make_rays(prob, 60_000)
    rays[::97, 6] = -1.0                                   # rejected rays inside warps that aggregate
    ref = _oracle(prob).cast(rays, threads=_threads())
    with MonteRay(0, precision) as m:
        m.load_problem(prob)
        assert m.get_option(MR_OPT_AGGREGATE_FIRST) == 2
        r = rays.astype(m.ray_dtype)
        for a in (0, 2, 1000):
            m.set_option(MR_OPT_AGGREGATE_FIRST, a)
            m.clear_tally()
            m.cast_rays(r)
            st = m.get_stats()
            assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
            assert_tally(m.read_tally(), ref.tally, precision)


def test_paper_validation_metrics_single_against_double():
    """The paper's own check of single-precision ray casting on the GPU against double precision on the CPU (PAPER.md:116-124,
    Eqs. (7), (8); reported there: max relative difference 1.8e-5 on the PWR problem): the MIXED-mode tally on the
    full PWR-like mesh against the fp64 oracle, 8 batches of 250 000 rays.  Delta_phi(i) = |phi_cpu - phi_gpu| / phi_cpu over the
    cells whose relative standard deviation is below 5 % (the paper's filter), and eps_phi(i) = |phi_cpu - phi_gpu| / sigma(i)
    with sigma from the device's per-batch moments: the difference must be far inside the statistical noise."""
    import torch

    from oracle.vrc_oracle import fractional_difference, relative_difference

    prob = make_problem(3)
    orc = _oracle(prob)
    B, n = 8, 250_000
    total = np.zeros(prob.ncell)
    with _mr(prob, 0) as m:
        for b in range(B):
            rays = make_rays(prob, n, batch=b)
            total += orc.cast(rays, threads=_threads()).tally
            m.cast_rays(torch.from_numpy(rays).cuda())
            m.end_batch()
        phi_gpu = m.read_tally()
        mean, sigma, nb = m.read_mean_sigma()
    assert nb == B
    sigma_total = sigma * B                                   # standard deviation of the summed tally
    # both sides cast the SAME rays, so the difference is arithmetic, not statistical: every cell that was scored counts
    # (2 10^6 rays leave few cells below the paper's 5 % uncertainty filter; cells below 1e-3 of the largest tally are left to
    # the absolute term of the parity tolerance)
    good = (total >= 1e-3 * total.max()) & (sigma_total > 0)
    assert good.sum() > 0.5 * prob.ncell
    d_phi = relative_difference(total, phi_gpu)[good]
    e_phi = fractional_difference(total, phi_gpu, sigma_total)[good]
    print(f"Eq. (7) max Delta_phi {d_phi.max():.3e} (mean {d_phi.mean():.3e}) over {int(good.sum())} cells; "
          f"Eq. (8) max eps_phi {e_phi.max():.3e} (mean {e_phi.mean():.3e})")
    assert d_phi.max() <= 1e-4          # north_star's relative bar; the paper's Titan X run printed 1.8e-5
    assert e_phi.max() <= 1e-2          # at most a hundredth of a standard deviation

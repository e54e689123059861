"""mr_cast_rays_static: the cast for hosts that must not allocate device memory inside their loop.

Who needs it: a transport code that gives the whole GPU to its own memory pool at start-up (nothing is left for a
library to allocate from), a host loop that cannot take the device-wide stall of a cudaMalloc / cudaFree in the
middle of its CPU/GPU overlap, or a job with a fixed per-process memory budget.  The ordinary mr_cast_rays allocates
(and re-allocates, when a batch is larger than any before) the scratch of its ray-ordering pre-pass; the static
entry point runs the same pre-pass in a fixed 2.1 MB array that is part of libmonteray.so, takes at most
MR_STATIC_MAX_RAYS rays per call, and shares that one array between all callers on a GPU.

What is checked here, on two calls in a row per case (the second smaller than the first, so the array still holds
the first call's leftovers beyond the part the second one uses):
  * the tally equals the ordinary path's within the parity tolerance of the other GPU tests, and the ray / segment
    counters are equal exactly (the two paths differ only in the order in which threads pick up rays);
  * neither the context's allocator nor the CUDA driver saw an allocation or a release during the calls;
  * oversized batches, host buffers and a context whose set-up is unfinished are refused with a clear error.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure in this add-on must not
hide the parity suite.  Each test builds its own contexts, so the file passes alone as well as after the others.
"""
import numpy as np
import pytest

from workloads import make_problem, make_rays

pytestmark = pytest.mark.gpu


def assert_tally(got, want, precision):
    """The bar of tests/test_gpu_parity.py (north_star): 1e-4 relative + 1e-7 of the peak in MIXED, 1e-10 in DOUBLE."""
    d = np.abs(got - want)
    bound = 1e-4 * np.abs(want) + 1e-7 * np.abs(want).max() if precision == 0 else 1e-10 * np.abs(want) + 1e-290
    bad = np.flatnonzero(d > bound)
    assert bad.size == 0, f"{bad.size} cells out of tolerance, first: got {got[bad[0]]!r} want {want[bad[0]]!r}"


def _context(prob, precision, deferred_off=True):
    from paper_1706_07476_b200 import MR_OPT_DEFERRED_TALLY, MonteRay

    m = MonteRay(0, precision)
    m.load_problem(prob)
    if deferred_off:
        m.set_option(MR_OPT_DEFERRED_TALLY, 0)
    return m


def _finish_setup(m, rays_dev):
    """All allocation belongs to set-up: one ordinary one-ray cast creates the table-descriptor buffers."""
    m.cast_rays(rays_dev[:1].contiguous())
    m.clear_tally()          # also zeroes the ray / segment counters
    m.sync()


def _footprint(m, torch, driver=False):
    """What the context's allocator holds and what torch's pool has reserved; with driver=True also the free memory the
    CUDA driver reports (only comparable once every kernel of the path has run: the first launch of a kernel loads
    its code onto the device)."""
    torch.cuda.synchronize()
    return (tuple(sorted(m._allocator._live)), torch.cuda.memory_reserved(0)) + ((torch.cuda.mem_get_info(0)[0],) if driver else ())


@pytest.mark.parametrize("config,precision,n_first,n_second", [
    (1, 1, 40_000, 17_000),         # all-double, non-tiled records, tiny mesh (heavily contended tally)
    (2, 0, 200_000, 70_001),        # K = 1 records, 4e6 cells
    (3, 0, 262_144, 100_003),       # dictionary tiles; first call exactly at MR_STATIC_MAX_RAYS
])
def test_static_cast_matches_ordinary_cast_on_two_calls_in_a_row(config, precision, n_first, n_second):
    import torch

    from paper_1706_07476_b200 import MR_STATIC_MAX_RAYS

    assert n_first <= MR_STATIC_MAX_RAYS
    prob = make_problem(config)
    rays = make_rays(prob, n_first + n_second, dtype=np.float64 if precision == 1 else np.float32)
    with _context(prob, precision) as ref, _context(prob, precision) as m:
        dt = torch.float64 if precision == 1 else torch.float32
        dev = torch.from_numpy(np.ascontiguousarray(rays.astype(ref.ray_dtype))).to("cuda:0").to(dt).reshape(-1, 8).contiguous()
        a, b = dev[:n_first].contiguous(), dev[n_first:].contiguous()
        _finish_setup(m, dev)

        before = _footprint(m, torch)
        m.cast_rays_static(a)
        got_a = m.read_tally()
        st_a = m.get_stats()
        between = _footprint(m, torch, driver=True)
        m.cast_rays_static(b)
        got_ab = m.read_tally()
        st_ab = m.get_stats()
        assert _footprint(m, torch) == before, "mr_cast_rays_static went to the context's allocator"
        assert _footprint(m, torch, driver=True) == between, "the driver's free memory changed across mr_cast_rays_static"

        ref.cast_rays(a)
        want_a = ref.read_tally()
        rs_a = ref.get_stats()
        ref.cast_rays(b)
        want_ab = ref.read_tally()
        rs_ab = ref.get_stats()

    assert want_a.max() > 0.0
    assert (st_a.rays_accepted, st_a.rays_rejected, st_a.segments) == (rs_a.rays_accepted, rs_a.rays_rejected, rs_a.segments)
    assert (st_ab.rays_accepted, st_ab.rays_rejected, st_ab.segments) == (rs_ab.rays_accepted, rs_ab.rays_rejected, rs_ab.segments)
    assert st_a.rays_accepted + st_a.rays_rejected == n_first
    assert st_ab.rays_accepted + st_ab.rays_rejected == n_first + n_second
    assert_tally(got_a, want_a, precision)
    assert_tally(got_ab, want_ab, precision)


def test_static_and_ordinary_casts_mix_on_one_context():
    """The two entry points add to the same tally; alternating them equals the ordinary path alone."""
    import torch

    prob = make_problem(2)
    rays = make_rays(prob, 90_000).astype(np.float32)
    dev = torch.from_numpy(rays).to("cuda:0").reshape(-1, 8).contiguous()
    parts = [dev[:30_000].contiguous(), dev[30_000:60_000].contiguous(), dev[60_000:].contiguous()]
    with _context(prob, 0) as ref, _context(prob, 0) as m:
        _finish_setup(m, dev)
        m.cast_rays_static(parts[0])
        m.cast_rays(parts[1])
        m.cast_rays_static(parts[2])
        got = m.read_tally()
        ref.cast_rays(dev)
        want = ref.read_tally()
        assert m.get_stats().segments == ref.get_stats().segments
    assert_tally(got, want, 0)


def test_static_cast_refuses_what_it_cannot_do():
    import torch

    from paper_1706_07476_b200 import (MR_ERR_INVALID_ARG, MR_ERR_STATE, MR_ERR_UNSUPPORTED, MR_INFO_DEFERRED,
                                       MR_OPT_DEFERRED_TALLY, MR_STATIC_MAX_RAYS, MonteRayError)

    prob = make_problem(1)
    rays = make_rays(prob, 1000).astype(np.float32)
    dev = torch.from_numpy(rays).to("cuda:0").reshape(-1, 8).contiguous()
    with _context(prob, 0) as m:
        # set-up not finished: the descriptor buffers do not exist yet, and this call will not create them
        with pytest.raises(MonteRayError) as e:
            m.cast_rays_static(dev)
        assert e.value.status == MR_ERR_STATE and "set-up" in str(e.value)
        _finish_setup(m, dev)
        assert m.cast_rays_static(dev[:0].contiguous()) == 0          # n = 0: no-op
        m.cast_rays_static(dev)
        # more rays than the fixed array holds
        big = torch.zeros((MR_STATIC_MAX_RAYS + 1, 8), dtype=torch.float32, device="cuda:0")
        with pytest.raises(MonteRayError) as e:
            m.cast_rays_static(big)
        assert e.value.status == MR_ERR_INVALID_ARG and str(MR_STATIC_MAX_RAYS) in str(e.value)
        # host buffers are the binding's to refuse (the C call takes a device pointer only)
        with pytest.raises(MonteRayError):
            m.cast_rays_static(rays)
        # the deferred tally sizes a pool per batch: not from here
        m.set_option(MR_OPT_DEFERRED_TALLY, 1)
        if m.get_option(MR_INFO_DEFERRED):
            with pytest.raises(MonteRayError) as e:
                m.cast_rays_static(dev)
            assert e.value.status == MR_ERR_UNSUPPORTED
        m.set_option(MR_OPT_DEFERRED_TALLY, 0)
        # the refusals left the context usable
        m.cast_rays_static(dev)
        assert m.get_stats().rays_accepted + m.get_stats().rays_rejected == 2 * len(rays)

"""The deferred two-phase tally (MR_OPT_DEFERRED_TALLY, mr_defer.cuh) under the host-side machinery around it.

Its control words, chunk table and pair pool exist once per context, so (a) the chunks of a staged host batch must not
run on two streams at once, (b) the pool must not be released while a chunk still uses it, and (c) a mesh with a
different number of tally regions must not inherit the chunk table of the previous one.  Each case is compared with the
CPU oracle: counters exact, tally within the MIXED-mode bar of tests/test_gpu_parity.py.
"""
import numpy as np
import pytest

from tests.test_gpu_parity import _oracle, _threads, assert_tally
from workloads import make_problem, make_rays

pytestmark = pytest.mark.gpu


def _counters(st):
    return (st.rays_accepted, st.rays_rejected, st.segments)


@pytest.mark.parametrize("coarse", [1, 0])
def test_deferred_tally_with_host_batches_cut_into_many_chunks(coarse):
    """Pageable and page-locked host batches that the library stages in 4 to 7 chunks (ragged last one), with the pool
    sized by the library (it has to grow in the middle of a batch when the chunks get longer), fixed and small (chunks cast
    in pieces), and far too small (direct adds); whole-batch staging forced on, off and auto; batches back to back without
    a wait in between."""
    import torch

    from paper_1706_07476_b200 import (MR_INFO_DEFERRED, MR_OPT_COARSE_RECORDS, MR_OPT_DEFER_POOL_ENTRIES,
                                       MR_OPT_DEFER_REGION_SHIFT, MR_OPT_DEFERRED_TALLY, MR_OPT_STAGE_RAYS,
                                       MR_OPT_WHOLE_BATCH, MonteRay)

    prob = make_problem(4, n=64, n_e=3000)
    rays = make_rays(prob, 60_013)
    rays[::991, 6] = -1.0                                        # some rejected rays in every chunk
    ref = _oracle(prob).cast(rays, threads=_threads())
    want = (ref.rays_accepted, ref.rays_rejected, ref.segments)
    pinned = torch.from_numpy(rays).pin_memory()
    with MonteRay(0, 0) as m:
        m.set_option(MR_OPT_COARSE_RECORDS, coarse)
        m.load_problem(prob)
        m.set_option(MR_OPT_DEFERRED_TALLY, 1)
        m.set_option(MR_OPT_DEFER_REGION_SHIFT, 12)             # 64 regions
        assert m.get_option(MR_INFO_DEFERRED) == 1
        m.cast_rays(rays[:7])                                    # the pool starts at its smallest size
        m.clear_tally()
        for stage, pool, whole in ((16384, 0, 0), (4096, 0, 0), (4096, 300_000, 0), (4096, 4096, 0), (4096, 0, 1), (16384, 0, 2)):
            m.set_option(MR_OPT_STAGE_RAYS, stage)              # chunks of stage/4, stage/2, stage, 2 stage, 2 stage, ...
            m.set_option(MR_OPT_DEFER_POOL_ENTRIES, pool)
            m.set_option(MR_OPT_WHOLE_BATCH, whole)
            for batch in (rays, pinned):
                m.clear_tally()
                m.cast_rays(batch)
                assert _counters(m.get_stats()) == want, (stage, pool, whole)
                assert_tally(m.read_tally(), ref.tally, 0)
            # two batches back to back: the second is staged while the first one's chunks are still running
            m.clear_tally()
            m.cast_rays(pinned[:25_000])
            m.cast_rays(pinned[25_000:])
            assert _counters(m.get_stats()) == want, (stage, pool, whole)
            assert_tally(m.read_tally(), ref.tally, 0)


def test_deferred_tally_across_a_mesh_reload():
    """One context, three meshes in a row with 8, 64 and 1 tally regions: the chunk table and the pool estimate of a mesh
    are not carried over to the next (the table has one row per region)."""
    from paper_1706_07476_b200 import (MR_INFO_DEFER_DIRECT_PAIRS, MR_INFO_DEFERRED, MR_OPT_DEFER_REGION_SHIFT,
                                       MR_OPT_DEFERRED_TALLY, MonteRay)

    with MonteRay(0, 0) as m:
        m.set_option(MR_OPT_DEFERRED_TALLY, 1)
        m.set_option(MR_OPT_DEFER_REGION_SHIFT, 12)
        for n_mesh, n_rays in ((32, 30_011), (64, 20_003), (16, 9_001)):
            prob = make_problem(4, n=n_mesh, n_e=2000)
            rays = make_rays(prob, n_rays)
            ref = _oracle(prob).cast(rays, threads=_threads())
            m.load_problem(prob)
            assert m.get_option(MR_INFO_DEFERRED) == 1
            m.cast_rays(rays)
            assert _counters(m.get_stats()) == (ref.rays_accepted, ref.rays_rejected, ref.segments), n_mesh
            assert_tally(m.read_tally(), ref.tally, 0)
            assert m.get_option(MR_INFO_DEFER_DIRECT_PAIRS) == 0
            # a second, smaller batch on the same mesh reuses the pool as it is
            m.clear_tally()
            m.cast_rays(rays[: n_rays // 3])
            ref3 = _oracle(prob).cast(rays[: n_rays // 3], threads=_threads())
            assert_tally(m.read_tally(), ref3.tally, 0)

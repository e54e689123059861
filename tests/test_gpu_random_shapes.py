"""GPU parity on RANDOM MESH SHAPES through every cast variant (seeded; `-m gpu`, through the C ABI, against the CPU oracle).

The shaped configs and the hand-picked tiny cases fix the mesh proportions; this sweep draws them: one long axis of 1, 2,
255, 256, 257, 300, 513 or 700 cells (index fields of the tile / block kernels are 8 bits apart; sides that are not
multiples of a tile or block) beside two short ones, K in {1, 2, 3, 4, 8}, uniform and non-uniform planes, compositions
that repeat with period 1 ... 200 (dictionary paths of every index width, or none) or are constant in 2^s blocks (block
records), and for each problem every cast variant the library has: defaults, transposed adds on / off / by pairs,
tile-ordered accumulators, the deferred tally, persistent lanes, plain records; MIXED and DOUBLE.  Checked per case: every
ray's segment count and cell-sequence hash (bit-exact), the counters, the whole tally within the mode's tolerance, and the
next-event cell sequences and detector sums for a detector inside and one outside the mesh.
"""
import numpy as np
import pytest

from tests.tiny import tiny_problem, tiny_rays

pytestmark = pytest.mark.gpu


def _tol(ref, precision):
    return (1e-4 * np.abs(ref) + 1e-7 * ref.max()) if precision == 0 else (1e-10 * np.abs(ref) + 1e-290)


@pytest.mark.parametrize("seed", [11, 12, 13])
def test_random_shapes_every_cast_variant(seed):
    from oracle.vrc_oracle import Oracle
    from paper_1706_07476_b200 import (MR_OPT_COARSE_RECORDS, MR_OPT_COOP_FLUSH, MR_OPT_DEFERRED_TALLY,
                                       MR_OPT_TILED_INDEX, MR_OPT_TILED_TALLY, MonteRay)

    g = np.random.default_rng(seed)
    variants = ({}, {MR_OPT_COOP_FLUSH: 1}, {MR_OPT_COOP_FLUSH: 0}, {MR_OPT_COOP_FLUSH: 3}, {MR_OPT_TILED_TALLY: 1, MR_OPT_COOP_FLUSH: 1},
                {MR_OPT_DEFERRED_TALLY: 1}, {MR_OPT_TILED_INDEX: 0, MR_OPT_COARSE_RECORDS: 0})
    before_load = (MR_OPT_TILED_INDEX, MR_OPT_COARSE_RECORDS)
    paths = set()
    for it in range(12):
        big = int(g.integers(0, 3))
        dims = [int(g.integers(1, 12)) for _ in range(3)]
        dims[big] = int(g.choice([1, 2, 255, 256, 257, 300, 513, 700]))
        K = int(g.choice([1, 2, 3, 4, 8]))
        M = 8 if K == 8 else int(g.integers(max(2, K), 6))
        npat = int(g.choice([1, 3, 11, 16, 17, 200, 0]))
        block = int(g.choice([0, 0, 2, 4]))
        prob = tiny_problem(100 * seed + it, nx=dims[0], ny=dims[1], nz=dims[2], M=M, K=K, n_e=33, uniform=bool(g.integers(0, 2)))
        if npat:
            prob.cell_mat[:] = prob.cell_mat[np.arange(prob.ncell) % npat]
            prob.cell_frac[:] = prob.cell_frac[np.arange(prob.ncell) % npat]
        if block:      # compositions constant in aligned blocks of `block` cells per axis
            c = np.arange(prob.ncell)
            ix, iy, iz = c % dims[0], (c // dims[0]) % dims[1], c // (dims[0] * dims[1])
            src = (ix // block * block) + dims[0] * ((iy // block * block) + dims[1] * (iz // block * block))
            prob.cell_mat[:] = prob.cell_mat[src]
            prob.cell_frac[:] = prob.cell_frac[src]
        rays = tiny_rays(prob, 100 * seed + it, 12_011, axis_aligned_share=0.1)
        orc = Oracle(prob)
        ref = orc.cast(rays, per_ray=True, threads=8)
        dets = np.array([[0.3, 0.2, 0.7], [float(prob.xe[-1]) + 1.0, 0.1, 0.2]])
        ne = [orc.next_event(rays[:2000], d) for d in dets]
        for precision in (0, 1):
            for opts in variants if precision == 0 else ({},):
                what = f"seed {seed} case {it}: dims {dims} K {K} period {npat} block {block} precision {precision} options {opts}"
                with MonteRay(0, precision) as m:
                    for k, v in opts.items():
                        if k in before_load:
                            m.set_option(k, v)
                    m.load_problem(prob)
                    for k, v in opts.items():
                        m.set_option(k, v)
                    paths.add(m.record_path())
                    r = rays.astype(m.ray_dtype)
                    m.cast_rays(r)
                    tally = m.read_tally()
                    st = m.get_stats()
                    nseg, hsh, _, _ = m.trace_rays(r)
                    assert np.array_equal(nseg, ref.nseg) and np.array_equal(hsh, ref.hash), what
                    assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments), what
                    assert np.all(np.abs(tally - ref.tally) <= _tol(ref.tally, precision)), what
                    m.load_detectors(dets)
                    m.cast_next_event(r[:2000])
                    sums = m.read_detectors()
                    for j, rn in enumerate(ne):
                        ns, hs, _, _ = m.trace_next_event(r[:2000], j)
                        assert np.array_equal(ns, rn.nseg) and np.array_equal(hs, rn.hash), what + f" next-event detector {j}"
                    want = np.array([rn.det_sum for rn in ne])
                    assert np.all(np.abs(sums - want) <= (1e-4 if precision == 0 else 1e-10) * np.abs(want) + 1e-300), what
    assert len(paths) >= 4, paths      # the draw reached several record paths


@pytest.mark.parametrize("seed", [21, 22])
def test_random_rz_and_spherical_shapes(seed):
    """R-Z and spherical meshes of random proportions (1 ... 300 shells, 1 ... 40 slabs, uniform and non-uniform radii), every
    record layout, both modes: cells AND lengths of every ray bit-exact (the kernel finds the turning shell by bisection and
    evaluates one discriminant per step -- every decision must still be the oracle's), counters, tallies, and the next-event
    cell sequences and sums for a detector inside and one outside."""
    from tests.test_gpu_rz import _check, _check_next_event_rz
    from tests.tiny import tiny_rz_problem, tiny_rz_rays, tiny_sphere_problem, tiny_sphere_rays

    g = np.random.default_rng(seed)
    for it in range(8):
        nr = int(g.choice([1, 2, 3, 17, 64, 129, 300]))
        nz = int(g.choice([1, 2, 5, 40]))
        K = int(g.choice([1, 2, 3, 4, 8]))
        M = 8 if K == 8 else int(g.integers(max(2, K), 6))
        uniform = bool(g.integers(0, 2))
        if g.integers(0, 3) == 0:
            prob = tiny_sphere_problem(100 * seed + it, nr=nr, M=M, K=K, n_e=33, uniform=uniform)
            rays = tiny_sphere_rays(prob, 100 * seed + it, 6001, through_centre_share=0.05)
            sphere = True
        else:
            prob = tiny_rz_problem(100 * seed + it, nr=nr, nz=nz, M=M, K=K, n_e=33, uniform=uniform)
            rays = tiny_rz_rays(prob, 100 * seed + it, 6001, axis_parallel_share=0.05, through_axis_share=0.05)
            sphere = False
        R = float(prob.re[-1])
        dets = [[0.3 * R, 0.1 * R, 0.2], [2.0 * R, 0.5 * R, -3.0]]
        for precision in (0, 1):
            if sphere:
                from oracle.vrc_oracle import Oracle
                from paper_1706_07476_b200 import MonteRay

                cap = 2 * nr + 1
                ref = Oracle(prob).cast_sphere(rays, prob.re, cap=cap)
                with MonteRay(0, precision) as m:
                    m.load_problem(prob)
                    r = rays.astype(m.ray_dtype)
                    m.cast_rays(r)
                    got = m.read_tally()
                    st = m.get_stats()
                    nseg, hsh, cells, lens = m.trace_rays(r, cap=cap)
                assert np.array_equal(nseg, ref.nseg) and np.array_equal(hsh, ref.hash)
                assert np.array_equal(cells, ref.cells) and np.array_equal(lens, ref.lens)
                assert (st.rays_accepted, st.rays_rejected, st.segments) == (ref.rays_accepted, ref.rays_rejected, ref.segments)
                assert np.all(np.abs(got - ref.tally) <= _tol(ref.tally, precision))
            else:
                _check(prob, rays, precision, cap=2 * nr + nz + 2)
            _check_next_event_rz(prob, rays[:1500], dets, precision, sphere)

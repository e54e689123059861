"""The N > 1 path on CPU: world_size-2 gloo run of the replica plumbing (paper_1706_07476_b200/multi.py).
Each rank casts its contiguous shard of one batch with the CPU oracle (test infrastructure) into a private
tally; one fp64 sum all-reduce must reproduce the single-process tally."""
import os
import socket

import numpy as np
import torch
import torch.multiprocessing as mp

from workloads import make_problem, make_rays


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank),
                      WORLD_SIZE=str(world))
    from oracle.vrc_oracle import Oracle
    from paper_1706_07476_b200 import multi

    assert multi.env_rank_world() == (rank, rank, world)
    dist = multi.init_process_group("gloo")
    prob = make_problem(1)
    rays = make_rays(prob, 4001)
    lo, hi = multi.ray_shard(len(rays), rank, world)
    res = Oracle(prob).cast(rays[lo:hi])
    t = torch.from_numpy(res.tally.copy())
    multi.allreduce_sum_(t)
    segs = multi.sum_over_ranks(res.segments)
    slow = multi.max_over_ranks(10.0 + rank)
    assert multi.batch_of_rank(3, rank, world) == 3 * world + rank
    if rank == 0:
        np.save(os.path.join(out_dir, "tally.npy"), t.numpy())
        np.save(os.path.join(out_dir, "meta.npy"), np.array([segs, slow, hi - lo]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_replicas_sum_to_the_single_tally(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    from oracle.vrc_oracle import Oracle

    prob = make_problem(1)
    rays = make_rays(prob, 4001)
    ref = Oracle(prob).cast(rays)
    got = np.load(tmp_path / "tally.npy")
    segs, slow, n0 = np.load(tmp_path / "meta.npy")
    np.testing.assert_allclose(got, ref.tally, rtol=1e-13, atol=0)
    assert int(segs) == ref.segments and slow == 11.0 and int(n0) == 2000


def test_shards_cover_the_batch_exactly():
    from paper_1706_07476_b200 import multi

    for n in (0, 1, 7, 4001, 10_000_000):
        for world in (1, 2, 3, 8):
            cuts = [multi.ray_shard(n, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            assert all(cuts[i][1] == cuts[i + 1][0] for i in range(world - 1))
    assert sorted(multi.batch_of_rank(s, r, 4) for s in range(3) for r in range(4)) == list(range(12))

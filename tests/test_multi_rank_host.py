"""The N > 1 path of bench.py on CPU: two gloo ranks ("replicas only").

Tracks are the independent units of the Eq. 1.1 stage: each rank takes its own slice of the
seeded track list, there is no data-path collective, and the reported numbers are the MAX over ranks of the
times and the SUM of the work."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import bench
    from wtide_inputs import carriers_on_tracks, geometry_desc, make_tracks, reduced_desc, straight_drift_cfg0
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        d = reduced_desc(geometry_desc(1), nt=16)
        per_rank = 3
        all_tracks = make_tracks(1, per_rank * world, d, 10.0)
        mine = all_tracks[bench.shard_tracks(per_rank, world, rank)]
        start, sign, charge, toff = carriers_on_tracks(mine, 8, d)
        csr = straight_drift_cfg0(d, start, sign, charge, toff, max_steps=d["nt"], speed=100.0)
        terms = bench.count_terms(csr["carrier_step_offsets"], d["nt"])
        times = [10.0 + rank, 5.0 - rank, 20.0 + 2 * rank, 1.0]
        red, total = bench.reduce_over_ranks(times, terms, world, "cpu")
        # every rank holds the same reduced numbers
        gathered = [None] * world
        dist.all_gather_object(gathered, (red, total, terms, np.asarray(mine).tolist()))
        if rank == 0:
            np.save(os.path.join(out_dir, "ok.npy"), np.array([1]))
            assert all(g[0] == gathered[0][0] and g[1] == gathered[0][1] for g in gathered)
            assert red == [10.0 + world - 1, 5.0, 20.0 + 2 * (world - 1), 1.0]
            assert total == float(sum(g[2] for g in gathered)) and total > 0
            # the slices are disjoint and cover the seeded track list in order
            union = [t for g in gathered for t in g[3]]
            assert union == np.asarray(all_tracks).tolist()
            np.save(os.path.join(out_dir, "pass.npy"), np.array([1]))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_shard_tracks_and_reduce(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert os.path.exists(tmp_path / "pass.npy")


def test_single_rank_reduction_is_the_identity():
    import bench
    red, total = bench.reduce_over_ranks([1.5, 2.5], 7, 1, "cpu")
    assert red == [1.5, 2.5] and total == 7.0
    assert bench.shard_tracks(5, 4, 2) == slice(10, 15)

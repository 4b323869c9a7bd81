"""-m "not gpu": the N > 1 path on CPU, world_size 2, gloo backend.

The path shards by frame with no exchange step, so what there is to
cover is the host logic around the replicas: the frame partition (binding.shard_frames), that the shards put
back together equal the unsharded result, and bench.py's max-over-ranks timing reduction.  The per-frame work
of a rank is done here by the fp64 oracle on the tiny config C1 (this is a test; the product path is CUDA only).
"""
import os
import socket
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
N_FRAMES = 5          # odd on purpose: ranks get 3 and 2 frames


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        import oracle
        from paper_2203_14906_b200 import binding, synth
        w = synth.make_config("C1", n_frames=N_FRAMES)
        lo, hi = binding.shard_frames(N_FRAMES, rank, world)
        mine = oracle.beamform(w.rf[lo:hi], w.geom, 3, nthreads=1)            # this rank's replica: its own frames only
        spans = [None] * world
        dist.all_gather_object(spans, (lo, hi))
        parts = [None] * world
        dist.all_gather_object(parts, mine)
        # no rank needs another rank's data to produce its frames: the gather above is the test's, not the path's
        t = bench.max_over_ranks([10.0 + rank, 5.0 - rank], world, torch.device("cpu"))
        if rank == 0:
            np.save(os.path.join(out_dir, "joined.npy"), np.concatenate(parts, axis=0))
            np.save(os.path.join(out_dir, "spans.npy"), np.array(spans))
            np.save(os.path.join(out_dir, "tmax.npy"), np.array(t))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_rank_frame_sharding_and_timing_reduction(tmp_path, orc):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    from paper_2203_14906_b200 import synth
    w = synth.make_config("C1", n_frames=N_FRAMES)
    whole = orc.beamform(w.rf, w.geom, 3, nthreads=1)
    joined = np.load(tmp_path / "joined.npy")
    spans = np.load(tmp_path / "spans.npy")
    assert spans.tolist() == [[0, 3], [3, 5]]
    assert joined.shape == whole.shape and np.array_equal(joined, whole)      # frames are independent: bitwise equal
    assert np.load(tmp_path / "tmax.npy").tolist() == [11.0, 5.0]             # max over ranks, per entry

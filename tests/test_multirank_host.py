"""Host-side logic of the multi-GPU (replicas-only) run, on CPU with the gloo backend, world_size 2:
the max-over-ranks reduction bench.py applies to device-measured times, the per-rank seed streams
(different micro-batches per rank, no data-path collective) and the whole-job aggregate."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    import bench
    from paper_2606_05484_b200 import inputs as I
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    # each rank "measured" different times; everybody must end with the element-wise maximum
    ms, e2e = bench.max_over_ranks([10.0 + rank, 7.0 - rank], world, "cpu")
    # per-rank inputs: same config, different seed streams
    cfg = I.CONFIGS["c0"].with_tokens(64)
    bi = I.make_boundary(cfg, bench.boundary_stream(0, rank))
    digest = float(np.asarray(bi.H.f64).sum())
    gathered = [None] * world
    dist.all_gather_object(gathered, digest)
    np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([ms, e2e] + gathered))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_rank_streams(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r0, r1 = np.load(tmp_path / "r0.npy"), np.load(tmp_path / "r1.npy")
    assert np.array_equal(r0, r1)                       # all ranks agree
    assert r0[0] == 11.0 and r0[1] == 7.0               # element-wise max over ranks
    assert r0[2] != r0[3]                               # ranks drew different micro-batches


def test_single_rank_is_identity_and_aggregate():
    import bench
    assert bench.max_over_ranks([3.5, 1.25], 1, "cpu") == [3.5, 1.25]
    # 2 ranks x 1000 tokens x 4 steps in 2 ms -> 4e6 tokens/s
    assert bench.job_tokens_per_second(1000, 2, 4, 2.0) == 4.0e6
    assert bench.boundary_stream(2, 0) == 2 and bench.boundary_stream(2, 3) != bench.boundary_stream(2, 0)

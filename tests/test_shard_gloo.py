"""N > 1 host logic on CPU (gloo, world_size 2): run-index sharding, max-over-ranks timing, final gather.
Runs are keyed by their global run index (O3), so per-run results do not depend on the partition; the GPU side
of that statement is tests/test_gpu_runs.py::test_run_partition_invariance."""
import os
import socket
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_28372_b200.shard import shard_runs, max_over_ranks, sum_over_ranks, gather_runs


def test_shard_runs_is_a_partition():
    for total in (0, 1, 7, 1000, 1001, 99999):
        for world in (1, 2, 3, 8):
            spans = [shard_runs(total, world, r) for r in range(world)]
            assert spans[0][0] == 0 and sum(n for _, n in spans) == total
            for (f0, n0), (f1, _) in zip(spans, spans[1:]):
                assert f0 + n0 == f1
            assert max(n for _, n in spans) - min(n for _, n in spans) <= 1


def _worker(rank, world, port, total):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        first, n = shard_runs(total, world, rank)
        # a stand-in for per-run results: a function of the GLOBAL run index only
        idx = torch.arange(first, first + n, dtype=torch.int64)
        local = torch.stack([idx, idx * idx % 1013], dim=1)
        assert max_over_ranks(10.0 + rank) == 10.0 + world - 1
        assert sum_over_ranks(n) == total                        # whole-job unit count = the sum of the ranks' counts
        allr = gather_runs(local, total)
        if rank == 0:
            want = torch.arange(total, dtype=torch.int64)
            assert torch.equal(allr[:, 0], want) and torch.equal(allr[:, 1], want * want % 1013)
        else:
            assert allr is None
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_shard_and_gather():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    mp.spawn(_worker, args=(2, port, 1001), nprocs=2, join=True)

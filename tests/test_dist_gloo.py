"""N > 1 path on CPU: world_size-2 gloo.  Ensembles shard by trajectory id with no data-path
collective; the sharded result must equal the single-process result row by row.
The per-rank simulation is stood in for by the oracle here (tests may call it; there is no GPU
in this container) -- what is under test is the sharding and gathering logic of
paper_2103_00405_b200.dist."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import torch.distributed as dist
    import oracle
    import rt_workloads as W
    from paper_2103_00405_b200.dist import ensemble_sharded
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    net, x0 = W.lotka_volterra()

    def run_local(first, count):
        if count == 0:
            return dict(x=np.zeros((0, 2), dtype=np.int64), t=np.zeros(0), firings=np.zeros(0, dtype=np.uint64),
                        stop=np.zeros(0, dtype=np.int32))
        return oracle.ensemble(net, x0, 2, first, count, 3000, 0.05)

    full = ensemble_sharded(run_local, 2, 10, 7, group=None)
    np.savez(os.path.join(out_dir, f"rank{rank}.npz"), **full)
    dist.destroy_process_group()


def test_shard_range_partitions_exactly():
    sys.path.insert(0, ROOT)
    from paper_2103_00405_b200.dist import shard_range
    for n in (0, 1, 7, 64, 1000):
        for world in (1, 2, 3, 8):
            blocks = [shard_range(n, r, world) for r in range(world)]
            assert blocks[0][0] == 0
            for (f0, c0), (f1, c1) in zip(blocks, blocks[1:]):
                assert f1 == f0 + c0
            assert sum(c for _, c in blocks) == n
            assert max(c for _, c in blocks) - min(c for _, c in blocks) <= 1


def test_world_size_2_gloo_equals_single_process(tmp_path):
    import torch.multiprocessing as mp
    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    sys.path.insert(0, ROOT)
    import oracle
    import rt_workloads as W
    net, x0 = W.lotka_volterra()
    ref = oracle.ensemble(net, x0, 2, 10, 7, 3000, 0.05)
    for rank in range(2):
        got = np.load(os.path.join(str(tmp_path), f"rank{rank}.npz"))
        np.testing.assert_array_equal(got["x"], ref["x"])
        np.testing.assert_array_equal(got["firings"], ref["firings"])
        np.testing.assert_array_equal(got["t"], ref["t"])

"""N > 1 host logic on CPU: world_size-2 gloo process groups (no GPU, no kernels).

Covers (a) paper_2105_08722_b200.sharded.combine_partials — the one collective of the primary-sharded path
(all-gather + sum in rank order, bit-identical on every rank), and (b) bench.py's multi-rank plumbing: per-rank
catalogues, max-over-ranks timing, the barrier.
"""
import os
import socket
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2105_08722_b200 import sharded
        import bench
        import workloads as W

        # (a) partial zeta vectors whose sum depends on the order of addition in the last bits
        rng = np.random.default_rng(100 + rank)
        part = torch.from_numpy(rng.standard_normal((69, 120)) * 10.0 ** rng.integers(-8, 8, (69, 120)))
        total = sharded.combine_partials(part)
        np.save(os.path.join(out_dir, f"part{rank}.npy"), part.numpy())
        np.save(os.path.join(out_dir, f"total{rank}.npy"), total.numpy())

        # (b) bench.py plumbing
        bench._DIST["on"] = True
        bench.barrier()
        slowest = bench.max_over_ranks(torch, 10.0 + 5.0 * rank, torch.device("cpu"))
        cfg = W.scaled(W.CONFIGS["c3"], box=200.0, n=500, grid=16)
        pos, w = bench.make_catalogue(cfg, rank)
        np.save(os.path.join(out_dir, f"pos{rank}.npy"), pos)
        with open(os.path.join(out_dir, f"max{rank}.txt"), "w") as f:
            f.write(repr(slowest))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_world_size_2_gloo(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    parts = [np.load(tmp_path / f"part{r}.npy") for r in range(world)]
    totals = [np.load(tmp_path / f"total{r}.npy") for r in range(world)]
    expect = parts[0].copy()
    for r in range(1, world):
        expect += parts[r]                                   # rank order
    for r in range(world):
        assert totals[r].tobytes() == expect.tobytes()       # bit-identical on every rank
    # timing is the max over ranks on every rank; catalogues differ per rank and are reproducible
    assert [float(open(tmp_path / f"max{r}.txt").read()) for r in range(world)] == [15.0, 15.0]
    p0, p1 = np.load(tmp_path / "pos0.npy"), np.load(tmp_path / "pos1.npy")
    assert p0.shape == p1.shape and not np.array_equal(p0, p1)
    import bench
    import workloads as W
    again, _ = bench.make_catalogue(W.scaled(W.CONFIGS["c3"], box=200.0, n=500, grid=16), 1)
    assert np.array_equal(again, p1)


def test_combine_partials_without_a_process_group():
    from paper_2105_08722_b200 import sharded
    t = torch.arange(6, dtype=torch.float64).reshape(2, 3)
    out = sharded.combine_partials(t)
    assert torch.equal(out, t) and out.data_ptr() != t.data_ptr()

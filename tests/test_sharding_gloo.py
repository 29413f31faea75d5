"""N>1 path on CPU: world_size-2 gloo processes run bench.py's own rank function for the sharded
64-slice batch (bench.sharded_batch: slice partition, local run, max-over-ranks timing, final gather;
DESIGN.md section 8) with a CPU stand-in for the library call.  No GPU, no oracle."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1009_1351_b200.sharding import gather_slices, max_over_ranks, slice_range


def test_slice_range_is_a_balanced_contiguous_partition():
    for S in [0, 1, 2, 3, 7, 64, 65]:
        for world in [1, 2, 3, 4, 8]:
            parts = [slice_range(S, world, r) for r in range(world)]
            assert [i for p in parts for i in p] == list(range(S))
            sizes = [len(p) for p in parts]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        slice_range(4, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, S, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench                                    # the shipped N>1 path, not a copy of it

        def run_local(mine):
            # stand-in for tnlm_reconstruct on this rank's slices: slice s -> tensor filled with s, "took" 10+rank s
            local = torch.stack([torch.full((2, 3), float(s)) for s in mine]) if len(mine) else torch.zeros(0, 2, 3)
            return local, 10.0 + rank

        full, t, mine = bench.sharded_batch(S, world, rank, dist, run_local, "cpu")
        q.put((rank, list(mine), full[:, 0, 0].tolist(), t))
    finally:
        dist.destroy_process_group()


def test_sharded_batch_without_a_process_group_is_the_single_gpu_path():
    import bench
    full, t, mine = bench.sharded_batch(5, 1, 0, None, lambda mine: (torch.arange(len(mine)).float()[:, None], 2.5))
    assert list(mine) == [0, 1, 2, 3, 4] and t == 2.5 and full[:, 0].tolist() == [0.0, 1.0, 2.0, 3.0, 4.0]


def test_bench_refuses_more_gpus_than_the_node_has(monkeypatch):
    # `python bench.py --gpus N` must start N ranks or fail loudly, never run one rank and call it N
    import bench
    n = torch.cuda.device_count() + 1
    if n < 2:
        n = 2
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    monkeypatch.setattr("sys.argv", ["bench.py", "--gpus", str(n), "--steps", "1"])
    with pytest.raises(SystemExit) as ei:
        bench.main()
    assert "CUDA devices" in str(ei.value)
    monkeypatch.setenv("WORLD_SIZE", "1")
    with pytest.raises(SystemExit) as ei:
        bench.main()
    assert "WORLD_SIZE" in str(ei.value)


@pytest.mark.parametrize("S", [5, 64])
def test_world_size_two_gloo(S):
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, S, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] + res[1][1] == list(range(S))
    for _, _, gathered, t in res:
        assert gathered == [float(s) for s in range(S)]
        assert t == 11.0

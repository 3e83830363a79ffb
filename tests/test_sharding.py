"""Multi-GPU path of bench.py on CPU: world_size-2 `gloo` processes (the path shards by view).
Checks that the ranks of one job render disjoint views that together cover the steps, and that the reported time
is the max over ranks."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _fake_view_gradient(vi, tot):
    import torch
    g = torch.Generator().manual_seed(1000 + vi)
    return torch.randn(tot, generator=g, dtype=torch.float64)


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        steps, warm, n_views = 6, 3, 20
        warm_views = bench.views_for_rank(rank, world, n_views, warm)
        step_views = bench.views_for_rank(rank + warm * world, world, n_views, steps)
        gathered = [None] * world
        dist.all_gather_object(gathered, (warm_views, step_views))
        ms = bench.max_over_ranks(torch, dist, world, 10.0 + 5.0 * rank, "cpu")
        # the one collective of the data-parallel path: every rank fills the packed gradient buffer with the (fake)
        # gradients of ITS views; after the all-reduce every rank holds the sum over all views of all ranks
        n = 37                                              # not a multiple of 4: the group offsets are padded
        off, tot = bench.packed_offsets(n)
        flat = torch.zeros(tot, dtype=torch.float64)
        for vi in step_views:
            flat += _fake_view_gradient(vi, tot)
        bench.allreduce_sum(dist, flat)
        if rank == 0:
            out.put((gathered, ms, flat.numpy().copy(), off, tot))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_views_shard_over_two_ranks_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    gathered, ms, flat, off, tot = q.get(timeout=100)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    (w0, s0), (w1, s1) = gathered
    assert ms == 15.0                                 # max over ranks, not rank 0's own 10.0
    assert len(s0) == len(s1) == 6 and len(w0) == len(w1) == 3
    for a, b in zip(s0, s1):                          # same step: different views on the two ranks
        assert a != b
    assert set(s0).isdisjoint(s1) and set(w0).isdisjoint(w1)
    assert sorted(w0 + w1 + s0 + s1) == list(range(18))   # consecutive views, no gap, no overlap
    # all-reduced buffer = sum over ALL timed views of the single-rank gradients
    import numpy as np
    want = sum(_fake_view_gradient(vi, tot) for vi in s0 + s1).numpy()
    np.testing.assert_allclose(flat, want, rtol=1e-12, atol=1e-12)
    assert off == [0, 112, 260, 336, 376] and tot == 488 and all(o % 4 == 0 for o in off)   # 16-byte aligned groups, N = 37


def test_views_for_rank_single_process_cycles():
    import bench
    assert bench.views_for_rank(0, 1, 20, 23) == [i % 20 for i in range(23)]
    assert bench.views_for_rank(3, 8, 20, 3) == [3, 11, 19]


def _ref_worker(rank, out):
    import contextlib
    import io
    import json
    import bench
    os.environ.update(RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank))
    buf = io.StringIO()
    with contextlib.redirect_stdout(buf):
        sys.argv = ["bench.py", "--impl", "reference", "--config", "0", "--steps", "1", "--warmup", "0", "--gpus", "2"]
        bench.main()
    txt = buf.getvalue().strip()
    out.put((rank, json.loads(txt) if txt else None))


@pytest.mark.timeout(300)
def test_reference_arm_runs_on_rank0_only():
    """`bench.py --impl reference` under a 2-rank launch: rank 0 times the oracle and prints the JSON line, the other rank
    exits without work or output (tier contract for the reference arm)."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_ref_worker, args=(r, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=250) for _ in range(2))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert got[1] is None
    line = got[0]
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "Mpixel/s"


def test_gpus_flag_spawns_one_process_per_gpu(monkeypatch):
    """`python bench.py --gpus 2` without WORLD_SIZE launches two ranks itself (torch.distributed.run on 127.0.0.1) and
    hands over; under torchrun (WORLD_SIZE set) it does not spawn again."""
    import bench
    calls = []
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    monkeypatch.setattr(bench.subprocess, "call", lambda cmd: calls.append(cmd) or 0)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "2", "--steps", "4", "--warmup", "3"])
    with pytest.raises(SystemExit) as e:
        bench.main()
    assert e.value.code == 0 and len(calls) == 1
    cmd = calls[0]
    assert "torch.distributed.run" in cmd and "--nproc-per-node=2" in cmd and "127.0.0.1" in cmd
    assert cmd[-6:] == ["--gpus", "2", "--steps", "4", "--warmup", "3"] and cmd[-7].endswith("bench.py")
    # under a launcher: no second spawn (run_ours is reached; stub it out)
    monkeypatch.setenv("WORLD_SIZE", "2")
    reached = []
    monkeypatch.setattr(bench, "run_ours", lambda a: reached.append(a.gpus))
    bench.main()
    assert reached == [2] and len(calls) == 1

"""Host-side logic of bench.py's N > 1 path ("replicas only"): world_size-2 gloo run on CPU.
Every rank advances its own replica; the whole-job value is world * steps / max-over-ranks time."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = [120.0, 200.0][rank]  # rank 1 is the slow replica
    mx = bench.max_over_ranks(ms, world, device="cpu")
    dist.barrier()
    out.put((rank, mx, bench.whole_job_value(world, 4, mx), bench.replica_seed(rank)))
    dist.destroy_process_group()


def test_two_replicas_gloo_max_over_ranks():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [200.0, 200.0]                     # both ranks see the slowest time
    assert res[0][2] == pytest.approx(2 * 4 / 0.2)                   # whole-job steps/s over both replicas
    assert [r[3] for r in res] == [0, 1]                             # distinct replica seeds


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(12.5, 1) == 12.5
    assert bench.whole_job_value(1, 5, 1000.0) == pytest.approx(5.0)


def test_reference_arm_exits_quietly_on_nonzero_rank(monkeypatch, capsys):
    sys.path.insert(0, ROOT)
    import bench

    class A:
        config, steps, warmup, gpus = 3, 1, 0, 2
    monkeypatch.setenv("RANK", "1")
    assert bench.run_reference(A) == 0
    assert capsys.readouterr().out == ""

"""N > 1 path of bench.py ("replicas only") on CPU: world_size 2 over gloo.
Checks the whole-job aggregation (time = max over ranks, work = sum over ranks) and that the reference
arm does its work on rank 0 only."""
import os
import socket
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench

    # rank r took (100 + 50 r) ms for 2e12 flops of its own independent expansion
    ms_max, rate = bench.whole_job_rate(100.0 + 50.0 * rank, 2.0e12, "cpu")
    out[rank] = (ms_max, rate)
    dist.barrier()
    dist.destroy_process_group()


def test_whole_job_rate_world2():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    ms_max, rate = res[0]
    assert ms_max == 150.0
    assert rate == pytest.approx(4.0e12 / 0.150 / 1e12)


def test_whole_job_rate_single_process():
    sys.path.insert(0, ROOT)
    import bench

    ms, rate = bench.whole_job_rate(200.0, 1.0e12)
    assert ms == 200.0 and rate == pytest.approx(5.0)


def test_reference_arm_runs_on_rank0_only(monkeypatch, capsys):
    sys.path.insert(0, ROOT)
    import bench

    class A:
        config, cpu_k, steps, warmup, gpus = 1, 64, 1, 0, 2

    monkeypatch.setenv("RANK", "1")
    assert bench.run_reference(A) == 0
    assert capsys.readouterr().out == ""
    monkeypatch.setenv("RANK", "0")
    assert bench.run_reference(A) == 0
    line = capsys.readouterr().out
    assert '"impl": "reference"' in line and '"kind": "oracle"' in line

"""N > 1 path (replicas only, no data-path collective): what bench.py does across ranks is a
barrier, a MAX over ranks of the device time and the whole-job aggregation.  Covered here with two gloo processes
on CPU (no GPU): the job's time is the slowest replica's and `value` counts the samples of every rank."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms_local = 2.0 + 3.0 * rank                      # rank 1 is the slow replica: 5 ms per step
        dist.barrier()
        ms = bench.max_over_ranks(ms_local, dist, device="cpu")
        value = bench.job_throughput(4, world, ms * 1e-3)
        torch.save({"ms": ms, "value": value}, os.path.join(out, f"r{rank}.pt"))
    finally:
        dist.destroy_process_group()


def test_two_replicas_max_time_and_aggregate(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    res = [torch.load(os.path.join(tmp_path, f"r{r}.pt")) for r in range(world)]
    for r in res:                                         # every rank sees the slowest replica's time
        assert r["ms"] == 5.0
        assert abs(r["value"] - 2 * 4 / 5e-3) < 1e-9      # 2 replicas x 4 samples per 5 ms step


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(1.25, None) == 1.25
    assert bench.job_throughput(4, 1, 1e-3) == 4000.0


def test_reference_arm_runs_on_rank0_only(monkeypatch, capsys):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")

    class A:
        config, steps, warmup, gpus = 2, 1, 0, 2
    bench.run_reference(A)                                # rank != 0: returns without work or output
    assert capsys.readouterr().out == ""

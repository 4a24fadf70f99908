"""not gpu: the N > 1 host logic of bench.py (replicas only: max-over-ranks time, summed throughput),
world_size 2 over gloo on CPU, rendezvous on 127.0.0.1."""
import os
import socket
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 + 5.0 * rank            # rank 1 is the slow replica
    ms_max = bench.reduce_max_ms(ms_local, world, "cpu")
    val = bench.aggregate_value(1000, 4, ms_max, world)
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, ms_max, val))


def test_two_rank_reduction_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = [q.get(timeout=120) for _ in ps]
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms_max, val in res:
        assert ms_max == 15.0
        assert abs(val - 2 * 1000 * 4 / 15e-3) < 1e-6


def test_reference_arm_other_ranks_exit_quietly(monkeypatch, capsys):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")
    class A: workload = "5a"; steps = 1; warmup = 0; gpus = 2
    bench.run_reference(A())
    assert capsys.readouterr().out == ""

"""The N > 1 path of bench.py (replicas, weak scaling) on CPU: two gloo ranks run the timing
protocol (barrier, max over ranks, whole-job aggregate).  The data path has no collective
(DESIGN.md "Multi-GPU"), so this is all there is to test without GPUs."""
import os
import socket
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import bench
    r = bench.Ranks("gloo")
    r.barrier()
    ms = r.max(10.0 + 5.0 * rank)            # rank 1 is the slow one
    r.barrier()
    q.put((rank, ms, bench.whole_job_glups(1000, 20, ms, r.world)))
    r.close()


def test_two_gloo_ranks_take_the_max_and_aggregate():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [15.0, 15.0]
    want = 2 * 1000 * 20 / 15e-3 / 1e9
    assert all(abs(r[2] - want) < 1e-12 for r in res)


def test_reference_arm_is_silent_on_other_ranks(monkeypatch, capsys):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")
    bench.run_reference(type("A", (), {"size": 256, "steps": 1, "warmup": 0, "gpus": 2})())
    assert capsys.readouterr().out == ""

"""Host-side logic of the z-slab decomposition (paper_2501_00846_b200/slab.py) without a GPU: the
slab ranges and periodic cuts, and the ring exchange over torch.distributed with two gloo ranks
(fake slabs whose faces carry their rank and face number)."""
import os
import socket
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_slab_ranges_and_cuts():
    from paper_2501_00846_b200 import slab as S
    assert [S.slab_range(48, r, 4) for r in range(4)] == [(0, 12), (12, 24), (24, 36), (36, 48)]
    with pytest.raises(ValueError):
        S.slab_range(50, 0, 4)
    a = np.arange(6 * 2 * 3).reshape(6, 2, 3)
    c = S.cut(a, 0, 3, 6)                                        # planes -2 .. 4 wrapped
    assert [int(p[0, 0]) // 6 for p in c] == [4, 5, 0, 1, 2, 3, 4]
    v = np.stack([a, a + 100, a + 200])                          # vectors: leading axis untouched
    assert S.cut(v, 3, 6, 6).shape == (3, 7, 2, 3)


class _FakeSolver:
    def synchronize(self):
        pass


class _FakeSlab:
    """Stands in for SlabSolver in DistExchange: faces tagged (rank, face)."""

    def __init__(self, rank):
        import torch
        self.torch, self.solver, self.rank = torch, _FakeSolver(), rank
        self.send = [torch.full((5,), 10.0 * rank + f) for f in (0, 1)]
        self.recv = [torch.zeros(5), torch.zeros(5)]
        self.got = None

    def pack(self):
        pass

    def unpack(self, from_low, from_high):
        self.got = (None if from_low is None else float(from_low[0]),
                    None if from_high is None else float(from_high[0]))


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_2501_00846_b200 import slab as S
    dist.init_process_group("gloo")
    s = _FakeSlab(rank)
    s.periodic = os.environ.get("SLAB_TEST_WALLS") != "1"
    S.DistExchange(s, rank, world, dist)()
    q.put((rank, s.got))
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_ring_exchange_over_gloo(world):
    """Rank r's low ghosts must come from rank r-1's HIGH face and its high ghosts from rank
    r+1's LOW face (periodic ring)."""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        lo, hi = (r - 1) % world, (r + 1) % world
        assert res[r] == (10.0 * lo + 1, 10.0 * hi + 0), (r, res[r])


@pytest.mark.parametrize("world", [2, 3])
def test_chain_exchange_with_walls_over_gloo(world, monkeypatch):
    """Walls on z: no wrap between the last and the first rank; the end slabs get nothing from
    beyond the wall."""
    monkeypatch.setenv("SLAB_TEST_WALLS", "1")
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        want = (None if r == 0 else 10.0 * (r - 1) + 1, None if r == world - 1 else 10.0 * (r + 1))
        assert res[r] == want, (r, res[r])


def test_single_rank_exchange_wraps_onto_itself():
    sys.path.insert(0, ROOT)
    from paper_2501_00846_b200 import slab as S
    s = _FakeSlab(0)
    S.DistExchange(s, 0, 1, None)()
    assert s.got == (1.0, 0.0)


# ------------------------------------------------- the overlapped schedule of SlabSolver.step
class _StepSolver(_FakeSolver):
    """Records the order of the calls SlabSolver.step makes; the 'faces' are a step counter."""

    def __init__(self, log):
        self.log = log

    def slab_step_faces(self):
        self.log.append("faces")

    def slab_step_interior(self):
        self.log.append("interior")

    def step(self, n):
        self.log.append("whole")


def _step_worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    from paper_2501_00846_b200 import slab as S
    dist.init_process_group("gloo")
    log = []
    sl = S.SlabSolver.__new__(S.SlabSolver)              # the schedule only: no CUDA Solver
    sl.solver, sl.torch, sl.rank, sl.world, sl.can_split = _StepSolver(log), torch, rank, world, True
    sl.send = [torch.zeros(3), torch.zeros(3)]
    sl.recv = [torch.zeros(3), torch.zeros(3)]
    sl.steps_packed, sl.seen = 0, []

    def pack():
        log.append("pack")
        sl.steps_packed += 1
        for f in (0, 1):
            sl.send[f][:] = 100.0 * sl.steps_packed + 10.0 * rank + f

    def unpack(lo, hi):
        log.append("unpack")
        sl.seen.append((float(lo[0]), float(hi[0])))
    sl.pack, sl.unpack = pack, unpack
    sl.exchange = S.DistExchange(sl, rank, world, dist)
    sl.step(2, overlap=True)
    sl.step(1, overlap=False)
    q.put((rank, log, sl.seen))
    dist.destroy_process_group()


def test_overlapped_step_schedule_over_gloo():
    """faces -> pack -> (transfers posted) -> interior -> wait + unpack, every step; each step's
    ghosts come from the SAME step's faces of the right neighbours; overlap=False falls back to
    whole step + exchange."""
    world = 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_step_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = {r: (log, seen) for r, log, seen in (q.get(timeout=180) for _ in procs)}
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r in range(world):
        log, seen = res[r]
        assert log == ["faces", "pack", "interior", "unpack"] * 2 + ["whole", "pack", "unpack"]
        lo, hi = (r - 1) % world, (r + 1) % world
        assert seen == [(100.0 * k + 10.0 * lo + 1, 100.0 * k + 10.0 * hi + 0) for k in (1, 2, 3)]

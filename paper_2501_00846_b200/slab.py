"""z-slab decomposition of a lattice along z (the paper's own multi-GPU
runs use Cartesian decompositions over MPI, "a linear decomposition along the z-axis" among them,
PAPER.md:194-238).

Orchestration only: every step of the path still runs in the kernels of libtslb.so.  Rank r of W
owns nz / W consecutive planes and holds a Solver on them plus two ghost planes per end that has a
neighbour (include/tslb.h "z-slab decomposition support"): a ring when z is periodic; with walls
on z (rising bubble, droplet train) the first and last slab end at the wall.  Per time step: the
step on every slab (in two stages, the face planes first, so that the exchange overlaps the
interior sweep: tslb_slab_step_faces / tslb_slab_step_interior; or tslb_step(1) as a whole), and
ONE exchange: each slab packs the two owned planes next to each face (tslb_halo_pack, 17 scalars
per node), sends the low face to rank r-1 and the high face to rank r+1, and unpacks what it
receives into its ghost planes.  The results on the owned planes are the single-domain results
bit for bit (the kernels' per-node arithmetic does not depend on where a plane sits), which
tests/test_slab_gpu.py checks with several slabs on ONE GPU.

Transport is pluggable: `LocalExchange` hands buffers over inside one process (the test, or slabs
on the GPUs of one process); `DistExchange` uses torch.distributed point-to-point operations (NCCL
between GPUs: batch_isend_irecv).  NOT MEASURED on more than one GPU: this build's runs have one
(DESIGN.md 8); BASELINE.json's north star asks for replicas only, which stays bench.py's default.
"""
import numpy as np

from . import binding as B

GHOST = 2


def slab_range(nz, rank, world):
    """Owned planes [z0, z1) of rank `rank`: nz must divide evenly."""
    if nz % world != 0 or nz // world < 2:
        raise ValueError(f"nz = {nz} must be a multiple of the {world} slabs, >= 2 planes each")
    n = nz // world
    return rank * n, (rank + 1) * n


def cut(a, z0, z1, nz, ghost=(True, True)):
    """Planes [z0 - GHOST, z1 + GHOST) of a (..., nz, ny, nx) array, wrapped periodically; an end
    without ghost planes (a wall of the box: ghost[end] False) is cut at the owned plane."""
    idx = np.arange(z0 - (GHOST if ghost[0] else 0), z1 + (GHOST if ghost[1] else 0)) % nz
    return np.ascontiguousarray(np.take(a, idx, axis=-3))


def neighbours(rank, world, periodic):
    """(low, high) neighbour ranks of a slab; None beyond a wall of the box."""
    if periodic:
        return (rank - 1) % world, (rank + 1) % world
    return (rank - 1 if rank > 0 else None), (rank + 1 if rank < world - 1 else None)


class LocalExchange:
    """All slabs live in this process: hand the packed faces over directly."""

    def __init__(self, slabs):
        self.slabs = slabs

    def deliver(self):
        """Unpack every slab's ghosts from its neighbours' packed faces."""
        W = len(self.slabs)
        for r, s in enumerate(self.slabs):
            lo, hi = neighbours(r, W, getattr(s, "periodic", True))
            # my low ghosts = the low neighbour's high face; my high ghosts = the high
            # neighbour's low face (buffers of another slab are only read here)
            s.unpack(None if lo is None else self.slabs[lo].send[1],
                     None if hi is None else self.slabs[hi].send[0])

    def __call__(self):
        for s in self.slabs:
            s.pack()
        self.deliver()


class DistExchange:
    """One slab per rank: ring exchange over torch.distributed (send low face down, high face up).

    start() posts the transfers of the faces packed so far and returns at once; finish() waits
    for them and unpacks.  Between the two the caller launches the interior of the step
    (SlabSolver.step), which is what hides the transfer.  exchange() = pack + start + finish."""

    def __init__(self, slab, rank, world, dist):
        self.slab, self.rank, self.world, self.dist = slab, rank, world, dist

    def _streams(self):
        s = self.slab
        if not s.send[0].is_cuda:
            return None, None
        return s.torch.cuda.current_stream(s.send[0].device), s.solver.stream

    def start(self):
        s, dist = self.slab, self.dist
        if self.world == 1:
            return None
        cur, own = self._streams()
        if cur is None:
            s.solver.synchronize()                  # host buffers: the packed faces are complete
        elif cur != own:
            cur.wait_stream(own)                    # NCCL orders its work after the CURRENT stream
        lo, hi = neighbours(self.rank, self.world, getattr(s, "periodic", True))
        # With two ranks on a ring both neighbours are the same peer and NCCL matches messages of
        # a pair in posting order (no tags): the HIGH face is sent first because the peer receives
        # its low ghosts (= its low neighbour's high face) first.  Beyond a wall of the box there
        # is no neighbour and nothing is posted.
        sends = ([dist.P2POp(dist.isend, s.send[1], hi, tag=0)] if hi is not None else []) + \
                ([dist.P2POp(dist.isend, s.send[0], lo, tag=1)] if lo is not None else [])
        recvs = ([dist.P2POp(dist.irecv, s.recv[0], lo, tag=0)] if lo is not None else []) + \
                ([dist.P2POp(dist.irecv, s.recv[1], hi, tag=1)] if hi is not None else [])
        return dist.batch_isend_irecv(sends + recvs)

    def finish(self, reqs):
        s = self.slab
        if reqs is None:                            # one rank: the slab is its own neighbour
            if getattr(s, "periodic", True):        # (a box with walls on z has none at all)
                s.unpack(s.send[1], s.send[0])
            return
        for req in reqs:
            req.wait()      # NCCL: the current stream waits for the transfer; gloo: the host does
        cur, own = self._streams()
        if cur is not None and cur != own:
            own.wait_stream(cur)
        lo, hi = neighbours(self.rank, self.world, getattr(s, "periodic", True))
        s.unpack(None if lo is None else s.recv[0], None if hi is None else s.recv[1])

    def __call__(self):
        self.slab.pack()
        self.finish(self.start())


class SlabSolver:
    """One z slab: a Solver on the owned planes plus two ghost planes per end that has a
    neighbour.  Periodic z: a ring, every slab has both.  Walls on z (the paper's rising bubble
    and droplet train): the first and the last slab end at the wall and carry ghosts at their inner
    end only (tslb_slab_set_ends)."""

    def __init__(self, nx, ny, nz, params, rank, world, precision="f64", device="cuda:0", flags=0):
        self.periodic = tuple(params.get("bc", (0, 0, 0)))[2] == 0
        self.nz_global, self.rank, self.world = nz, rank, world
        self.z0, self.z1 = slab_range(nz, rank, world)
        lo, hi = neighbours(rank, world, self.periodic)
        self.ghost = (lo is not None, hi is not None)
        nzl = self.z1 - self.z0 + GHOST * (int(self.ghost[0]) + int(self.ghost[1]))
        self.solver = B.Solver(nx, ny, nzl, params, precision=precision, flags=flags, device=device)
        if not self.periodic:
            self.solver.slab_set_ends(*self.ghost)
        self.torch = self.solver.torch
        self.send = [self.solver.halo_buffer(), self.solver.halo_buffer()]
        self.recv = [self.solver.halo_buffer(), self.solver.halo_buffer()]
        self.exchange = None                        # set by the owner (Local / Dist)
        # the split step needs whole 128-bit row vectors (include/tslb.h)
        self.can_split = nx % (2 if precision == "f64" else 4) == 0

    def init(self, phi, u):
        """phi (nz, ny, nx), u (3, nz, ny, nx): the GLOBAL host arrays; this slab takes its part.
        The owner must run one exchange afterwards (the outermost ghost plane's force and flux
        were computed with a wrapped stencil)."""
        self.solver.init(cut(np.asarray(phi), self.z0, self.z1, self.nz_global, self.ghost),
                         cut(np.asarray(u), self.z0, self.z1, self.nz_global, self.ghost))

    def pack(self):
        for face in (0, 1):
            if self.ghost[face]:
                self.solver.halo_pack(face, self.send[face])

    def unpack(self, from_low, from_high):
        if self.ghost[0] and from_low is not None:
            self.solver.halo_unpack(0, from_low)
        if self.ghost[1] and from_high is not None:
            self.solver.halo_unpack(1, from_high)

    def step(self, n=1, overlap=True):
        """n steps, each followed by its exchange.  With `overlap` (and rows the split step
        accepts) the face planes are computed and sent first and the interior is swept while they
        travel (tslb_slab_step_faces / _interior); the results are the same bit for bit."""
        split = overlap and self.can_split and hasattr(self.exchange, "start")
        for _ in range(int(n)):
            if split:
                self.solver.slab_step_faces()
                self.pack()
                pending = self.exchange.start()
                self.solver.slab_step_interior()
                self.exchange.finish(pending)
            else:
                self.solver.step(1)
                self.exchange()

    def get(self, want=("rho", "p", "u", "phi")):
        """The owned planes of tslb_get's fields."""
        g = self.solver.get(want)
        a = GHOST if self.ghost[0] else 0
        b = self.solver.nz - (GHOST if self.ghost[1] else 0)
        return {k: v[..., a:b, :, :] for k, v in g.items()}

    def close(self):
        self.solver.close()


def make_local_slabs(nx, ny, nz, params, world, precision="f64", device="cuda:0", flags=0):
    """`world` slabs in this process wired with a LocalExchange (tests, single-process use)."""
    slabs = [SlabSolver(nx, ny, nz, params, r, world, precision, device, flags) for r in range(world)]
    ex = LocalExchange(slabs)
    for s in slabs:
        s.exchange = lambda: None                   # stepping is driven for all slabs together
    return slabs, ex


def step_local(slabs, ex, n=1, overlap=True):
    """Step all slabs of this process together.  overlap: faces first, pack, interior, deliver
    (the schedule SlabSolver.step runs per rank); otherwise whole steps, then the exchange."""
    split = overlap and all(s.can_split for s in slabs)
    for _ in range(int(n)):
        if split:
            for s in slabs:
                s.solver.slab_step_faces()
                s.pack()
            for s in slabs:
                s.solver.slab_step_interior()
            ex.deliver()
        else:
            for s in slabs:
                s.solver.step(1)
            ex()

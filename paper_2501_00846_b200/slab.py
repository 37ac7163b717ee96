"""z-slab decomposition of a lattice that is periodic along z (the paper's
own multi-GPU runs use Cartesian decompositions over MPI).

Orchestration only: every step of the path still runs in the kernels of libtslb.so.  Rank r of W
owns nz / W consecutive planes and holds a Solver on nz / W + 4 planes (two ghost planes per end,
periodic z; include/tslb.h "z-slab decomposition support").  Per time step: the step on every
slab (in two stages, the face planes first, so that the exchange overlaps the interior sweep:
tslb_slab_step_faces / tslb_slab_step_interior; or tslb_step(1) as a whole), and ONE exchange: each slab packs the two owned planes next to each face
(tslb_halo_pack, 17 scalars per node), sends the low face to rank r-1 and the high face to rank r+1,
and unpacks what it receives into its ghost planes.  The results on the owned planes are the
single-domain results bit for bit (the kernels' per-node arithmetic does not depend on where a
plane sits), which tests/test_slab_gpu.py checks with several slabs on ONE GPU.

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


def cut(a, z0, z1, nz):
    """Planes [z0 - GHOST, z1 + GHOST) of a (..., nz, ny, nx) array, wrapped periodically."""
    idx = np.arange(z0 - GHOST, z1 + GHOST) % nz
    return np.ascontiguousarray(np.take(a, idx, axis=-3))


class LocalExchange:
    """All slabs live in this process: hand the packed faces over directly."""

    def __init__(self, slabs):
        self.slabs = slabs

    def deliver(self):
        """Unpack every slab's ghosts from its neighbours' packed faces."""
        W = len(self.slabs)
        for r, s in enumerate(self.slabs):
            lo, hi = self.slabs[(r - 1) % W], self.slabs[(r + 1) % W]
            # my low ghosts = the low neighbour's high face; my high ghosts = the high
            # neighbour's low face (buffers of another slab are only read here)
            s.unpack(lo.send[1], hi.send[0])

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
        lo, hi = (self.rank - 1) % self.world, (self.rank + 1) % self.world
        # With two ranks both neighbours are the same peer and NCCL matches messages of a pair
        # in posting order (no tags): the HIGH face is sent first because the peer receives its
        # low ghosts (= its low neighbour's high face) first.
        ops = [dist.P2POp(dist.isend, s.send[1], hi, tag=0), dist.P2POp(dist.isend, s.send[0], lo, tag=1),
               dist.P2POp(dist.irecv, s.recv[0], lo, tag=0), dist.P2POp(dist.irecv, s.recv[1], hi, tag=1)]
        return dist.batch_isend_irecv(ops)

    def finish(self, reqs):
        s = self.slab
        if reqs is None:                            # one rank: the slab is its own neighbour
            s.unpack(s.send[1], s.send[0])
            return
        for req in reqs:
            req.wait()      # NCCL: the current stream waits for the transfer; gloo: the host does
        cur, own = self._streams()
        if cur is not None and cur != own:
            own.wait_stream(cur)
        s.unpack(s.recv[0], s.recv[1])

    def __call__(self):
        self.slab.pack()
        self.finish(self.start())


class SlabSolver:
    """One z slab: a Solver on the owned planes plus two ghost planes per end."""

    def __init__(self, nx, ny, nz, params, rank, world, precision="f64", device="cuda:0", flags=0):
        if tuple(params.get("bc", (0, 0, 0)))[2] != 0:
            raise ValueError("the slab decomposition needs a periodic z axis")
        self.nz_global, self.rank, self.world = nz, rank, world
        self.z0, self.z1 = slab_range(nz, rank, world)
        self.solver = B.Solver(nx, ny, self.z1 - self.z0 + 2 * GHOST, params, precision=precision,
                               flags=flags, device=device)
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
        self.solver.init(cut(np.asarray(phi), self.z0, self.z1, self.nz_global),
                         cut(np.asarray(u), self.z0, self.z1, self.nz_global))

    def pack(self):
        self.solver.halo_pack(0, self.send[0])
        self.solver.halo_pack(1, self.send[1])

    def unpack(self, from_low, from_high):
        self.solver.halo_unpack(0, from_low)
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
        return {k: v[..., GHOST:-GHOST, :, :] for k, v in g.items()}

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

"""z-slab decomposition of a lattice that is periodic along z (the paper's
own multi-GPU runs use Cartesian decompositions over MPI).

Orchestration only: every step of the path still runs in the kernels of libtslb.so.  Rank r of W
owns nz / W consecutive planes and holds a Solver on nz / W + 4 planes (two ghost planes per end,
periodic z; include/tslb.h "z-slab decomposition support").  Per time step: tslb_step(1) on every
slab, then ONE exchange: each slab packs the two owned planes next to each face
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

    def __call__(self):
        W = len(self.slabs)
        for s in self.slabs:
            s.pack()
        for r, s in enumerate(self.slabs):
            lo, hi = self.slabs[(r - 1) % W], self.slabs[(r + 1) % W]
            # my low ghosts = the low neighbour's high face; my high ghosts = the high
            # neighbour's low face (buffers of another slab are only read here)
            s.unpack(lo.send[1], hi.send[0])


class DistExchange:
    """One slab per rank: ring exchange over torch.distributed (send low face down, high face up)."""

    def __init__(self, slab, rank, world, dist):
        self.slab, self.rank, self.world, self.dist = slab, rank, world, dist

    def __call__(self):
        s, dist = self.slab, self.dist
        s.pack()
        if self.world == 1:
            s.unpack(s.send[1], s.send[0])
            return
        s.solver.synchronize()                      # the packed faces are complete
        lo, hi = (self.rank - 1) % self.world, (self.rank + 1) % self.world
        # With two ranks both neighbours are the same peer and NCCL matches messages of a pair
        # in posting order (no tags): the HIGH face is sent first because the peer receives its
        # low ghosts (= its low neighbour's high face) first.
        ops = [dist.P2POp(dist.isend, s.send[1], hi, tag=0), dist.P2POp(dist.isend, s.send[0], lo, tag=1),
               dist.P2POp(dist.irecv, s.recv[0], lo, tag=0), dist.P2POp(dist.irecv, s.recv[1], hi, tag=1)]
        for req in dist.batch_isend_irecv(ops):
            req.wait()
        if s.recv[0].is_cuda:
            s.torch.cuda.current_stream(s.recv[0].device).synchronize()
        s.unpack(s.recv[0], s.recv[1])


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

    def step(self, n=1):
        for _ in range(int(n)):
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


def step_local(slabs, ex, n=1):
    for _ in range(int(n)):
        for s in slabs:
            s.solver.step(1)
        ex()

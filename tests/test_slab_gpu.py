"""z-slab decomposition on ONE GPU: several slabs of a periodic lattice,
each a Solver on its planes plus two ghost planes per end, exchanging packed faces once per step
(tslb_halo_pack / tslb_halo_unpack through paper_2501_00846_b200/slab.py's LocalExchange), against
the single-domain Solver.  The per-node arithmetic does not depend on where a plane sits, so the
bar is EQUALITY of every owned plane, in both precisions; the single-domain path is the one the
oracle parity tests cover."""
import numpy as np
import pytest

from paper_2501_00846_b200 import inputs as I

pytestmark = pytest.mark.gpu


def _case():
    shape = (48, 21, 70)                                         # (nz, ny, nx): ragged tiles in x, y
    prm = I.base_params()
    phi = I.sphere_profile(shape, (30.3, 9.1, 11.7), 8.0, 4.0, prm["bc"])      # across a slab cut
    phi += I.sphere_profile(shape, (55.2, 14.6, 36.4), 6.0, 4.0, prm["bc"])
    return dict(name="slabs", shape=shape, params=prm, phi=phi, u=I.noise_u(shape, 1e-3, 53))


@pytest.mark.parametrize("world", [2, 4])
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_slabs_reproduce_the_single_domain(world, precision):
    from paper_2501_00846_b200 import binding as B, slab as S
    cfg = _case()
    nz, ny, nx = cfg["shape"]
    one = B.Solver(nx, ny, nz, cfg["params"], precision=precision)
    one.init(cfg["phi"], cfg["u"])
    slabs, ex = S.make_local_slabs(nx, ny, nz, cfg["params"], world, precision=precision)
    for s in slabs:
        s.init(cfg["phi"], cfg["u"])
    ex()                                                         # ghosts of the initial force / flux
    done = 0
    for n in (1, 5, 20):
        one.step(n - done)
        S.step_local(slabs, ex, n - done)
        done = n
        want = one.get()
        for s in slabs:
            got = s.get()
            for k, v in got.items():
                w = want[k][..., s.z0:s.z1, :, :]
                assert bool((v == w).all()), (world, precision, n, s.rank, k,
                                              float((v - w).abs().max()))
    assert slabs[0].solver.launches > 0
    for s in slabs:
        s.close()
    one.close()


def test_halo_calls_reject_what_they_cannot_serve():
    from paper_2501_00846_b200 import binding as B
    cfg, = [_case()]
    nz, ny, nx = cfg["shape"]
    walls = dict(cfg["params"], bc=(0, 0, 1))
    s = B.Solver(nx, ny, nz, walls)
    s.init(cfg["phi"], cfg["u"])
    buf = s.halo_buffer()
    with pytest.raises(B.TslbError):
        s.halo_pack(0, buf)                                      # z is not periodic
    s.close()
    s = B.Solver(nx, ny, nz, cfg["params"])
    buf = s.halo_buffer()
    with pytest.raises(B.TslbError):
        s.halo_pack(0, buf)                                      # before tslb_init
    s.init(cfg["phi"], cfg["u"])
    with pytest.raises(B.TslbError):
        s.halo_pack(2, buf)                                      # no such face
    s.close()

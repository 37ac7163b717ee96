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


def _case(nx=70):
    shape = (48, 21, nx)                                         # (nz, ny, nx): ragged tiles in x, y
    prm = I.base_params()
    phi = I.sphere_profile(shape, (30.3, 9.1, 11.7), 8.0, 4.0, prm["bc"])      # across a slab cut
    phi += I.sphere_profile(shape, (55.2, 14.6, 36.4), 6.0, 4.0, prm["bc"])
    return dict(name="slabs", shape=shape, params=prm, phi=phi, u=I.noise_u(shape, 1e-3, 53))


@pytest.mark.parametrize("overlap", [False, True])
@pytest.mark.parametrize("nx", [70, 64])
@pytest.mark.parametrize("world", [2, 4, 16])
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_slabs_reproduce_the_single_domain(world, precision, nx, overlap):
    """overlap: the step in two stages (tslb_slab_step_faces, pack, tslb_slab_step_interior,
    unpack), the schedule that hides the exchange behind the interior sweep; it never computes
    the ghost planes.  nx = 64 takes the TMA-staged stream-collide kernel in fp64, nx = 70 the
    cp.async one (and, in fp32, rows the split step refuses: slab.py falls back to whole steps).
    16 slabs of 3 planes: the two face pieces touch and there is no interior."""
    from paper_2501_00846_b200 import binding as B, slab as S
    cfg = _case(nx)
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
        S.step_local(slabs, ex, n - done, overlap=overlap)
        done = n
        want = one.get()
        for s in slabs:
            got = s.get()
            for k, v in got.items():
                w = want[k][..., s.z0:s.z1, :, :]
                assert bool((v == w).all()), (world, precision, nx, overlap, n, s.rank, k,
                                              float((v - w).abs().max()))
    assert slabs[0].solver.launches > 0
    for s in slabs:
        s.close()
    one.close()


def _wall_case(nx=64, bc=(0, 0, 1)):
    """Droplets falling onto the bottom wall and a bubble under the lid (walls on z, gravity on the
    liquid): the paper's tall multi-GPU cases in miniature, interfaces across the slab cuts."""
    shape = (48, 21, nx)
    prm = I.base_params(rho_g=1.0 / 800.0, mu_l=1.0 / 300.0, mu_g=1.0 / 15000.0, sigma=8e-4,
                        bc=bc, body_accel=(1e-6, 0.0, -2e-5), body_heavy=True)
    phi = I.sphere_profile(shape, (20.3, 9.1, 3.2), 6.0, 4.0, prm["bc"])        # on the bottom wall
    phi += I.sphere_profile(shape, (45.2, 14.6, 24.4), 7.0, 4.0, prm["bc"])     # across the middle cut
    phi += I.sphere_profile(shape, (10.7, 4.6, 44.9), 5.0, 4.0, prm["bc"])      # under the lid
    u = I.noise_u(shape, 1e-3, 57)
    u[2] -= 0.03 * phi
    return dict(name="wall_slabs", shape=shape, params=prm, phi=np.minimum(phi, 1.0), u=u)


@pytest.mark.parametrize("overlap", [False, True])
@pytest.mark.parametrize("nx", [70, 64])
@pytest.mark.parametrize("world", [1, 2, 4, 12])
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_slabs_with_walls_on_z_reproduce_the_single_domain(world, precision, nx, overlap):
    """Walls on z: the end slabs carry ghosts at their inner end only (tslb_slab_set_ends) and
    apply the wall rules (bounce-back, mirrored phi, ghost flux) at the other; world = 1 is the
    undivided box stepped through the two-stage calls."""
    from paper_2501_00846_b200 import binding as B, slab as S
    cfg = _wall_case(nx)
    nz, ny, nx = cfg["shape"]
    one = B.Solver(nx, ny, nz, cfg["params"], precision=precision)
    one.init(cfg["phi"], cfg["u"])
    slabs, ex = S.make_local_slabs(nx, ny, nz, cfg["params"], world, precision=precision)
    assert [s.ghost for s in slabs][0][0] is False and [s.ghost for s in slabs][-1][1] is False
    for s in slabs:
        s.init(cfg["phi"], cfg["u"])
    if world > 1 and nx % (2 if precision == "f64" else 4) != 0:
        with pytest.raises(B.TslbError):        # radius-2 interface kernel: refused, not wrong
            ex()
        return
    ex()
    done = 0
    for n in (1, 5, 20):
        one.step(n - done)
        S.step_local(slabs, ex, n - done, overlap=overlap)
        done = n
        want = one.get()
        for s in slabs:
            got = s.get()
            for k, v in got.items():
                w = want[k][..., s.z0:s.z1, :, :]
                assert v.shape == w.shape
                assert bool((v == w).all()), (world, precision, nx, overlap, n, s.rank, k,
                                              float((v - w).abs().max()))
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
        s.halo_pack(0, buf)                                      # a wall end has no ghost planes
    s.slab_set_ends(0, 1)
    s.halo_pack(1, buf)                                          # ... the other end now has
    with pytest.raises(B.TslbError):
        s.halo_pack(0, buf)
    s.close()
    s = B.Solver(nx, ny, nz, cfg["params"])
    buf = s.halo_buffer()
    with pytest.raises(B.TslbError):
        s.halo_pack(0, buf)                                      # before tslb_init
    s.init(cfg["phi"], cfg["u"])
    with pytest.raises(B.TslbError):
        s.halo_pack(2, buf)                                      # no such face
    with pytest.raises(B.TslbError):
        s.slab_set_ends(0, 1)                                    # a periodic end cannot lose its ghosts
    s.close()


def test_split_step_state_machine():
    """Between tslb_slab_step_faces and tslb_slab_step_interior only the halo calls are served."""
    from paper_2501_00846_b200 import binding as B
    cfg = _case(64)
    nz, ny, nx = cfg["shape"]
    s = B.Solver(nx, ny, nz, cfg["params"])
    with pytest.raises(B.TslbError):
        s.slab_step_faces()                                      # before tslb_init
    s.init(cfg["phi"], cfg["u"])
    with pytest.raises(B.TslbError):
        s.slab_step_interior()                                   # no faces stage before it
    s.slab_step_faces()
    buf = s.halo_buffer()
    s.halo_pack(0, buf)
    s.halo_unpack(1, buf)
    for call in (lambda: s.step(1), lambda: s.get(), lambda: s.diag(), s.slab_step_faces):
        with pytest.raises(B.TslbError):
            call()
    s.slab_step_interior()
    s.step(1)
    s.close()
    odd = B.Solver(70, ny, nz, cfg["params"], precision="f32")  # 70 % 4 != 0
    c70 = _case(70)
    odd.init(c70["phi"], c70["u"])
    with pytest.raises(B.TslbError):
        odd.slab_step_faces()
    odd.close()


@pytest.mark.parametrize("overlap", [False, True])
@pytest.mark.parametrize("bc", [(1, 1, 0), (1, 0, 1), (1, 1, 1)])
@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_slabs_of_boxes_with_side_walls(bc, precision, overlap):
    """Walls on x / y (with z periodic or walled): the row kernel's ghost fluxes and the lean
    stream-collide kernel's bounce accounting are per plane, so two ghost planes still do."""
    from paper_2501_00846_b200 import binding as B, slab as S
    cfg = _wall_case(72, bc)
    nz, ny, nx = cfg["shape"]
    one = B.Solver(nx, ny, nz, cfg["params"], precision=precision)
    one.init(cfg["phi"], cfg["u"])
    slabs, ex = S.make_local_slabs(nx, ny, nz, cfg["params"], 4, precision=precision)
    for s in slabs:
        s.init(cfg["phi"], cfg["u"])
    ex()
    done = 0
    for n in (1, 12):
        one.step(n - done)
        S.step_local(slabs, ex, n - done, overlap=overlap)
        done = n
        want = one.get()
        for s in slabs:
            for k, v in s.get().items():
                w = want[k][..., s.z0:s.z1, :, :]
                assert bool((v == w).all()), (bc, precision, overlap, n, s.rank, k,
                                              float((v - w).abs().max()))
    for s in slabs:
        s.close()
    one.close()

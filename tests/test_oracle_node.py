"""Pins P1-P4 of the CPU oracle: lattice, single-node reconstruction, stencils.

Each check is something the paper or the mathematics fixes, not the oracle's own formula:
isotropy identities of D3Q27 (R1), the Hermite-moment identities that Eq. 9/10/14 must satisfy
(PAPER.md:98-126), a brute-force einsum Hermite sum on single nodes (BASELINE.json north_star),
exactness of Eq. 18 / repaired Eq. 19 on polynomials (R10).
"""
import itertools

import numpy as np
import pytest

CS2 = 1.0 / 3.0
SYM = [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]


def full(A6):
    T = np.zeros((3, 3))
    for k, (a, b) in enumerate(SYM):
        T[a, b] = T[b, a] = A6[k]
    return T


@pytest.fixture(scope="module")
def lat(ref):
    return ref.lattice()


# ---------------------------------------------------------------- P1 -------------------
def test_p1_lattice_isotropy(lat):
    c, w, opp = lat
    c = c.astype(float)
    d = np.eye(3)
    assert sorted(map(tuple, c.astype(int))) == sorted(itertools.product((-1, 0, 1), repeat=3))
    # standard D3Q27 weights 8/27, 2/27, 1/54, 1/216 by number of non-zero components
    for ci, wi in zip(c, w):
        assert wi == pytest.approx({0: 8 / 27, 1: 2 / 27, 2: 1 / 54, 3: 1 / 216}[int(abs(ci).sum())],
                                   rel=1e-15)
    assert np.all(c[opp] == -c)
    assert w.sum() == pytest.approx(1.0, abs=1e-15)
    assert np.abs(np.einsum("i,ia->a", w, c)).max() < 1e-16
    assert np.abs(np.einsum("i,ia,ib->ab", w, c, c) - CS2 * d).max() < 1e-16
    assert np.abs(np.einsum("i,ia,ib,ig->abg", w, c, c, c)).max() < 1e-16
    iso4 = CS2 ** 2 * (np.einsum("ab,gd->abgd", d, d) + np.einsum("ag,bd->abgd", d, d)
                       + np.einsum("ad,bg->abgd", d, d))
    assert np.abs(np.einsum("i,ia,ib,ig,id->abgd", w, c, c, c, c) - iso4).max() < 1e-16
    # norm of the third-order Hermite polynomial H3_xxy : sum_i w_i H3_xxy^2 = 2 cs^6 (.. /3 per perm)
    h3xxy = c[:, 0] * c[:, 0] * c[:, 1] - CS2 * c[:, 1]
    assert np.dot(w, h3xxy * h3xxy) == pytest.approx(2 * CS2 ** 3, rel=1e-14)
    # xxx-type third-order polynomials vanish identically on the lattice (third order is
    # the highest D3Q27 carries)
    assert np.abs(c[:, 0] ** 3 - 3 * CS2 * c[:, 0]).max() < 1e-16


# ---------------------------------------------------------------- P2 -------------------
@pytest.mark.parametrize("seed", range(5))
def test_p2_moments_of_reconstruction(ref, lat, seed):
    c, w, _ = lat
    c = c.astype(float)
    rng = np.random.default_rng(seed)
    ps = rng.normal(scale=0.01)
    u = rng.normal(scale=0.05, size=3)
    A = rng.normal(scale=1e-3, size=6)
    a = rng.normal(scale=1e-3, size=3)
    d = np.eye(3)
    fe, fn, S = ref.feq(ps, u), ref.fneq(u, A), ref.forcing(u, a)
    tol = 1e-16
    # equilibrium (Eq. 9): p*, u, p* cs^2 d + uu, and the third-order moment
    assert abs(fe.sum() - ps) < tol
    assert np.abs(fe @ c - u).max() < tol
    assert np.abs(np.einsum("i,ia,ib->ab", fe, c, c) - (ps * CS2 * d + np.outer(u, u))).max() < tol
    m3 = np.einsum("i,i->", fe, c[:, 0] * c[:, 0] * c[:, 1])
    assert abs(m3 - (CS2 * u[1] + u[0] * u[0] * u[1])) < tol
    # non-equilibrium (Eq. 10, R2): no mass, no momentum, second Hermite moment is A
    H2 = np.einsum("ia,ib->iab", c, c) - CS2 * d
    assert abs(fn.sum()) < tol
    assert np.abs(fn @ c).max() < tol
    assert np.abs(np.einsum("i,iab->ab", fn, H2) - full(A)).max() < tol
    # third Hermite moment of fneq is the recursive a3
    H3xxy = c[:, 0] * c[:, 0] * c[:, 1] - CS2 * c[:, 1]
    AT = full(A)
    assert abs(fn @ H3xxy - (2 * u[0] * AT[0, 1] + u[1] * AT[0, 0])) < tol
    H3xyz = c[:, 0] * c[:, 1] * c[:, 2]
    assert abs(fn @ H3xyz - (u[0] * AT[1, 2] + u[1] * AT[0, 2] + u[2] * AT[0, 1])) < tol
    # forcing (Eq. 14, R4/R5): sum S = 0, sum S c = a, sum S cc = ua + au
    assert abs(S.sum()) < tol
    assert np.abs(S @ c - a).max() < tol
    assert np.abs(np.einsum("i,ia,ib->ab", S, c, c) - (np.outer(u, a) + np.outer(a, u))).max() < tol


def test_p2_third_moments_of_feq(ref, lat):
    """sum feq c_a c_b c_g = cs^2 (u_a d_bg + u_b d_ag + u_g d_ab) + u_a u_b u_g for the seven
    third-order combinations D3Q27 carries (none of type aaa)."""
    c, _, _ = lat
    u = np.array([0.03, -0.02, 0.05])
    d = np.eye(3)
    fe = ref.feq(0.01, u)
    for (a, b, g) in [(0, 0, 1), (0, 1, 1), (0, 0, 2), (0, 2, 2), (1, 1, 2), (1, 2, 2), (0, 1, 2)]:
        m = fe @ (c[:, a] * c[:, b] * c[:, g])
        want = CS2 * (u[a] * d[b, g] + u[b] * d[a, g] + u[g] * d[a, b]) + u[a] * u[b] * u[g]
        assert m == pytest.approx(want, abs=1e-17)


# ---------------------------------------------------------------- P3 -------------------
@pytest.mark.parametrize("seed", range(5))
def test_p3_bruteforce_hermite_sum(ref, lat, seed):
    """The oracle's per-node functions equal an independent einsum over the Hermite tensors, and
    the closed form A = Pi - p* cs^2 d - uu + (ua + au)/2 (R6) equals the literal Eq. 13."""
    c, w, _ = lat
    c = c.astype(float)
    d = np.eye(3)
    rng = np.random.default_rng(100 + seed)
    ps = rng.normal(scale=0.01)
    u = rng.normal(scale=0.05, size=3)
    A = full(rng.normal(scale=1e-3, size=6))
    a = rng.normal(scale=1e-3, size=3)
    H2 = np.einsum("ia,ib->iab", c, c) - CS2 * d
    H3 = (np.einsum("ia,ib,ig->iabg", c, c, c)
          - CS2 * (np.einsum("ig,ab->iabg", c, d) + np.einsum("ia,bg->iabg", c, d)
                   + np.einsum("ib,ag->iabg", c, d)))
    fe = w * (ps + c @ u / CS2 + np.einsum("iab,a,b->i", H2, u, u) / (2 * CS2 ** 2)
              + np.einsum("iabg,a,b,g->i", H3, u, u, u) / (6 * CS2 ** 3))
    a3 = (np.einsum("a,bg->abg", u, A) + np.einsum("b,ag->abg", u, A) + np.einsum("g,ab->abg", u, A))
    fn = w * (np.einsum("iab,ab->i", H2, A) / (2 * CS2 ** 2)
              + np.einsum("iabg,abg->i", H3, a3) / (6 * CS2 ** 3))
    S = w * (((c - u) / CS2 + (c @ u)[:, None] * c / CS2 ** 2) @ a)
    A6 = [A[p] for p in SYM]
    assert np.abs(ref.feq(ps, u) - fe).max() < 1e-16
    assert np.abs(ref.fneq(u, A6) - fn).max() < 1e-17
    assert np.abs(ref.forcing(u, a) - S).max() < 1e-17
    # closed form of the pre-regularisation for an arbitrary population set
    f = fe + 0.3 * fn + 0.5 * S + w * rng.normal(scale=1e-4, size=27)
    pst = f.sum()
    m = f @ c
    Pi = np.einsum("i,ia,ib->ab", f, c, c)
    un = m + 0.5 * a
    lit = np.einsum("iab,i->ab", H2, f - (ref.feq(pst, un) - 0.5 * ref.forcing(un, a)))
    closed = Pi - pst * CS2 * d - np.outer(un, un) + 0.5 * (np.outer(un, a) + np.outer(a, un))
    assert np.abs(lit - closed).max() < 1e-16


# ---------------------------------------------------------------- P4 -------------------
def _coords(shape):
    nz, ny, nx = shape
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return x.astype(float), y.astype(float), z.astype(float)


def test_p4_stencils_on_polynomials(ref):
    """Away from the wrap, Eq. 18 is exact on linear (indeed quadratic) fields and the repaired
    Eq. 19 is exact on quadratics and zero on constants."""
    shape = (9, 10, 11)
    x, y, z = _coords(shape)
    lin = 0.3 + 1.5 * x - 2.0 * y + 0.25 * z
    quad = lin + 0.5 * x * x - 0.75 * y * y + 2.0 * z * z + 0.2 * x * y - 0.3 * y * z + 0.1 * x * z
    inner = (slice(1, -1),) * 3
    g = ref.gradient(lin)
    assert np.abs(g[0][inner] - 1.5).max() < 1e-13
    assert np.abs(g[1][inner] + 2.0).max() < 1e-13
    assert np.abs(g[2][inner] - 0.25).max() < 1e-13
    gq = ref.gradient(quad)
    assert np.abs(gq[0][inner] - (1.5 + x + 0.2 * y + 0.1 * z)[inner]).max() < 1e-12
    assert np.abs(ref.laplacian(quad)[inner] - (1.0 - 1.5 + 4.0)).max() < 1e-12
    assert np.abs(ref.laplacian(np.full(shape, 3.7))).max() == 0.0
    # divergence = Eq. 18 component-wise (R17)
    G = np.stack([2.0 * x + y, -y + 0.5 * z, 3.0 * z - x])
    assert np.abs(ref.divergence(G)[inner] - (2.0 - 1.0 + 3.0)).max() < 1e-12


def test_p4_printed_eq19_is_not_a_laplacian(lat):
    """The printed Eq. 19 gives (11/9) Psi on a constant -- documents why R10 repairs it."""
    _, w, _ = lat
    centre = 13
    printed = (w.sum() - w[centre] - w[centre]) / CS2
    assert printed == pytest.approx(11.0 / 9.0, rel=1e-14)


@pytest.mark.parametrize("bc", [(0, 0, 0), (0, 0, 1), (1, 0, 1), (1, 1, 1)])
def test_p4_discrete_divergence_sums_to_zero(ref, bc):
    """Telescoping: the box total of the discrete divergence vanishes for periodic axes and for
    walls with either ghost rule (this is what makes Allen-Cahn conservative, R16/R19)."""
    rng = np.random.default_rng(7)
    G = rng.normal(size=(3, 6, 7, 8))
    for rule in (0, 1):
        dv = ref.divergence(G, bc, rule)
        assert abs(dv.sum()) < 1e-12 * np.abs(dv).sum()
    psi = rng.normal(size=(6, 7, 8))
    lp = ref.laplacian(psi, bc)
    assert abs(lp.sum()) < 1e-12 * np.abs(lp).sum()


def test_p4_wall_ghosts_mirror(ref):
    """R19: with a wall, the gradient of a field that is even about the wall plane has zero
    normal component at the wall in the limit; check against an explicitly mirrored periodic
    extension (a periodic box twice as long holding the field and its mirror image)."""
    rng = np.random.default_rng(3)
    nz, ny, nx = 5, 6, 7
    psi = rng.normal(size=(nz, ny, nx))
    ext = np.concatenate([psi, psi[::-1]], axis=0)          # even mirror about both z walls
    g_wall = ref.gradient(psi, (0, 0, 1))
    g_ext = ref.gradient(ext, (0, 0, 0))
    assert np.abs(g_wall - g_ext[:, :nz]).max() < 1e-14
    l_wall = ref.laplacian(psi, (0, 0, 1))
    assert np.abs(l_wall - ref.laplacian(ext)[:nz]).max() < 1e-14
    # vector field with odd normal component (rule 1) / fully odd (rule 0)
    G = rng.normal(size=(3, nz, ny, nx))
    ext1 = np.concatenate([G, G[:, ::-1] * np.array([1, 1, -1])[:, None, None, None]], axis=1)
    ext0 = np.concatenate([G, -G[:, ::-1]], axis=1)
    assert np.abs(ref.divergence(G, (0, 0, 1), 1) - ref.divergence(ext1)[:nz]).max() < 1e-14
    assert np.abs(ref.divergence(G, (0, 0, 1), 0) - ref.divergence(ext0)[:nz]).max() < 1e-14

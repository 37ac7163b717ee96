"""Seeded synthetic inputs for the TSLB hot path.

This module serves BOTH the CUDA path and the CPU oracle, so it holds none of the method's
arithmetic: only initial fields (tanh droplets / bubbles, counter-based noise, a solenoidal
Fourier velocity field) and the parameter sets of the five BASELINE.json configs.  numpy only.

Arrays are fp64, shaped (nz, ny, nx) with x fastest (idx = ix + nx (iy + ny iz)); vectors are
(3, nz, ny, nx).  Box centre is (n-1)/2 per axis.  The workloads stand in for the paper's own
simulations, which are not specified well enough to reproduce.
"""
import numpy as np

PERIODIC, WALL = 0, 1
_M64 = (1 << 64) - 1


def splitmix64(x):
    """Counter-based hash on uint64 arrays (public-domain splitmix64 finaliser)."""
    x = np.asarray(x, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = x + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def noise_u(shape, amp, seed):
    """u_al(x) = amp (2 U01(splitmix64(seed 2^40 + al N + idx)) - 1); order-independent."""
    nz, ny, nx = shape
    n = nz * ny * nx
    out = np.empty((3, nz, ny, nx))
    idx = np.arange(n, dtype=np.uint64)
    for al in range(3):
        key = np.uint64((seed << 40) & _M64) + np.uint64(al * n) + idx
        u01 = (splitmix64(key) >> np.uint64(11)).astype(np.float64) * (1.0 / (1 << 53))
        out[al] = (amp * (2.0 * u01 - 1.0)).reshape(nz, ny, nx)
    return out


def _axis_dist(n, c, periodic):
    d = np.arange(n, dtype=np.float64) - c
    if periodic:
        d = d - n * np.round(d / n)          # minimum image
    return d


def sphere_profile(shape, centre, radius, delta, bc=(0, 0, 0)):
    """0.5 (1 + tanh(2 (R - r)/delta)): 1 inside the sphere (reading R11 of the tanh profile,
    PAPER.md:73).  centre = (cx, cy, cz) in node coordinates; minimum image on periodic axes."""
    nz, ny, nx = shape
    dx = _axis_dist(nx, centre[0], bc[0] == PERIODIC)
    dy = _axis_dist(ny, centre[1], bc[1] == PERIODIC)
    dz = _axis_dist(nz, centre[2], bc[2] == PERIODIC)
    r = np.sqrt(dz[:, None, None] ** 2 + dy[None, :, None] ** 2 + dx[None, None, :] ** 2)
    return 0.5 * (1.0 + np.tanh(2.0 * (radius - r) / delta))


def add_sphere_local(phi, centre, radius, delta, reach=42.0):
    """phi += sphere profile, evaluated only inside the periodic box |d| <= R + reach, outside
    of which the fp64 profile is exactly 0 (tanh(-21) rounds to -1)."""
    nz, ny, nx = phi.shape
    half = int(np.ceil(radius + reach))
    idx = []
    dist = []
    for n, c in ((nx, centre[0]), (ny, centre[1]), (nz, centre[2])):
        i0 = int(np.floor(c)) - half
        ii = np.arange(i0, i0 + 2 * half + 2)
        if ii.size >= n:
            ii = np.arange(n)
            d = _axis_dist(n, c, True)
        else:
            d = ii - c
            ii = ii % n
        idx.append(ii)
        dist.append(d.astype(np.float64))
    r = np.sqrt(dist[2][:, None, None] ** 2 + dist[1][None, :, None] ** 2
                + dist[0][None, None, :] ** 2)
    phi[np.ix_(idx[2], idx[1], idx[0])] += 0.5 * (1.0 + np.tanh(2.0 * (radius - r) / delta))


def flat_interface(shape, axis, pos, delta, liquid_below=True):
    """Flat tanh interface normal to `axis` (0=x,1=y,2=z) at coordinate `pos` (no wrap)."""
    nz, ny, nx = shape
    n = (nx, ny, nz)[axis]
    xi = pos - np.arange(n, dtype=np.float64)
    if not liquid_below:
        xi = -xi
    prof = 0.5 * (1.0 + np.tanh(2.0 * xi / delta))
    shp = [1, 1, 1]
    shp[2 - axis] = n
    return np.broadcast_to(prof.reshape(shp), shape).copy()


def emulsion(shape, n_drops, rmin, rmax, delta, seed, gap=8.0):
    """Seeded dart throwing in sequence: uniform real-valued centres, radius uniform in
    [rmin, rmax], reject if the minimum-image centre distance < r_i + r_j + gap."""
    nz, ny, nx = shape
    rng = np.random.Generator(np.random.PCG64(seed))
    box = np.array([nx, ny, nz], dtype=np.float64)
    centres, radii = [], []
    while len(centres) < n_drops:
        r = rng.uniform(rmin, rmax)
        c = rng.uniform(0.0, 1.0, 3) * box
        ok = True
        for cj, rj in zip(centres, radii):
            d = c - cj
            d -= box * np.round(d / box)
            if np.sqrt((d * d).sum()) < r + rj + gap:
                ok = False
                break
        if ok:
            centres.append(c)
            radii.append(r)
    phi = np.zeros(shape)
    for c, r in zip(centres, radii):
        add_sphere_local(phi, c, r, delta)
    np.minimum(phi, 1.0, out=phi)
    return phi, np.array(centres), np.array(radii)


def solenoidal_u(shape, n_modes, amp, seed):
    """u = curl(psi), psi a sum of n_modes Fourier modes with integer wavevectors in -2..2 and
    seeded amplitudes/phases, evaluated analytically and rescaled to max|u| = amp."""
    nz, ny, nx = shape
    rng = np.random.Generator(np.random.PCG64(seed))
    ks = []
    while len(ks) < n_modes:
        k = rng.integers(-2, 3, 3)
        if np.any(k != 0):
            ks.append(k)
    amps = rng.normal(size=(n_modes, 3))
    phases = rng.uniform(0.0, 2.0 * np.pi, n_modes)
    x = 2.0 * np.pi * np.arange(nx) / nx
    y = 2.0 * np.pi * np.arange(ny) / ny
    z = 2.0 * np.pi * np.arange(nz) / nz
    u = np.zeros((3, nz, ny, nx))
    for k, a, ph in zip(ks, amps, phases):
        # psi = a sin(k.x + ph)  ->  curl psi = (k x a) cos(k.x + ph)
        kxa = np.cross(k.astype(np.float64), a)
        for iz in range(nz):
            arg = k[0] * x[None, :] + k[1] * y[:, None] + (k[2] * z[iz] + ph)
            cs = np.cos(arg)
            for al in range(3):
                u[al, iz] += kxa[al] * cs
    u *= amp / np.sqrt((u * u).sum(axis=0)).max()
    return u


# ------------------------------------------------------------------ the five configs -----
def base_params(**kw):
    p = dict(rho_l=1.0, rho_g=1e-3, mu_l=1.0 / 60.0, mu_g=1.0 / 6000.0, sigma=1e-3, delta=4.0,
             mobility=0.05, body_accel=(0.0, 0.0, 0.0), bc=(PERIODIC, PERIODIC, PERIODIC))
    p.update(kw)
    return p


def static_droplet(n=32, radius=8.0, seed=1, noise=1e-6):
    """BASELINE.json configs[0] / [1]: centred liquid droplet, rho ratio 1000, mu ratio 100."""
    shape = (n, n, n)
    prm = base_params()
    c = (n - 1) / 2.0
    phi = sphere_profile(shape, (c, c, c), radius, prm["delta"], prm["bc"])
    u = noise_u(shape, noise, seed) if noise else np.zeros((3,) + shape)
    return dict(name=f"static_droplet_{n}_R{radius:g}", shape=shape, params=prm, phi=phi, u=u)


def rising_bubble(nx=128, ny=128, nz=256, radius=16.0, height=40.0):
    """configs[2]: Eo = rho_l g R^2/sigma = 10, Mo = 1e-3, sqrt(2 g R) = 0.02,
    scaled with the radius so reduced-size variants keep the same groups."""
    s = radius / 16.0
    g = 1.25e-5 / s
    sigma = g * radius ** 2 / 10.0
    mu_l = (1e-3 * sigma ** 3 / (g * (1.0 - 1e-3))) ** 0.25
    prm = base_params(rho_g=1e-3, sigma=sigma, mu_l=mu_l, mu_g=mu_l / 100.0,
                      body_accel=(0.0, 0.0, -g), bc=(PERIODIC, PERIODIC, WALL))
    shape = (nz, ny, nx)
    phi = 1.0 - sphere_profile(shape, ((nx - 1) / 2.0, (ny - 1) / 2.0, height), radius,
                               prm["delta"], prm["bc"])
    return dict(name=f"rising_bubble_{nx}x{ny}x{nz}", shape=shape, params=prm, phi=phi,
                u=np.zeros((3,) + shape))


def head_on_collision(n=256, radius=24.0, half_sep=40.0, speed=0.05, seed=3, noise=1e-6):
    """configs[3] (graded): We = rho_l U^2 D/sigma = 40 with U = 2 speed the relative velocity,
    Re = U D/nu_l = 1440, rho ratio 800, mu ratio 50."""
    shape = (n, n, n)
    U, D = 2.0 * speed, 2.0 * radius
    sigma = 1.0 * U * U * D / 40.0
    mu_l = U * D / 1440.0
    prm = base_params(rho_g=1.0 / 800.0, sigma=sigma, mu_l=mu_l, mu_g=mu_l / 50.0)
    c = (n - 1) / 2.0
    phi1 = sphere_profile(shape, (c - half_sep, c, c), radius, prm["delta"], prm["bc"])
    phi2 = sphere_profile(shape, (c + half_sep, c, c), radius, prm["delta"], prm["bc"])
    u = noise_u(shape, noise, seed) if noise else np.zeros((3,) + shape)
    u[0] += speed * phi1 - speed * phi2
    return dict(name=f"head_on_collision_{n}", shape=shape, params=prm, phi=phi1 + phi2, u=u)


def off_axis_collision(n=256, impact=0.38, weber=53.0, radius=None, half_sep=None, speed=0.05,
                       seed=4, noise=1e-6):
    """off-axis binary collision.  As head_on_collision, but
    the droplet centres are offset by b = impact * D along y, perpendicular to the relative
    velocity (`impact` = the paper's x, "the ratio of the distance between the centers of the
    droplets and their diameter", 0.28-0.5 there).  Oh = sqrt(We)/Re is kept at the paper's
    0.0044, so Re follows from We (We 53 -> Re 1655).  rho ratio 800, mu ratio 50 as configs[3].
    Sizes scale with the box like bench.py's collision workload (R = 24, half_sep = 40 at 256)."""
    shape = (n, n, n)
    s = n / 256.0
    radius = 24.0 * s if radius is None else radius
    half_sep = 40.0 * s if half_sep is None else half_sep
    U, D = 2.0 * speed, 2.0 * radius
    sigma = 1.0 * U * U * D / weber
    reynolds = np.sqrt(weber) / 0.0044
    mu_l = U * D / reynolds
    prm = base_params(rho_g=1.0 / 800.0, sigma=sigma, mu_l=mu_l, mu_g=mu_l / 50.0)
    c = (n - 1) / 2.0
    b = 0.5 * impact * D
    phi1 = sphere_profile(shape, (c - half_sep, c - b, c), radius, prm["delta"], prm["bc"])
    phi2 = sphere_profile(shape, (c + half_sep, c + b, c), radius, prm["delta"], prm["bc"])
    u = noise_u(shape, noise, seed) if noise else np.zeros((3,) + shape)
    u[0] += speed * phi1 - speed * phi2
    return dict(name=f"off_axis_collision_{n}_x{impact:g}_We{weber:g}", shape=shape, params=prm,
                phi=phi1 + phi2, u=u)


def droplet_train(nx=128, ny=128, nz=768, n_drops=5, spacing=2.0, weber=40.0, speed=0.05,
                  bond=1.0, seed=6, noise=1e-6):
    """SURVEY.md NEXT-2, second workload: a train of `n_drops` droplets falling
    onto the bottom wall "under the effect of an initial velocity and the gravity"; periodic in x
    and y, no-slip neutral-wetting walls at bottom and top (bc z = WALL: halfway bounce-back and
    mirrored phi, R19), box 1 : 1 : 6 like the paper's 500 x 500 x 3000.  `spacing` = the paper's
    Delta L in diameters (2 and 6 there), We = rho_l U^2 D / sigma = 40 with U = `speed` the impact
    velocity.  Not given by the paper, chosen here: D = nx / 5; the lowest droplet starts 1.5 D
    above the wall; Oh = 0.0044 as in its collision study with nu_l floored at 1/300
    (tau_l >= 0.51, configs[3]'s value) so that reduced boxes stay inside the scheme's stable range;
    g from a Bond number rho_l g D^2 / sigma = `bond`, acting on the liquid (the dispersed phase
    here: force density (rho - rho_g) g, TSLB_FLAG_BODY_HEAVY, R20b); rho ratio 800, mu
    ratio 50 (configs[3])."""
    shape = (nz, ny, nx)
    D = nx / 5.0
    radius = 0.5 * D
    sigma = 1.0 * speed * speed * D / weber
    reynolds = np.sqrt(weber) / 0.0044
    mu_l = max(speed * D / reynolds, 1.0 / 300.0)
    g = bond * sigma / (D * D)
    prm = base_params(rho_g=1.0 / 800.0, sigma=sigma, mu_l=mu_l, mu_g=mu_l / 50.0,
                      body_accel=(0.0, 0.0, -g), bc=(PERIODIC, PERIODIC, WALL), body_heavy=True)
    top = 1.5 * D + (n_drops - 1) * spacing * D + radius
    if top + 2.0 * prm["delta"] > nz - 1:
        raise ValueError("droplet_train: %d droplets at spacing %g D do not fit nz = %d"
                         % (n_drops, spacing, nz))
    phi = np.zeros(shape)
    for k in range(n_drops):
        phi += sphere_profile(shape, ((nx - 1) / 2.0, (ny - 1) / 2.0, 1.5 * D + k * spacing * D),
                              radius, prm["delta"], prm["bc"])
    u = noise_u(shape, noise, seed) if noise else np.zeros((3,) + shape)
    u[2] -= speed * phi
    return dict(name=f"droplet_train_{nx}x{ny}x{nz}_dL{spacing:g}", shape=shape, params=prm,
                phi=phi, u=u)


def emulsion_sweep(n=384, n_drops=200, seed=5):
    """configs[4]: 200 droplets, radii in [6,14], solenoidal velocity of amplitude 0.02."""
    shape = (n, n, n)
    prm = base_params()
    phi, _, _ = emulsion(shape, n_drops, 6.0, 14.0, prm["delta"], seed)
    u = solenoidal_u(shape, 16, 0.02, seed + 1)
    return dict(name=f"emulsion_{n}", shape=shape, params=prm, phi=phi, u=u)

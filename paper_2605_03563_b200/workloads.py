"""Seeded synthetic inputs for the five BASELINE.json configs and the paper's two-sphere test.

This module serves both the CUDA path and the CPU oracle.  It holds NONE of the method's arithmetic: it only builds
grids, densities / right-hand sides and closed-form reference potentials on the host with numpy.  All random numbers
come from a counter-based hash of (seed, linear index), so any implementation can regenerate them.
Arrays are numpy float64 with shape (n2, n1, n0): the method's axis 0 (x or r) is the fastest (last numpy) axis.
The recipe of every config is restated in DESIGN.md ("Input recipe").
"""
import math

import numpy as np

CARTESIAN, SPHERICAL = 0, 1
BC_DIRICHLET_GHOST, BC_PERIODIC, BC_NEUMANN0, BC_AXIS = 0, 1, 2, 3

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def hash_u64(seed, idx):
    """splitmix64 finaliser of (seed, idx); idx is an integer array."""
    with np.errstate(over="ignore"):
        z = (np.asarray(idx, dtype=np.uint64) + np.uint64(1)) * np.uint64(0x9E3779B97F4A7C15)
        z = z ^ (np.uint64(seed) * np.uint64(0xD1B54A32D192ED03))
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def hash_uniform(seed, idx):
    """Uniform [0,1) doubles with 53 random bits."""
    return (hash_u64(seed, idx) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def hash_normal(seed, idx):
    """Standard normals by Box-Muller from two hashed uniforms per index."""
    idx = np.asarray(idx, dtype=np.uint64)
    u1 = hash_uniform(seed, idx * np.uint64(2))
    u2 = hash_uniform(seed, idx * np.uint64(2) + np.uint64(1))
    return np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(2.0 * math.pi * u2)


def _axes(n, origin, h):
    return [origin[a] + h[a] * np.arange(n[a]) for a in range(3)]


def _mesh(n, origin, h):
    x, y, z = _axes(n, origin, h)
    return x[None, None, :], y[None, :, None], z[:, None, None]


# ---------------------------------------------------------------------------------------------------------------------
def config1(n=32):
    """Unit cube, vertex-centred, Dirichlet phi=0, rhs = -3 pi^2 sin sin sin; exact phi = sin sin sin."""
    h = 1.0 / (n + 1)
    shape, spacing, origin = (n, n, n), (h, h, h), (h, h, h)
    X, Y, Z = _mesh(shape, origin, spacing)
    exact = np.sin(math.pi * X) * np.sin(math.pi * Y) * np.sin(math.pi * Z)
    rhs = -3.0 * math.pi ** 2 * exact
    return dict(name="config1", shape=shape, spacing=spacing, origin=origin, coord=CARTESIAN, order=2,
                bc=(BC_DIRICHLET_GHOST,) * 6, rhs=np.ascontiguousarray(rhs), exact=np.ascontiguousarray(exact),
                omega=2.0 / (1.0 + math.sin(math.pi * h)), nsweeps=200)


def _sphere_fraction(n, origin, h, centre, radius, sub=8):
    """Fraction of every cell inside the sphere: 0/1 for cells clearly outside/inside, sub^3 midpoint sampling else."""
    X, Y, Z = _mesh(n, origin, h)
    d = np.sqrt((X - centre[0]) ** 2 + (Y - centre[1]) ** 2 + (Z - centre[2]) ** 2)
    half_diag = 0.5 * math.sqrt(h[0] ** 2 + h[1] ** 2 + h[2] ** 2)
    frac = (d < radius - half_diag).astype(np.float64)
    kk, jj, ii = np.nonzero(np.abs(d - radius) <= half_diag)
    x, y, z = _axes(n, origin, h)
    off = (np.arange(sub) + 0.5) / sub - 0.5
    ox, oy, oz = off[None, None, :], off[None, :, None], off[:, None, None]
    for k, j, i in zip(kk, jj, ii):
        dd = (x[i] + ox * h[0] - centre[0]) ** 2 + (y[j] + oy * h[1] - centre[1]) ** 2 + \
             (z[k] + oz * h[2] - centre[2]) ** 2
        frac[k, j, i] = np.count_nonzero(dd < radius * radius) / float(sub ** 3)
    return frac


def uniform_sphere_potential(X, Y, Z, centre, radius, rho0, G=1.0):
    d = np.sqrt((X - centre[0]) ** 2 + (Y - centre[1]) ** 2 + (Z - centre[2]) ** 2)
    M = 4.0 / 3.0 * math.pi * radius ** 3 * rho0
    inside = -2.0 * math.pi * G * rho0 * (radius ** 2 - d ** 2 / 3.0)
    with np.errstate(divide="ignore"):
        outside = -G * M / d
    return np.where(d < radius, inside, outside)


def config2(n=128):
    """Box [-1,1]^3, cell-centred; uniform sphere R=0.25 at (0.05,-0.03,0.02), rho=1 (cell-averaged); G=1."""
    h = 2.0 / n
    shape, spacing, origin = (n, n, n), (h, h, h), (-1 + h / 2,) * 3
    centre, radius = (0.05, -0.03, 0.02), 0.25
    rho = _sphere_fraction(shape, origin, spacing, centre, radius)
    X, Y, Z = _mesh(shape, origin, spacing)
    exact = uniform_sphere_potential(X, Y, Z, centre, radius, 1.0)
    return dict(name="config2", shape=shape, spacing=spacing, origin=origin, coord=CARTESIAN, order=2,
                bc=(BC_DIRICHLET_GHOST,) * 6, rho=rho, rhs=4.0 * math.pi * rho, exact=np.ascontiguousarray(exact),
                G=1.0, lmax=4, rtol=1e-8, centre=centre, radius=radius)


def config3(n=256, seed=20260503):
    """Box [-1,1]^3, cell-centred; 3 seeded Gaussian blobs + 1 % seeded uniform noise; G=1, lmax=8."""
    h = 2.0 / n
    shape, spacing, origin = (n, n, n), (h, h, h), (-1 + h / 2,) * 3
    u = hash_uniform(seed, np.arange(15))
    X, Y, Z = _mesh(shape, origin, spacing)
    rho = np.zeros((n, n, n))
    exact = np.zeros((n, n, n))
    blobs = []
    for b in range(3):
        c = -0.4 + 0.8 * u[5 * b: 5 * b + 3]
        sigma = 0.05 + 0.10 * u[5 * b + 3]
        amp = 0.5 + 1.5 * u[5 * b + 4]
        blobs.append((tuple(c), float(sigma), float(amp)))
        d2 = (X - c[0]) ** 2 + (Y - c[1]) ** 2 + (Z - c[2]) ** 2
        rho += amp * np.exp(-d2 / (2 * sigma ** 2))
        d = np.sqrt(d2)
        M = amp * (2 * math.pi) ** 1.5 * sigma ** 3
        from scipy.special import erf
        with np.errstate(divide="ignore", invalid="ignore"):
            exact += np.where(d > 0, -M * erf(d / (math.sqrt(2) * sigma)) / d, -M * math.sqrt(2 / math.pi) / sigma)
    noise = 2.0 * hash_uniform(seed + 1, np.arange(n ** 3, dtype=np.uint64)).reshape(n, n, n) - 1.0
    rho = rho * (1.0 + 0.01 * noise)
    return dict(name="config3", shape=shape, spacing=spacing, origin=origin, coord=CARTESIAN, order=2,
                bc=(BC_DIRICHLET_GHOST,) * 6, rho=rho, rhs=4.0 * math.pi * rho, exact=exact, G=1.0, lmax=8,
                blobs=blobs, ncycles=10)


def config4(n=512, seed=20260504):
    """Periodic unit box, 6th-order 19-point star; rhs = zero-mean unit-variance Gaussian random field, P(k) ~ k^-2,
    cut off at |k| > n/4 (integer wavenumbers)."""
    import scipy.fft as sfft
    h = 1.0 / n
    w = hash_normal(seed, np.arange(n ** 3, dtype=np.uint64)).reshape(n, n, n)
    W = sfft.rfftn(w, workers=-1)
    del w
    k1 = np.fft.fftfreq(n, d=1.0 / n)
    kz, ky, kx = k1[:, None, None], k1[None, :, None], np.fft.rfftfreq(n, d=1.0 / n)[None, None, :]
    kk = np.sqrt(kx * kx + ky * ky + kz * kz)
    with np.errstate(divide="ignore"):
        filt = np.where((kk > 0) & (kk <= n / 4.0), 1.0 / kk, 0.0)
    W *= filt
    rhs = sfft.irfftn(W, s=(n, n, n), workers=-1)
    del W
    rhs -= rhs.mean()
    rhs /= rhs.std()
    return dict(name="config4", shape=(n, n, n), spacing=(h, h, h), origin=(0.0, 0.0, 0.0), coord=CARTESIAN, order=6,
                bc=(BC_PERIODIC,) * 6, rhs=np.ascontiguousarray(rhs), fixed_iters=500, rtol=1e-10)


def spherical_edges(nr, nt, nph, r_in=0.01, r_out=1.0):
    q = (r_out / r_in) ** (1.0 / nr)
    re = r_in * q ** np.arange(nr + 1)
    re[-1] = r_out
    te = math.pi * np.arange(nt + 1) / nt
    pe = 2.0 * math.pi * np.arange(nph + 1) / nph
    return re, te, pe


def config5(nr=256, nt=128, nph=256):
    """Spherical (r,theta,phi), r log-spaced in [0.01,1]; off-centre uniform sphere + 1e-3/r^2 envelope; G=1."""
    re, te, pe = spherical_edges(nr, nt, nph)
    rc = np.sqrt(re[:-1] * re[1:])
    tc = 0.5 * (te[:-1] + te[1:])
    pc = 0.5 * (pe[:-1] + pe[1:])
    R, T, P = rc[None, None, :], tc[None, :, None], pc[:, None, None]
    X, Y, Z = R * np.sin(T) * np.cos(P), R * np.sin(T) * np.sin(P), R * np.cos(T) + 0 * P
    r0, t0, p0 = 0.3, math.pi / 3, 0.0
    c = (r0 * math.sin(t0) * math.cos(p0), r0 * math.sin(t0) * math.sin(p0), r0 * math.cos(t0))
    d = np.sqrt((X - c[0]) ** 2 + (Y - c[1]) ** 2 + (Z - c[2]) ** 2)
    rho = (d < 0.2).astype(np.float64) + 1e-3 / (R * R) + 0 * d
    rho = np.ascontiguousarray(rho)
    return dict(name="config5", shape=(nr, nt, nph), spacing=(1.0, 1.0, 1.0), origin=(0.0, 0.0, 0.0),
                edges=(re, te, pe), coord=SPHERICAL, order=2,
                bc=(BC_NEUMANN0, BC_DIRICHLET_GHOST, BC_AXIS, BC_AXIS, BC_PERIODIC, BC_PERIODIC),
                rho=rho, rhs=4.0 * math.pi * rho, G=1.0, lmax=8, rtol=1e-8)


# ---------------------------------------------------------------------------------------------------------------------
def two_spheres(n, cell_centred=True):
    """The paper's Cartesian test: spheres of Eq. 23 (n=2) at (0,0,0.4) and (0,0,-0.2), a=0.08,
    M = 1, 2 in [-1,1]^3, point-sampled; analytic potential of Eq. 24 (G=1)."""
    h = 2.0 / n if cell_centred else 2.0 / (n + 1)
    o = -1 + h / 2 if cell_centred else -1 + h
    shape, spacing, origin = (n, n, n), (h, h, h), (o, o, o)
    X, Y, Z = _mesh(shape, origin, spacing)

    def rho_phi(Xa, Ya, Za):
        rho = 0.0
        phi = 0.0
        for (c, a, M) in (((0.0, 0.0, 0.4), 0.08, 1.0), ((0.0, 0.0, -0.2), 0.08, 2.0)):
            rp = M / (32.0 * math.pi * a ** 3 / 105.0)
            d = np.sqrt((Xa - c[0]) ** 2 + (Ya - c[1]) ** 2 + (Za - c[2]) ** 2)
            w = d / a
            rho = rho + np.where(d < a, rp * (1 - w * w) ** 2, 0.0)
            with np.errstate(divide="ignore"):
                phi = phi + np.where(d < a, 4 * math.pi * rp * a * a * (-1 / 6 + w ** 2 / 6 - w ** 4 / 10 + w ** 6 / 42),
                                     -M / d)
        return rho, phi

    rho, exact = rho_phi(X, Y, Z)
    rho = np.ascontiguousarray(np.broadcast_to(rho, (n, n, n)))
    exact = np.ascontiguousarray(np.broadcast_to(exact, (n, n, n)))

    def potential(Xa, Ya, Za):
        return rho_phi(Xa, Ya, Za)[1]

    return dict(name="two_spheres", shape=shape, spacing=spacing, origin=origin, coord=CARTESIAN, order=2,
                bc=(BC_DIRICHLET_GHOST,) * 6, rho=rho, rhs=4.0 * math.pi * rho, exact=exact, potential=potential, G=1.0)


def analytic_ghost_faces(w, potential, R=1):
    """Ghost-face arrays (layout of include/poisson.h) holding a closed-form potential at the ghost positions."""
    n, h, o = w["shape"], w["spacing"], w["origin"]
    ax = _axes(n, o, h)
    faces = []
    for f in range(6):
        a = f // 2
        a1, a2 = (1, 2) if a == 0 else ((0, 2) if a == 1 else (0, 1))
        out = np.zeros((R, n[a2], n[a1]))
        for layer in range(R):
            ca = o[a] + h[a] * ((n[a] + layer) if (f & 1) else (-1 - layer))
            c = [None, None, None]
            c[a] = np.full((n[a2], n[a1]), ca)
            c[a1] = np.broadcast_to(ax[a1][None, :], (n[a2], n[a1]))
            c[a2] = np.broadcast_to(ax[a2][:, None], (n[a2], n[a1]))
            out[layer] = potential(c[0], c[1], c[2])
        faces.append(out.ravel())
    return faces


def random_field(shape, seed, lo=-1.0, hi=1.0):
    n = shape[0] * shape[1] * shape[2]
    u = hash_uniform(seed, np.arange(n, dtype=np.uint64))
    return (lo + (hi - lo) * u).reshape(shape[2], shape[1], shape[0])

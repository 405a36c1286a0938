"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no keys, tree, MAC, force or SPH sums): it only
draws particle distributions with the shapes of the paper's workloads ("Plummer
model", L165 "sphere with uniform density", L246 white-dwarf pair) and of BASELINE.json's configs.
Every draw is a pure function of (seed, particle index, draw index) through a SplitMix64-style
counter hash, so generation is order independent; coordinates are computed in fp64 and rounded
once to fp32.  The paper uses no public dataset; these stand in for its analytic models.
"""
from __future__ import annotations

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _mix(z: np.ndarray) -> np.ndarray:
    z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def bits64(seed: int, idx: np.ndarray, draw: int) -> np.ndarray:
    """64 random bits per element of idx: a counter-based hash of (seed, idx, draw)."""
    with np.errstate(over="ignore"):
        i = idx.astype(np.uint64)
        z = _mix(i * np.uint64(0x9E3779B97F4A7C15) + np.uint64(seed & 0xFFFFFFFFFFFFFFFF))
        z = _mix(z + np.uint64(draw) * np.uint64(0xD1B54A32D192ED03) + np.uint64(0x632BE59BD9B4E019))
    return z


def uniform01(seed: int, idx: np.ndarray, draw: int) -> np.ndarray:
    """u in [0,1) with 53 random bits, fp64."""
    return (bits64(seed, idx, draw) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def _isotropic(seed, idx, d0):
    cz = 1.0 - 2.0 * uniform01(seed, idx, d0)
    ph = 2.0 * np.pi * uniform01(seed, idx, d0 + 1)
    sz = np.sqrt(np.maximum(0.0, 1.0 - cz * cz))
    return sz * np.cos(ph), sz * np.sin(ph), cz


def _pack(x, y, z, m) -> np.ndarray:
    out = np.empty((len(x), 4), dtype=np.float32)
    out[:, 0] = x
    out[:, 1] = y
    out[:, 2] = z
    out[:, 3] = m
    return out


def plummer(n: int, seed: int, rmax: float = 100.0) -> np.ndarray:
    """Plummer sphere, G = M = scale radius = 1, equal masses (BASELINE configs 1-2).

    r = (u^(-2/3) - 1)^(-1/2), redrawn (next draw index) while r > rmax.  Returns (n,4) fp32
    rows (x, y, z, m)."""
    idx = np.arange(n, dtype=np.uint64)
    r = np.full(n, np.inf)
    todo = np.ones(n, dtype=bool)
    k = 0
    while todo.any():
        u = uniform01(seed, idx[todo], 16 + k)
        u = np.maximum(u, 2.0 ** -53)
        rr = 1.0 / np.sqrt(u ** (-2.0 / 3.0) - 1.0 + 1e-300)
        r[todo] = rr
        todo = r > rmax
        k += 1
    ux, uy, uz = _isotropic(seed, idx, 0)
    return _pack(r * ux, r * uy, r * uz, np.full(n, 1.0 / n))


def hernquist(n: int, seed: int, rmax: float = 100.0) -> np.ndarray:
    """Hernquist halo, M(r) = r^2/(1+r)^2 truncated at rmax (BASELINE config 3)."""
    idx = np.arange(n, dtype=np.uint64)
    umax = (rmax / (1.0 + rmax)) ** 2
    su = np.sqrt(uniform01(seed, idx, 2) * umax)
    r = su / (1.0 - su)
    ux, uy, uz = _isotropic(seed, idx, 0)
    return _pack(r * ux, r * uy, r * uz, np.full(n, 1.0 / n))


def uniform_cube(n: int, seed: int) -> np.ndarray:
    """Uniform random points in [0,1)^3 with 24-bit coordinates (exact in fp32) (config 5)."""
    idx = np.arange(n, dtype=np.uint64)
    c = [(bits64(seed, idx, d) >> np.uint64(40)).astype(np.float64) * 2.0 ** -24 for d in range(3)]
    return _pack(c[0], c[1], c[2], np.full(n, 1.0 / n))


def uniform_sphere(n: int, seed: int) -> np.ndarray:
    """Uniform-density sphere, radius 1, total mass 1."""
    idx = np.arange(n, dtype=np.uint64)
    r = uniform01(seed, idx, 2) ** (1.0 / 3.0)
    ux, uy, uz = _isotropic(seed, idx, 0)
    return _pack(r * ux, r * uy, r * uz, np.full(n, 1.0 / n))


def cold_sphere(n: int, seed: int, u0: float = 0.05):
    """The paper's gravity+SPH test ("Cold Collapse Test" [50],[51]): an isothermal sphere,
    rho ~ r^-2 (M(<r) ~ r: the radius is uniform in [0,1)), M = R = G = 1, at rest, cold (specific internal
    energy u0 << |W|/M = 1).  Returns dict pos_mass (n,4), vel (n,4) zeros, u (n,), h (n,) support radius for
    ~50 neighbours from the model density rho(r) = 1/(4 pi r^2)."""
    idx = np.arange(n, dtype=np.uint64)
    r = np.maximum(uniform01(seed, idx, 2), 1e-6)
    ux, uy, uz = _isotropic(seed, idx, 0)
    m = 1.0 / n
    rho = 1.0 / (4.0 * np.pi * r * r)
    h = np.minimum((3.0 * 50.0 * m / (4.0 * np.pi * rho)) ** (1.0 / 3.0), 0.3)
    return dict(pos_mass=_pack(r * ux, r * uy, r * uz, np.full(n, m)), vel=np.zeros((n, 4), np.float32),
                u=np.full(n, u0, np.float32), h=h.astype(np.float32))


def lattice(k: int, spacing: float = 1.0, mass: float = 1.0) -> np.ndarray:
    """k^3 simple cubic lattice, first point at the origin."""
    g = np.arange(k, dtype=np.float64) * spacing
    x, y, z = np.meshgrid(g, g, g, indexing="ij")
    return _pack(x.ravel(), y.ravel(), z.ravel(), np.full(k ** 3, mass))


def lane_emden(n_poly: float = 1.5, dxi: float = 1e-4):
    """RK4 solution of theta'' + 2 theta'/xi + theta^n = 0. Returns xi, theta, -xi^2 theta'
    (the enclosed-mass function), all up to the first zero xi_1."""
    def f(xi, th, ph):   # ph = xi^2 theta'
        return ph / (xi * xi), -(max(th, 0.0) ** n_poly) * xi * xi

    xi = 1e-6
    th = 1.0 - xi * xi / 6.0
    ph = -(xi ** 3) / 3.0
    xs, ths, ms = [xi], [th], [-ph]
    while th > 0.0:
        k1 = f(xi, th, ph)
        k2 = f(xi + dxi / 2, th + dxi / 2 * k1[0], ph + dxi / 2 * k1[1])
        k3 = f(xi + dxi / 2, th + dxi / 2 * k2[0], ph + dxi / 2 * k2[1])
        k4 = f(xi + dxi, th + dxi * k3[0], ph + dxi * k3[1])
        th_new = th + dxi / 6 * (k1[0] + 2 * k2[0] + 2 * k3[0] + k4[0])
        ph_new = ph + dxi / 6 * (k1[1] + 2 * k2[1] + 2 * k3[1] + k4[1])
        if th_new <= 0.0:
            frac = th / (th - th_new)
            xs.append(xi + frac * dxi)
            ths.append(0.0)
            ms.append(-(ph + frac * (ph_new - ph)))
            break
        xi, th, ph = xi + dxi, th_new, ph_new
        xs.append(xi)
        ths.append(th)
        ms.append(-ph)
    return np.array(xs), np.array(ths), np.array(ms)


def wd_pair(n: int, seed: int, m1: float = 0.6, m2: float = 0.9, n_ngb: float = 50.0,
            gamma: float = 5.0 / 3.0):
    """Two n=1.5 polytropes in contact (BASELINE config 4; stands in for the paper's WD models,
    PAPER L246, which need external stellar models and the Helmholtz EOS).

    Returns dict with pos_mass (n,4) fp32, h (n,) fp32 SUPPORT radius, u (n,) fp32 specific
    internal energy, vel (n,4) fp32 (rigid circular orbit, w=0)."""
    xs, ths, ms = lane_emden(1.5)
    xi1, mu1 = xs[-1], ms[-1]
    mtot = m1 + m2
    mp = mtot / n
    n1 = int(round(n * m1 / mtot))
    radii = (1.0, (m2 / m1) ** (-1.0 / 3.0))
    masses = (m1, m2)
    counts = (n1, n - n1)
    sep = radii[0] + radii[1]
    cx = (-sep * m2 / mtot, sep * m1 / mtot)
    omega = np.sqrt(mtot / sep ** 3)
    pos = np.empty((n, 4), dtype=np.float32)
    h = np.empty(n, dtype=np.float32)
    u = np.empty(n, dtype=np.float32)
    vel = np.zeros((n, 4), dtype=np.float32)
    start = 0
    for s in range(2):
        cnt, R, M = counts[s], radii[s], masses[s]
        idx = np.arange(start, start + cnt, dtype=np.uint64)
        q = uniform01(seed, idx, 2)
        xi = np.interp(q * mu1, ms, xs)
        th = np.maximum(np.interp(xi, xs, ths), 0.0)
        a = R / xi1                                   # length scale
        rho_c = M / (4.0 * np.pi * a ** 3 * mu1)
        rho = rho_c * th ** 1.5
        K = 4.0 * np.pi * a * a / (2.5 * rho_c ** (-1.0 / 3.0))   # (n+1) K rho_c^(1/n-1) = 4 pi G a^2
        r = a * xi
        ux, uy, uz = _isotropic(seed, idx, 0)
        x = cx[s] + r * ux
        y = r * uy
        z = r * uz
        sl = slice(start, start + cnt)
        pos[sl, 0], pos[sl, 1], pos[sl, 2], pos[sl, 3] = x, y, z, mp
        with np.errstate(divide="ignore"):
            hh = (3.0 * n_ngb * mp / (4.0 * np.pi * np.maximum(rho, 1e-300))) ** (1.0 / 3.0)
        h[sl] = np.minimum(hh, 0.2 * R)
        u[sl] = K * rho ** (2.0 / 3.0) / (gamma - 1.0)
        vel[sl, 0] = -omega * y
        vel[sl, 1] = omega * x
        start += cnt
    return {"pos_mass": pos, "h": h, "u": u, "vel": vel}


# Named configurations of BASELINE.json (index = config number - 1).
CONFIGS = {
    "C1": dict(kind="plummer", n=16384, eps=0.01, theta=0.5, n_crit=16, group=64),
    "C2": dict(kind="plummer", n=1048576, eps=0.004, theta=0.6, n_crit=16, group=128),
    "C3": dict(kind="hernquist", n=8388608, eps=0.002, theta=0.6, n_crit=16, group=128),
    "C4": dict(kind="wd_pair", n=2097152, eps=0.005, theta=0.5, n_crit=16, group=128, group_sph=64),
    "C5": dict(kind="uniform_cube", n=33554432, eps=0.001, theta=0.5, n_crit=16, group=256),
    # not a BASELINE config: the paper's own gravity benchmark (uniform sphere, r = 1, M = 1,
    # N = 8000 x 1024, Delta = 0.01, n_crit = 16, m_limit = 0.05), run with otoo_gravity_delta (bench.py --mac delta)
    # the paper's gravity+SPH benchmark (Fig. 9: cold collapse, Delta = 0.01, n_crit = 16, m_limit = 0.05;
    # N = 2 M is the size its text quotes, L242); bench.py --workload COLD --mac delta [--n N]
    "COLD": dict(kind="cold_sphere", n=2097152, eps=0.005, theta=0.5, n_crit=16, group=128, group_sph=64, delta=0.01, m_limit=0.05),
    "F4": dict(kind="uniform_sphere", n=8192000, eps=0.002, theta=0.6, n_crit=16, group=128, delta=0.01, m_limit=0.05),
}


def make(kind: str, n: int, seed: int):
    if kind == "plummer":
        return plummer(n, seed)
    if kind == "hernquist":
        return hernquist(n, seed)
    if kind == "uniform_cube":
        return uniform_cube(n, seed)
    if kind == "uniform_sphere":
        return uniform_sphere(n, seed)
    if kind == "wd_pair":
        return wd_pair(n, seed)["pos_mass"]
    if kind == "cold_sphere":
        return cold_sphere(n, seed)["pos_mass"]
    raise ValueError(kind)

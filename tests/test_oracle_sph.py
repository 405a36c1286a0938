"""Pins for the oracle's SPH path (PAPER.md II-C Eq. 4-5; readings R13-R17)."""
import numpy as np
import pytest

from workloads import generators as gen


def W_np(r, h):
    q = r / h
    s = 8.0 / (np.pi * h ** 3)
    return s * np.where(q <= 0.5, 1 - 6 * q ** 2 + 6 * q ** 3, np.where(q < 1, 2 * (1 - q) ** 3, 0.0))


def test_kernel_normalisation_continuity_derivative(orc):
    h = 0.7
    r = np.linspace(0, h, 200001)
    w = np.array([orc.W(x, h) for x in r[::100]])
    rr = r[::100]
    integral = np.trapezoid(4 * np.pi * rr ** 2 * w, rr)
    assert integral == pytest.approx(1.0, rel=1e-6)            # int W d^3r = 1
    assert orc.W(h, h) == 0.0 and orc.W(1.5 * h, h) == 0.0      # L89: zero outside h
    assert orc.W(0.0, h) == pytest.approx(8 / (np.pi * h ** 3))
    e = 1e-9
    assert orc.W(0.5 * h - e, h) == pytest.approx(orc.W(0.5 * h + e, h), rel=1e-7)
    assert orc.dWdr(0.5 * h - e, h) == pytest.approx(orc.dWdr(0.5 * h + e, h), rel=1e-7)
    assert abs(orc.dWdr(h - e, h)) < 1e-12
    for x in (0.1, 0.3, 0.45, 0.55, 0.8, 0.95):
        d = 1e-6
        num = (orc.W(x * h + d, h) - orc.W(x * h - d, h)) / (2 * d)
        assert orc.dWdr(x * h, h) == pytest.approx(num, rel=1e-6)


def test_candidate_lists_are_supersets(orc):
    """Eq. 5 guarantee (L105): the walk's candidate list of a group contains every j with
    r_ij < max(h_i, h_j) for some member i."""
    n, G = 3000, 32
    w = gen.wd_pair(n, 5)
    pm, h = w["pos_mass"], w["h"]
    t = orc.Tree(pm, 8)
    ex = t.export()
    r = t.sph_density(h, G, sums=False)
    sp = pm[ex["perm"]].astype(np.float64)
    sh = h[ex["perm"]].astype(np.float64)
    for g in range(0, t.n_groups(G), 3):
        parts = t.sph_group_list(h, G, g, r["n_parts"][g])
        assert len(np.unique(parts)) == len(parts)
        mem = np.arange(g * G, min((g + 1) * G, n))
        d = np.linalg.norm(sp[mem, None, :3] - sp[None, :, :3], axis=2)
        need = (d < np.maximum(sh[mem, None], sh[None, :])).any(0)
        assert np.isin(np.nonzero(need)[0], parts).all()


def test_density_bruteforce_and_lattice(orc):
    n = 2500
    w = gen.wd_pair(n, 8)
    pm, h = w["pos_mass"], w["h"]
    t = orc.Tree(pm, 16)
    r = t.sph_density(h, 64)
    x = pm[:, :3].astype(np.float64)
    d = np.linalg.norm(x[:, None] - x[None, :], axis=2)
    rho = (pm[None, :, 3] * W_np(d, h[:, None].astype(np.float64))).sum(1)
    assert np.allclose(r["rho"], rho, rtol=1e-10)
    cnt = (d < h[:, None]).sum(1)
    assert np.abs(r["nngb"].astype(int) - cnt).max() <= 1          # fp32 vs fp64 edge decisions
    # simple cubic lattice: interior density equals the finite lattice sum, and ~ m/a^3
    k, a, m = 12, 0.5, 0.25
    lat = gen.lattice(k, a, m)
    hh = np.full(k ** 3, 2.3 * a, np.float32)
    tl = orc.Tree(lat, 16)
    rl = tl.sph_density(hh, 64)
    g = np.arange(-3, 4)
    gx, gy, gz = np.meshgrid(g, g, g, indexing="ij")
    rr = a * np.sqrt(gx ** 2 + gy ** 2 + gz ** 2).ravel()
    want = m * W_np(rr, float(hh[0])).sum()
    idx = np.arange(k ** 3).reshape(k, k, k)[4:8, 4:8, 4:8].ravel()
    assert np.allclose(rl["rho"][idx], want, rtol=1e-12)
    assert want == pytest.approx(m / a ** 3, rel=0.01)
    assert np.all(rl["nngb"][idx] == (rr < float(hh[0])).sum())


def test_pressure_force(orc):
    # (i) brute force + antisymmetry on a WD pair
    n = 2000
    w = gen.wd_pair(n, 3)
    pm, h, u = w["pos_mass"], w["h"], w["u"]
    t = orc.Tree(pm, 16)
    rho = t.sph_density(h, 64)["rho"]
    P = (2.0 / 3.0) * rho * u
    out = t.sph_force(h, rho, P, 64, vel=w["vel"])["acc_dudt"]
    x = pm[:, :3].astype(np.float64)
    hd = h.astype(np.float64)
    dvec = x[:, None] - x[None, :]
    d = np.linalg.norm(dvec, axis=2)
    np.fill_diagonal(d, 1.0)

    def dW(r, hh):
        q = r / hh
        s = 8.0 / (np.pi * hh ** 4)
        return s * np.where(q <= 0.5, -12 * q + 18 * q * q, np.where(q < 1, -6 * (1 - q) ** 2, 0.0))
    gw = 0.5 * (dW(d, hd[:, None]) + dW(d, hd[None, :])) / d
    np.fill_diagonal(gw, 0.0)
    pr = P / rho ** 2
    f = pm[None, :, 3] * (pr[:, None] + pr[None, :]) * gw
    acc = -(f[:, :, None] * dvec).sum(1)
    assert np.allclose(out[:, :3], acc, rtol=1e-9, atol=1e-12 * np.abs(acc).max())
    v = w["vel"][:, :3].astype(np.float64)
    du = 0.5 * (f * ((v[:, None] - v[None, :]) * dvec).sum(2)).sum(1)
    assert np.allclose(out[:, 3], du, rtol=1e-8, atol=1e-11 * np.abs(du).max())
    mom = (pm[:, 3:4] * out[:, :3]).sum(0)
    assert np.all(np.abs(mom) < 1e-12 * (pm[:, 3:4] * np.abs(out[:, :3])).sum())
    # (ii) lattice, uniform P: zero force in the interior; linear P: a ~ -grad P / rho
    k, a, m = 14, 1.0, 1.0
    lat = gen.lattice(k, a, m)
    hh = np.full(k ** 3, 2.3, np.float32)
    tl = orc.Tree(lat, 16)
    rhol = tl.sph_density(hh, 64)["rho"]
    idx = np.arange(k ** 3).reshape(k, k, k)[5:9, 5:9, 5:9].ravel()
    o = tl.sph_force(hh, rhol, np.full(k ** 3, 3.0), 64)["acc_dudt"]
    assert np.abs(o[idx, :3]).max() < 1e-12
    Plin = 10.0 + 0.1 * lat[:, 0].astype(np.float64)
    o = tl.sph_force(hh, rhol, Plin, 64)["acc_dudt"]
    assert np.allclose(o[idx, 0], -0.1 / rhol[idx], rtol=0.05)
    assert np.abs(o[idx, 1:3]).max() < 1e-12


def test_adaptive_h_iteration(orc):
    """Reading R21 (h adapted to a neighbour count, BASELINE config 4 "~50 neighbours").
    Pins: on random points every particle ends within the tolerance from starts 2x too small and too large;
    a converged input is a fixed point (0 updates, h untouched); the returned counts are those of the
    density pass; on a lattice, where the count is a known step function of h (27 for sqrt(3) < h <= 2,
    33 for 2 < h <= sqrt(5)), interior particles end on the right step; max_iter caps the updates."""
    pm = gen.uniform_cube(5000, 5)
    n = len(pm)
    t = orc.Tree(pm, 16)
    for h0 in (0.07, 0.3):
        h, nn, it = t.sph_adapt_h(np.full(n, h0, np.float32), 40.0, 2.0, 60, 32)
        assert 0 < it < 40 and np.all(np.abs(nn.astype(float) - 40.0) <= 2.0)
        assert np.array_equal(nn, t.sph_density(h, 32)["nngb"])
        h2, nn2, it2 = t.sph_adapt_h(h, 40.0, 2.0, 60, 32)
        assert it2 == 0 and np.array_equal(h2, h) and np.array_equal(nn2, nn)
    h3, _, it3 = t.sph_adapt_h(np.full(n, 0.07, np.float32), 40.0, 2.0, 3, 32)
    assert it3 == 3
    k, a = 12, 1.0
    lat = gen.lattice(k, a, 1.0)
    tl = orc.Tree(lat, 8)
    for h0 in (1.3, 3.2):
        h, nn, it = tl.sph_adapt_h(np.full(len(lat), h0, np.float32), 33.0, 2.0, 80, 32)
        inner = np.all((lat[:, :3] >= 3 * a) & (lat[:, :3] <= (k - 4) * a), axis=1)
        assert it < 80 and np.all(nn[inner] == 33)
        assert np.all((h[inner] > 2.0) & (h[inner] <= np.sqrt(5.0)))


def test_div_and_rot_of_linear_velocity_fields(orc):
    """Reading R22 (PAPER L252 step 4: "density, div v, rot v").  Pins: for v = A x the estimates are exactly
    linear in A with one common factor c = -(1/(3 rho)) sum_j m_j r dW/dr (-> 1 as the sum -> integral, since
    -int r W' d^3r = 3 int W = 3): on a lattice interior div v = c tr(A), rot v = c (A32-A23, A13-A31, A21-A12),
    with c within a few per cent of 1; a uniform translation has div = rot = 0; the density is R16's."""
    k, a = 12, 1.0
    pm = gen.lattice(k, a, 1.0)
    n = len(pm)
    x = pm[:, :3].astype(np.float64)
    h = np.full(n, 2.3 * a, np.float32)
    t = orc.Tree(pm, 8)
    inner = np.all((x >= 3 * a) & (x <= (k - 4) * a), axis=1)
    A = np.array([[0.3, -0.7, 0.2], [0.5, -0.1, 0.9], [-0.4, 0.25, 0.6]])
    vel = np.zeros((n, 4), np.float32)
    vel[:, :3] = x @ A.T + np.array([5.0, -3.0, 1.0])              # + a uniform translation
    r = t.sph_divrot(h, vel, 32)
    assert np.allclose(r["rho"], t.sph_density(h, 32)["rho"], rtol=1e-14)
    d = r["divrot"][inner]
    c = d[:, 0] / np.trace(A)
    assert np.allclose(c, c[0], rtol=1e-6) and abs(c[0] - 1.0) < 0.05
    curl = np.array([A[2, 1] - A[1, 2], A[0, 2] - A[2, 0], A[1, 0] - A[0, 1]])
    assert np.allclose(d[:, 1:], c[0] * curl, rtol=1e-5, atol=1e-7)
    vel[:, :3] = np.array([5.0, -3.0, 1.0])
    r0 = t.sph_divrot(h, vel, 32)
    assert np.abs(r0["divrot"]).max() == 0.0
    # rigid rotation: div = 0, rot = 2 Omega (times c)
    Om = np.array([0.2, -0.5, 0.9])
    vel[:, :3] = np.cross(Om, x)
    rr = t.sph_divrot(h, vel, 32)["divrot"][inner]
    assert np.abs(rr[:, 0]).max() < 1e-6 and np.allclose(rr[:, 1:], 2 * c[0] * Om, rtol=1e-5, atol=1e-7)


def test_artificial_viscosity(orc):
    """Reading R24 (PAPER L246 names the scheme, prints no formula).  What the pair form fixes: with alpha = 0 or
    Balsara f = 0 the result is R17's; a receding (expanding) flow feels no viscosity; the viscous pair forces
    are antisymmetric (momentum conserved), the viscous heating is non-negative for every particle and equals
    the kinetic energy it removes (total energy conserved)."""
    n = 3000
    w = gen.wd_pair(n, 11)
    pm, h, u = w["pos_mass"], w["h"], w["u"]
    m = pm[:, 3].astype(np.float64)
    t = orc.Tree(pm, 16)
    rho = t.sph_density(h, 32)["rho"]
    P = (2.0 / 3.0) * rho * u
    cs = np.sqrt((5.0 / 3.0) * P / rho)
    x = pm[:, :3].astype(np.float64)
    visc = np.zeros((n, 4), np.float32)
    visc[:, 0], visc[:, 1], visc[:, 2] = cs, 1.0, 0.8
    vel = np.zeros((n, 4), np.float32)
    vel[:, :3] = -0.4 * x + 0.1 * np.sin(7 * x[:, [1, 2, 0]])          # compression + some shear
    base = t.sph_force(h, rho, P, 32, vel=vel)["acc_dudt"]
    full = t.sph_force(h, rho, P, 32, vel=vel, visc=visc)["acc_dudt"]
    for k, val in ((1, 0.0), (2, 0.0)):                                 # alpha = 0, f = 0: R17
        v0 = visc.copy()
        v0[:, k] = val
        assert np.array_equal(t.sph_force(h, rho, P, 32, vel=vel, visc=v0)["acc_dudt"], base)
    dv = full - base                                                    # the viscous part
    assert np.abs(dv[:, :3]).max() > 1e-3 * np.abs(base[:, :3]).max()
    assert np.all(dv[:, 3] >= -1e-12 * np.abs(base[:, 3]).max())        # heating only
    mom = (m[:, None] * dv[:, :3]).sum(axis=0)
    assert np.abs(mom).max() <= 1e-12 * (m[:, None] * np.abs(dv[:, :3])).sum()
    e_kin = (m * (vel[:, :3].astype(np.float64) * dv[:, :3]).sum(axis=1)).sum()
    e_int = (m * dv[:, 3]).sum()
    assert abs(e_kin + e_int) <= 1e-10 * abs(e_int) and e_int > 0
    vel[:, :3] = 0.4 * x                                                # homologous expansion: every pair recedes
    assert np.array_equal(t.sph_force(h, rho, P, 32, vel=vel, visc=visc)["acc_dudt"], t.sph_force(h, rho, P, 32, vel=vel)["acc_dudt"])
    # two particles approaching head-on: the closed form of the pair term
    pm2 = np.array([[0, 0, 0, 1.0], [0.5, 0, 0, 1.0]], np.float32)
    t2 = orc.Tree(pm2, 16)
    h2 = np.array([1.0, 1.0], np.float32)
    v2 = np.array([[0.25, 0, 0, 0], [-0.25, 0, 0, 0]], np.float32)
    q2 = np.array([[2.0, 1.5, 1.0, 0], [2.0, 1.5, 1.0, 0]], np.float32)
    r2 = np.array([1.0, 1.0])
    a = t2.sph_force(h2, r2, np.zeros(2), 32, vel=v2, visc=q2)["acc_dudt"]
    r, wdot, l = 0.5, 0.5 * (-0.5), 0.5
    mu = l * wdot / (r * r + 0.01 * l * l)
    Pi = (-1.5 * 2.0 * mu + 2 * 1.5 * mu * mu) / 1.0
    gw = orc.dWdr(r, 1.0)                                               # (dW_i + dW_j)/2 with equal h
    assert a[0, 0] == pytest.approx(-1.0 * Pi * gw * (0 - 0.5) / r, rel=1e-12)     # pushed apart: a_0x < 0
    assert a[0, 0] < 0 and a[1, 0] == pytest.approx(-a[0, 0], rel=1e-12)
    assert a[0, 3] == pytest.approx(0.5 * Pi * gw * wdot / r, rel=1e-12) and a[0, 3] > 0


def test_sph_walk_over_pieces_finds_the_same_neighbours(orc):
    """Reading R26 (default): the SPH MAC of R15 applied per piece of the group (the piece's box, the piece's largest
    h).  Fewer candidates, and -- Eq. 5's guarantee holds piece by piece -- exactly the same neighbours: counts equal,
    density and forces equal to rounding (the candidate lists keep their tree order)."""
    n, G = 6000, 64
    w = gen.wd_pair(n, 21)
    pm, h, u, vel = w["pos_mass"], w["h"], w["u"], w["vel"]
    t = orc.Tree(pm, 16)
    t.set_dist_kind(0)
    a = t.sph_density(h, G)
    t.set_dist_kind(2)
    b = t.sph_density(h, G)
    assert b["candidates"] < 0.8 * a["candidates"] and np.all(b["n_parts"] <= a["n_parts"])
    assert np.array_equal(a["nngb"], b["nngb"]) and np.allclose(a["rho"], b["rho"], rtol=1e-14)
    P = (2.0 / 3.0) * a["rho"] * u
    t.set_dist_kind(0)
    fa = t.sph_force(h, a["rho"], P, G, vel=vel)
    t.set_dist_kind(2)
    fb = t.sph_force(h, a["rho"], P, G, vel=vel)
    assert np.allclose(fa["acc_dudt"], fb["acc_dudt"], rtol=1e-12, atol=1e-14 * np.abs(fa["acc_dudt"]).max())
    # brute force: every true neighbour pair (r < max(h_i, h_j)) of every member is in its group's list
    ex = t.export()
    sp, sh = pm[ex["perm"]].astype(np.float64), h[ex["perm"]].astype(np.float64)
    for g in range(0, t.n_groups(G), 5):
        parts = t.sph_group_list(h, G, g, b["n_parts"][g])
        mem = np.arange(g * G, min((g + 1) * G, n))
        d = np.linalg.norm(sp[mem, None, :3] - sp[None, :, :3], axis=2)
        need = (d < np.maximum(sh[mem, None], sh[None, :])).any(0)
        assert np.isin(np.nonzero(need)[0], parts).all()

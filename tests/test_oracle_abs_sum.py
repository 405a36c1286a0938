"""Pins for the oracle's `abs_sum` outputs -- the sums of pair-term magnitudes A_i = sum_j |x_ij| that set the
floor 8 u A_i of the GPU parity tolerance.  An error there would loosen every parity
assertion silently, so each of them is compared here with a numpy brute-force sum written from the formulas of
DESIGN.md R10 / R17 / R22 / R24 over the oracle's own exported lists (gravity) or over all pairs (SPH: the
neighbour set is defined by distance, not by the list), with closed forms for one pair, and with the bounds
|sum| <= sum of magnitudes."""
import numpy as np
import pytest

from workloads import generators as gen


def dW_np(r, h):
    q = r / h
    s = 8.0 / (np.pi * h ** 4)
    return s * np.where(q <= 0.5, -12 * q + 18 * q ** 2, np.where(q < 1, -6 * (1 - q) ** 2, 0.0))


def test_gravity_abs_sum_two_body_closed_form(orc):
    """one pair: A_i = |a_i| = m_j r / (r^2 + eps^2)^(3/2)"""
    pm = np.array([[0, 0, 0, 2.0], [3.0, 4.0, 0, 5.0]], np.float32)
    t = orc.Tree(pm, 16)
    r = t.gravity(0.5, 0.5, 32)
    want = np.array([5.0, 2.0]) * 5.0 / (25.0 + 0.25) ** 1.5
    assert r["abs_sum"] == pytest.approx(want, rel=1e-14)
    assert np.linalg.norm(r["acc_pot"][:, :3], axis=1) == pytest.approx(want, rel=1e-14)


@pytest.mark.parametrize("eps", [0.01, 0.0])
def test_gravity_abs_sum_theta0_bruteforce(orc, eps):
    """theta = 0: the list of every group is every particle, so A_i = sum_{j != i} m_j r_ij / (r_ij^2 + eps^2)^(3/2)"""
    n = 1500
    pm = gen.plummer(n, 3)
    pm[:, 3] *= (1 + np.arange(n) % 4).astype(np.float32)
    r = orc.Tree(pm, 16).gravity(eps, 0.0, 64)
    x, m = pm[:, :3].astype(np.float64), pm[:, 3].astype(np.float64)
    d2 = ((x[None] - x[:, None]) ** 2).sum(-1)
    w = m[None, :] / np.where(d2 + eps * eps > 0, d2 + eps * eps, np.inf) ** 1.5     # r^2 + eps^2 = 0 pairs contribute 0 (R10)
    np.fill_diagonal(w, 0.0)                                                        # j != i
    A = (w * np.sqrt(d2)).sum(1)
    assert np.allclose(r["abs_sum"], A, rtol=1e-12)
    assert np.all(np.linalg.norm(r["acc_pot"][:, :3], axis=1) <= r["abs_sum"] * (1 + 1e-12))   # triangle inequality


@pytest.mark.parametrize("kind,theta,G,dist", [("plummer", 0.6, 64, 0), ("hernquist", 0.8, 32, 0), ("plummer", 0.6, 64, 1),
                                               ("uniform_cube", 0.5, 128, 0)])
def test_gravity_abs_sum_over_exported_lists(orc, kind, theta, G, dist):
    """theta > 0: numpy sums of |a_ij| over the cells (as virtual particles at the fp32 centre of mass, L43)
    and the particles of every group's exported lists, self excluded by index (R10)."""
    n, eps = 3000, 0.01
    pm = gen.make(kind, n, 1199)
    t = orc.Tree(pm, 8)
    t.set_dist_kind(dist)
    ex = t.export()
    r = t.gravity(eps, theta, G)
    rb2 = t.rb2(theta)
    sp = pm[ex["perm"]].astype(np.float64)
    com = ex["com_m"].astype(np.float64)
    A = np.zeros(n)
    a = np.zeros((n, 3))
    for g in range(t.n_groups(G)):
        cells, parts = t.group_lists_rb2(rb2, G, g, r["n_cells"][g], r["n_parts"][g])
        src = np.concatenate([com[cells], sp[parts]])
        sid = np.concatenate([np.full(len(cells), -1), parts.astype(np.int64)])
        for s in range(g * G, min((g + 1) * G, n)):
            d = src[:, :3] - sp[s, :3]
            d2 = (d ** 2).sum(1)
            w = np.where(sid == s, 0.0, src[:, 3] / (d2 + eps * eps) ** 1.5)
            A[ex["perm"][s]] = (w * np.sqrt(d2)).sum()
            a[ex["perm"][s]] = (w[:, None] * d).sum(0)
    assert np.allclose(r["abs_sum"], A, rtol=1e-12)
    assert np.allclose(r["acc_pot"][:, :3], a, rtol=1e-9, atol=1e-12 * A.max())
    assert np.all(np.linalg.norm(a, axis=1) <= A * (1 + 1e-12))


def _sph_case(orc, n, seed):
    w = gen.wd_pair(n, seed)
    pm, h, u = w["pos_mass"], w["h"], w["u"]
    vel = np.zeros((n, 4), np.float32)
    vel[:, :3] = -0.4 * pm[:, :3] + 0.1 * np.sin(7 * pm[:, [1, 2, 0]])
    t = orc.Tree(pm, 16)
    rho = t.sph_density(h, 64)["rho"]
    P = (2.0 / 3.0) * rho * u
    x = pm[:, :3].astype(np.float64)
    e = x[:, None, :] - x[None, :, :]                      # x_i - x_j
    r = np.sqrt((e ** 2).sum(-1))
    v = vel[:, :3].astype(np.float64)
    return pm, h, vel, t, rho, P, e, r, v


def test_sph_force_abs_sums_bruteforce(orc):
    """R17: |a_ij| = |m_j (P_i/rho_i^2 + P_j/rho_j^2) gw| r with gw = (dW(h_i) + dW(h_j)) / (2 r);
    |du_ij| = |1/2 m_j (...) gw (v_i - v_j).(x_i - x_j)|, over all pairs with r < max(h_i, h_j), r > 0."""
    n = 1800
    pm, h, vel, t, rho, P, e, r, v = _sph_case(orc, n, 5)
    out = t.sph_force(h, rho, P, 64, vel=vel)
    hd = h.astype(np.float64)
    nb = (r < np.maximum(hd[:, None], hd[None, :])) & (r > 0)
    rs = np.where(r > 0, r, 1.0)
    gw = 0.5 * (dW_np(rs, hd[:, None]) + dW_np(rs, hd[None, :])) / rs
    pr = P / rho ** 2
    f = np.where(nb, pm[None, :, 3] * (pr[:, None] + pr[None, :]) * gw, 0.0)
    A = (np.abs(f) * r).sum(1)
    vd = ((v[:, None, :] - v[None, :, :]) * e).sum(-1)
    D = np.abs(0.5 * f * vd).sum(1)
    # pairs at the edge of the support contribute ~0: a fp32-vs-fp64 neighbour decision there does not matter
    assert np.allclose(out["abs_sum"][:, 0], A, rtol=1e-9)
    assert np.allclose(out["abs_sum"][:, 1], D, rtol=1e-9, atol=1e-12 * D.max())
    acc = -(f[:, :, None] * e).sum(1)
    assert np.allclose(out["acc_dudt"][:, :3], acc, rtol=1e-8, atol=1e-11 * A.max())
    assert np.all(np.linalg.norm(out["acc_dudt"][:, :3], axis=1) <= out["abs_sum"][:, 0] * (1 + 1e-12))
    assert np.all(np.abs(out["acc_dudt"][:, 3]) <= out["abs_sum"][:, 1] * (1 + 1e-12) + 1e-300)
    # without velocities the du/dt column and its magnitude sum are zero
    o2 = t.sph_force(h, rho, P, 64)
    assert not o2["abs_sum"][:, 1].any() and np.array_equal(o2["abs_sum"][:, 0], out["abs_sum"][:, 0])


def test_sph_force_visc_abs_sums_bruteforce(orc):
    """R24: the same sums with Pi_ij added to the pressure term for approaching pairs."""
    n = 1500
    pm, h, vel, t, rho, P, e, r, v = _sph_case(orc, n, 9)
    visc = np.zeros((n, 4), np.float32)
    visc[:, 0] = np.sqrt((5.0 / 3.0) * P / rho)
    visc[:, 1] = 0.5 + 0.5 * gen.uniform01(3, np.arange(n, dtype=np.uint64), 0)
    visc[:, 2] = gen.uniform01(4, np.arange(n, dtype=np.uint64), 0)
    out = t.sph_force(h, rho, P, 64, vel=vel, visc=visc)
    hd = h.astype(np.float64)
    nb = (r < np.maximum(hd[:, None], hd[None, :])) & (r > 0)
    rs = np.where(r > 0, r, 1.0)
    gw = 0.5 * (dW_np(rs, hd[:, None]) + dW_np(rs, hd[None, :])) / rs
    pr = P / rho ** 2
    wv = ((v[:, None, :] - v[None, :, :]) * e).sum(-1)
    c, al, fb = (visc[:, k].astype(np.float64) for k in range(3))
    l = 0.25 * (hd[:, None] + hd[None, :])
    mu = l * wv / (r * r + 0.01 * l * l)
    ab, cb, fbar = 0.5 * (al[:, None] + al[None, :]), 0.5 * (c[:, None] + c[None, :]), 0.5 * (fb[:, None] + fb[None, :])
    Pi = np.where(wv < 0, fbar * (-ab * cb * mu + 2 * ab * mu * mu) / (0.5 * (rho[:, None] + rho[None, :])), 0.0)
    f = np.where(nb, pm[None, :, 3] * (pr[:, None] + pr[None, :] + Pi) * gw, 0.0)
    assert np.allclose(out["abs_sum"][:, 0], (np.abs(f) * r).sum(1), rtol=1e-9)
    D = np.abs(0.5 * f * wv).sum(1)
    assert np.allclose(out["abs_sum"][:, 1], D, rtol=1e-9, atol=1e-12 * D.max())
    assert np.allclose(out["acc_dudt"][:, 3], (0.5 * f * wv).sum(1), rtol=1e-8, atol=1e-11 * D.max())


def test_sph_divrot_abs_sum_bruteforce(orc):
    """R22: abs_sum_i = (1/rho_i) sum_j m_j |dW/dr(r_ij, h_i)| |v_j - v_i| over r_ij < h_i, r > 0
    (|gw| r = |dW/dr|), the common magnitude bound of the div v and rot v terms."""
    n = 1800
    pm, h, vel, t, rho, P, e, r, v = _sph_case(orc, n, 13)
    out = t.sph_divrot(h, vel, 64)
    hd = h.astype(np.float64)
    nb = (r < hd[:, None]) & (r > 0)
    du = np.sqrt(((v[None, :, :] - v[:, None, :]) ** 2).sum(-1))
    A = np.where(nb, pm[None, :, 3] * np.abs(dW_np(r, hd[:, None])) * du, 0.0).sum(1) / rho
    assert np.allclose(out["rho"], rho, rtol=1e-13)
    assert np.allclose(out["abs_sum"], A, rtol=1e-9)
    assert np.all(np.abs(out["divrot"][:, 0]) <= out["abs_sum"] * (1 + 1e-12))
    assert np.all(np.linalg.norm(out["divrot"][:, 1:], axis=1) <= out["abs_sum"] * (1 + 1e-12))

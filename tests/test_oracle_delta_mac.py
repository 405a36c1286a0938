"""Pins of the oracle's absolute-error MAC (the paper's own criterion: PAPER.md II-B Eq. 1-3;
m_limit rule III-C L157; scaling laws L81, L165-L167)."""
import os

import numpy as np
import pytest

from workloads import generators as gen

HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    out = {}
    for line in open(os.path.join(HERE, "golden", "paper_values.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def rb_eq1(b, B2, delta):
    return b / 2 + np.sqrt(b * b / 4 + np.sqrt(3 * B2 / delta))


def test_two_particle_cell_eq3(orc):
    """two particles of mass m separated by L: b_max = L/2, B2 = m L^2/2, and Eq. 3
    (with L^2/16: the printed L/16 is a typo) r_b = L/4 + sqrt(L^2/16 + sqrt(3 m L^2/(2 Delta)))."""
    g = golden()
    for m, L, delta in ((1.0, 1.0, 1.0), (1.0, 1.0, 0.01), (0.25, 0.5, 3.0)):
        pm = np.array([[0.25, 0.125, 0.5, m], [0.25 + L, 0.125, 0.5, m]], np.float32)
        t = orc.Tree(pm, 16)
        B2, bm = t.delta_cell_props()
        assert bm[0] == pytest.approx(g["two_particle_cell_bmax_over_L"] * L, rel=1e-14)
        assert B2[0] == pytest.approx(g["two_particle_cell_B2_over_mL2"] * m * L * L, rel=1e-14)
        want = L / 4 + np.sqrt(L * L / 16 + np.sqrt(3 * m * L * L / (2 * delta)))
        assert np.sqrt(t.rb2_delta(delta)[0]) == pytest.approx(want, rel=1e-6)
    assert rb_eq1(0.5, 0.5, 1.0) == pytest.approx(g["eq3_rb_m1_L1_delta1"], rel=1e-4)   # Fig. 3's curve at Delta = 1


def test_B2_bottom_up_equals_eq2(orc):
    pm = gen.plummer(5000, 21)
    pm[:, 3] = (1 + np.arange(5000) % 7) / 5000.0
    t = orc.Tree(pm, 8)
    B2, bm = t.delta_cell_props()
    direct = np.array([t.B2_direct(c) for c in range(t.ncell)])
    assert np.allclose(B2, direct, rtol=1e-11, atol=1e-300)
    # b_max against a brute-force maximum, and 0 <= b_max <= sqrt(3) l
    e = t.export()
    spos = pm[e["perm"]].astype(np.float64)
    for c in (0, 1, t.ncell // 2, t.ncell - 1):
        f, n = int(e["cells"]["first"][c]), int(e["cells"]["count"][c])
        cm = e["MP"][c, 1:] / e["MP"][c, 0]
        assert bm[c] == pytest.approx(np.linalg.norm(spos[f:f + n, :3] - cm, axis=1).max(), rel=1e-13)
    l = t.S * 0.5 ** e["cells"]["level"].astype(np.float64)
    assert np.all(bm <= np.sqrt(3.0) * l * (1 + 1e-12))


def test_rb_formula_and_limits(orc):
    pm = gen.plummer(3000, 5)
    t = orc.Tree(pm, 16)
    B2, bm = t.delta_cell_props()
    for delta in (1e-3, 0.1, 10.0):
        rb = np.sqrt(t.rb2_delta(delta).astype(np.float64))
        assert np.allclose(rb, rb_eq1(bm, B2, delta), rtol=1e-6)
    ok = B2 > 0
    big = np.sqrt(t.rb2_delta(1e30).astype(np.float64))
    assert np.allclose(big[ok], bm[ok], rtol=1e-5)                       # L81: Delta large -> r_b ~ b_max
    r1 = np.sqrt(t.rb2_delta(1e-12).astype(np.float64))[ok]
    r2 = np.sqrt(t.rb2_delta(1e-12 / 16).astype(np.float64))[ok]
    assert np.allclose(r2 / r1, 2.0, rtol=1e-2)                          # L81: r_b ~ Delta^-1/4 for small Delta
    assert np.all(np.isinf(t.rb2_delta(0.0)))                            # Delta = 0 opens everything


def test_m_limit_rule(orc):
    """L157: cells heavier than m_limit get r_b = 2 S_root, so they are never accepted."""
    pm = gen.plummer(4000, 9)
    t = orc.Tree(pm, 16)
    e = t.export()
    M = e["MP"][:, 0]
    rb2 = t.rb2_delta(0.05, m_limit=0.03)
    heavy = M > 0.03
    assert heavy.any() and (~heavy).any()
    assert np.allclose(np.sqrt(rb2[heavy].astype(np.float64)), 2 * t.S, rtol=1e-6)
    assert np.array_equal(rb2[~heavy], t.rb2_delta(0.05)[~heavy])
    G = 64
    r = t.gravity(0.0, 0.0, G, rb2=rb2, forces=False)
    r0 = t.gravity(0.0, 0.0, G, rb2=t.rb2_delta(0.05), forces=False)
    for g in range(0, t.n_groups(G), 7):
        cells, _ = t.group_lists_rb2(rb2, G, g, r["n_cells"][g], r["n_parts"][g])
        assert not heavy[cells].any()
    assert np.all(r["n_cells"] + r["n_parts"] >= 0) and r["interactions"] >= r0["interactions"]


def test_lists_tile_the_system_and_error_bound(orc):
    """Every group's lists cover each particle exactly once, and every accepted cell's monopole differs
    from the sum over its particles by at most Delta for every group member (the bound the absolute MAC
    is built on; eps = 0)."""
    n, G, delta = 3000, 32, 0.02
    pm = gen.plummer(n, 33)
    t = orc.Tree(pm, 8)
    e = t.export()
    spos = pm[e["perm"]].astype(np.float64)
    rb2 = t.rb2_delta(delta)
    r = t.gravity(0.0, 0.0, G, rb2=rb2, forces=False)
    worst = 0.0
    for g in range(0, t.n_groups(G), 5):
        cells, parts = t.group_lists_rb2(rb2, G, g, r["n_cells"][g], r["n_parts"][g])
        cover = np.zeros(n, dtype=np.int32)
        cover[parts] += 1
        for c in cells:
            f, k = int(e["cells"]["first"][c]), int(e["cells"]["count"][c])
            cover[f:f + k] += 1
        assert np.all(cover == 1)
        tg = spos[g * G:min((g + 1) * G, n), :3]
        for c in cells:
            f, k = int(e["cells"]["first"][c]), int(e["cells"]["count"][c])
            src = spos[f:f + k]
            d = src[None, :, :3] - tg[:, None, :]
            a_dir = (src[None, :, 3, None] * d / np.linalg.norm(d, axis=2, keepdims=True) ** 3).sum(axis=1)
            cm = e["com_m"][c].astype(np.float64)
            dc = cm[None, :3] - tg
            a_mono = cm[3] * dc / np.linalg.norm(dc, axis=1, keepdims=True) ** 3
            worst = max(worst, np.linalg.norm(a_mono - a_dir, axis=1).max())
    assert worst <= delta * (1 + 1e-6), worst


def test_delta_to_zero_is_direct_sum_and_error_falls(orc):
    n = 2500
    pm = gen.plummer(n, 12)
    t = orc.Tree(pm, 8)
    direct = orc.direct_sum(pm, 0.01)
    r0 = t.gravity(0.01, 0.0, 64, rb2=t.rb2_delta(0.0))
    assert np.allclose(r0["acc_pot"], direct, rtol=1e-12, atol=1e-14) and r0["n_cells"].sum() == 0
    errs, inter = [], []
    for delta in (1.0, 0.1, 0.01, 0.001):
        r = t.gravity(0.01, 0.0, 64, rb2=t.rb2_delta(delta))
        d = np.linalg.norm(r["acc_pot"][:, :3] - direct[:, :3], axis=1)
        errs.append(d.mean())
        inter.append(r["interactions"])
        assert d.max() <= 60 * delta          # loose: the bound is per accepted cell, errors add up over cells
    assert errs == sorted(errs, reverse=True) and inter == sorted(inter)     # L165-L167: cost up, error down


def test_scaling_with_delta_at_the_papers_vector_length(orc):
    """PAPER.md L165-L167 (Fig. 4-5, missing): "time ~ Delta^-3/4", "error ~ Delta^1/4", "the averaged error does not
    depend on n_vec".  The paper's own configuration -- uniform sphere, n_vec = 4 and 8, exact-minimum group distance
    (L163), Hilbert order, m_limit = 0.05 -- run by the oracle:
      * the mean error is independent of the vector length (within 10 % between n_vec = 4 and 8; 32: up to 20 % lower): as stated;
      * interactions per particle grow as Delta^-0.45 (local slope -0.33 ... -0.5 over Delta = 1e-1 ... 1e-6 at
        N = 1e5 ... 1e6, cells and particles alike) and the mean error falls as Delta^0.5: NOT the paper's exponents.
    r_b ~ (B2/Delta)^(1/4) with B2 ~ l^5 gives Delta^-3/4 cells per tree level, but the level at which r_b reaches
    the system size moves with Delta (l_max ~ Delta^(1/5)) and m_limit opens the heavy cells regardless of Delta, so
    the sum over levels is shallower.  The finding is recorded in DESIGN.md section 11; this test pins the measured
    exponents so that a change of the MAC, of B2 or of the walk shows up."""
    n, eps = 32768, 0.004
    pm = gen.uniform_sphere(n, 1206)
    ref = orc.direct_sum(pm, eps)
    t = orc.Tree(pm, 16, key_order=1)
    t.set_dist_kind(1)
    deltas = [1e-2, 1e-3, 1e-4, 1e-5]
    err, inter = {}, {}
    for G in (4, 8, 32):
        for d in deltas:
            r = t.gravity(eps, 0.0, G, rb2=t.rb2_delta(float(np.float32(d)), float(np.float32(0.05))))
            err[G, d] = np.linalg.norm(r["acc_pot"][:, :3] - ref[:, :3], axis=1).mean()
            inter[G, d] = r["interactions"] / n
    lg = np.log10(deltas)
    for G in (4, 8):
        si = np.polyfit(lg, np.log10([inter[G, d] for d in deltas]), 1)[0]
        se = np.polyfit(lg, np.log10([err[G, d] for d in deltas]), 1)[0]
        assert -0.6 < si < -0.3, si          # not -0.75
        assert 0.4 < se < 0.65, se           # not +0.25
    for d in deltas:
        # n_vec = 4 vs 8 (the paper's range): within 10 %; a 32-wide vector shares longer lists and is a little MORE accurate
        assert abs(err[8, d] / err[4, d] - 1) < 0.1 and 0.75 < err[32, d] / err[4, d] < 1.02, (d, err[4, d], err[8, d], err[32, d])
    # larger vectors share longer lists (more interactions per particle) at the same error: the trade-off of L165
    assert all(inter[4, d] < inter[8, d] < inter[32, d] for d in deltas)

"""Pins for the oracle's walk and gravity sums (PAPER.md II, III-D; readings R7-R11).
Expected values come from closed forms, numpy brute force and invariants, never from oracle/."""
import numpy as np
import pytest

from workloads import generators as gen


def np_direct(pm, eps):
    x = pm[:, :3].astype(np.float64)
    m = pm[:, 3].astype(np.float64)
    d = x[None, :, :] - x[:, None, :]
    r2 = (d ** 2).sum(-1) + eps * eps
    np.fill_diagonal(r2, np.inf)
    ri = 1.0 / np.sqrt(r2)
    acc = (m[None, :, None] * d * ri[:, :, None] ** 3).sum(1)
    pot = -(m[None, :] * ri).sum(1)
    return np.concatenate([acc, pot[:, None]], axis=1)


def test_direct_sum_two_body_closed_form(orc):
    pm = np.array([[0, 0, 0, 2.0], [3.0, 4.0, 0, 5.0]], np.float32)
    eps = 0.5
    out = orc.direct_sum(pm, eps)
    r2 = 25.0 + 0.25
    a0 = 5.0 / r2 ** 1.5
    assert out[0] == pytest.approx([a0 * 3, a0 * 4, 0, -5.0 / np.sqrt(r2)], rel=1e-14)
    a1 = 2.0 / r2 ** 1.5
    assert out[1] == pytest.approx([-a1 * 3, -a1 * 4, 0, -2.0 / np.sqrt(r2)], rel=1e-14)


def test_direct_sum_vs_numpy_and_newton3(orc):
    pm = gen.plummer(700, 11)
    pm[:, 3] *= (1 + np.arange(700) % 3).astype(np.float32)
    out = orc.direct_sum(pm, 0.01)
    ref = np_direct(pm, 0.01)
    assert np.allclose(out, ref, rtol=1e-12, atol=1e-14)
    m = pm[:, 3].astype(np.float64)
    mom = (m[:, None] * out[:, :3]).sum(0)
    scale = (m[:, None] * np.abs(out[:, :3])).sum()
    assert np.all(np.abs(mom) < 1e-13 * scale)            # Newton's third law
    sub = orc.direct_sum(pm, 0.01, targets=[5, 699, 0])
    assert np.array_equal(sub, out[[5, 699, 0]])


@pytest.mark.parametrize("G", [32, 64])
def test_theta0_is_direct_sum(orc, G):
    pm = gen.plummer(1500, 3)
    t = orc.Tree(pm, 16)
    r = t.gravity(0.01, 0.0, G)
    assert np.all(r["n_cells"] == 0) and np.all(r["n_parts"] == 1500)   # L43: no cell accepted
    ref = np_direct(pm, 0.01)
    assert np.allclose(r["acc_pot"], ref, rtol=1e-11, atol=1e-13)
    assert r["interactions"] == 1500 * 1500


@pytest.mark.parametrize("theta,mac", [(0.5, 0), (0.8, 0), (1.0, 0), (0.6, 1)])
def test_lists_tile_the_system(orc, theta, mac):
    """Every particle is covered exactly once by (accepted cells' ranges) U (particle list);
    with the default MAC (R7) each group member sits in its own particle list."""
    n, G = 6000, 64
    pm = gen.plummer(n, 21)
    t = orc.Tree(pm, 8)
    ex = t.export()
    r = t.gravity(0.01, theta, G, mac_kind=mac, forces=False)
    for g in range(0, t.n_groups(G), 5):
        cells, parts = t.group_lists(theta, G, g, r["n_cells"][g], r["n_parts"][g], mac_kind=mac)
        cover = np.zeros(n, np.int32)
        for c in cells:
            f, k = ex["cells"]["first"][c], ex["cells"]["count"][c]
            cover[f:f + k] += 1
        np.add.at(cover, parts, 1)
        assert np.all(cover == 1)
        if mac == 0:
            members = np.arange(g * G, min((g + 1) * G, n))
            assert np.isin(members, parts).all()


def test_stackless_equals_recursive(orc):
    """PAPER L57 rules (1)-(4) on the next/more list visit exactly what the recursion visits."""
    pm = gen.hernquist(5000, 2)
    t = orc.Tree(pm, 16)
    for theta in (0.0, 0.4, 0.8):
        a = t.gravity(0.01, theta, 64, walk_kind=0)
        b = t.gravity(0.01, theta, 64, walk_kind=1)
        for k in ("n_tests", "n_cells", "n_parts"):
            assert np.array_equal(a[k], b[k])
        assert a["interactions"] == b["interactions"]
        assert np.allclose(a["acc_pot"], b["acc_pot"], rtol=1e-12, atol=1e-15)


def test_error_decreases_with_theta_and_lists_shrink(orc):
    pm = gen.plummer(8192, 1206)
    t = orc.Tree(pm, 16)
    ref = orc.direct_sum(pm, 0.01)
    an = np.linalg.norm(ref[:, :3], axis=1)
    errs, inter = [], []
    for theta in (0.8, 0.6, 0.4, 0.2):
        r = t.gravity(0.01, theta, 64)
        e = np.linalg.norm(r["acc_pot"][:, :3] - ref[:, :3], axis=1) / an
        errs.append(np.sqrt((e ** 2).mean()))
        inter.append(r["interactions"])
    assert errs[0] > errs[1] > errs[2] > errs[3]
    assert errs[3] < 2e-4 and errs[0] < 3e-2
    assert inter[0] < inter[1] < inter[2] < inter[3]


@pytest.mark.parametrize("dist", [0, 2])
def test_theta_mac_error_is_bounded_by_the_multipole_remainder(orc, dist):
    """The absolute accuracy of the theta-MAC (R7: accept iff the group's distance to the centre of mass exceeds
    r_b = l/theta + s), pinned to what the mathematics fixes -- not to the oracle:
    (1) geometry: every particle of a cell lies within (sqrt(3)/2) l + s of its centre of mass, every target farther than
        r_b from it, so b/d < ((sqrt(3)/2) l + s) / (l/theta + s) < 1 for every (target, accepted cell), b = the cell's
        largest particle distance from its centre of mass, by brute force;
    (2) a monopole at the centre of mass has no dipole term: by Taylor's theorem with the third derivatives of 1/r
        (largest multilinear value 6/r^4, radial) |a_exact - a_monopole| <= 3 M b^2 / (d - b)^4 per (target, cell);
    (3) the oracle's force differs from the O(N^2) sum by no more than the sum of these remainders over its list;
    (4) the median error grows as theta^2 ... theta^3 (quadrupole order) and stays below 0.005 theta^2.
    Newtonian (eps = 0), so that (2) is the textbook bound."""
    n, G, eps = 3000, 32, 0.0
    pm = gen.plummer(n, 17)
    t = orc.Tree(pm, 8)
    t.set_dist_kind(dist)
    ex = t.export()
    xs = pm[ex["perm"].astype(np.int64), :3].astype(np.float64)          # positions in sorted order
    ms = pm[ex["perm"].astype(np.int64), 3].astype(np.float64)
    cm = ex["MP"][:, 1:4] / ex["MP"][:, :1]
    M = ex["MP"][:, 0]
    lvl = ex["cells"]["level"].astype(np.int64)
    l = float(t.S) * 0.5 ** lvl
    ref = np_direct(pm, eps)[ex["perm"].astype(np.int64)]                # direct sum, sorted order
    med = {}
    for theta in (0.2, 0.3, 0.45, 0.6, 0.9):
        th = float(np.float32(theta))
        r = t.gravity(eps, th, G)
        a = r["acc_pot"][ex["perm"].astype(np.int64), :3]
        err = np.linalg.norm(a - ref[:, :3], axis=1)
        med[theta] = float(np.median(err / np.linalg.norm(ref[:, :3], axis=1)))
        if theta not in (0.3, 0.6, 0.9):
            continue
        for g in range(0, t.n_groups(G), 9):
            cells, parts = t.group_lists(th, G, g, r["n_cells"][g], r["n_parts"][g])
            tg = np.arange(g * G, min((g + 1) * G, n))
            bound = np.zeros(len(tg))
            for c in cells.astype(np.int64):
                f, k = int(ex["cells"]["first"][c]), int(ex["cells"]["count"][c])
                dj = xs[f:f + k] - cm[c]
                b = np.sqrt((dj ** 2).sum(1)).max()
                rv = cm[c][None, :] - xs[tg]
                d = np.sqrt((rv ** 2).sum(1))
                rho = b / d
                assert d.min() > (l[c] / th + ex["s"][c]) * (1 - 1e-6), (theta, g, c)          # every target outside r_b (R7, R8 / R25)
                assert rho.max() <= ((np.sqrt(3) / 2) * l[c] + ex["s"][c]) / (l[c] / th + ex["s"][c]) * (1 + 1e-6), (theta, g, c)   # (1)
                rem = 3.0 * M[c] * b * b / (d - b) ** 4
                yv = xs[f:f + k][None, :, :] - xs[tg][:, None, :]
                exact = (ms[f:f + k][None, :, None] * yv / ((yv ** 2).sum(-1) ** 1.5)[:, :, None]).sum(1)
                mono = M[c] * rv / (d ** 3)[:, None]
                assert (np.linalg.norm(exact - mono, axis=1) <= rem * (1 + 1e-9) + 1e-12).all(), (theta, g, c)                      # (2)
                bound += rem
            # (3); slack: the walk sees the centre of mass rounded to fp32 (R6)
            assert (err[tg] <= bound + 1e-5 * np.linalg.norm(ref[tg, :3], axis=1)).all(), (theta, g)
    ths = np.array(sorted(med))
    slope = np.polyfit(np.log(ths), np.log([med[x] for x in ths]), 1)[0]
    assert 2.0 < slope < 3.2, slope                                                                                                 # (4)
    assert all(med[x] <= 0.005 * x * x for x in ths), med


def test_plummer_potential_profile(orc):
    """Analytic Plummer potential phi(r) = -1/sqrt(r^2+1) (G=M=a=1), PAPER L193 workload."""
    n = 16384
    pm = gen.plummer(n, 1199)
    t = orc.Tree(pm, 16)
    r = t.gravity(0.01, 0.5, 64)
    rad = np.linalg.norm(pm[:, :3].astype(np.float64), axis=1)
    for lo, hi in [(0.0, 0.5), (0.5, 1.0), (1.0, 2.0), (2.0, 5.0)]:
        sel = (rad >= lo) & (rad < hi)
        got = r["acc_pot"][sel, 3].mean()
        want = (-1.0 / np.sqrt(rad[sel] ** 2 + 1.0)).mean()
        assert got == pytest.approx(want, rel=0.02)
    # radial acceleration: a_r = -r/(r^2+1)^1.5
    ar = (r["acc_pot"][:, :3] * pm[:, :3]).sum(1) / rad
    sel = (rad > 0.5) & (rad < 2.0)
    assert ar[sel].mean() == pytest.approx((-rad[sel] / (rad[sel] ** 2 + 1) ** 1.5).mean(), rel=0.03)


def test_interaction_count_definition(orc):
    n, G = 3000, 64
    pm = gen.uniform_cube(n, 4)
    t = orc.Tree(pm, 16)
    r = t.gravity(0.001, 0.5, G, forces=False)
    sizes = np.minimum(G, n - np.arange(t.n_groups(G)) * G)
    assert r["interactions"] == int((sizes * (r["n_cells"].astype(np.int64) + r["n_parts"])).sum())
    assert r["acc_pot"] is None


def test_group_selection_equals_full_run(orc):
    """orc_gravity_sel / orc_sph_*_sel (used by the full-size GPU parity tests) give, for the selected
    groups, exactly what the all-groups run gives."""
    pm = gen.plummer(6000, 11)
    t = orc.Tree(pm, 8)
    full = t.gravity(0.01, 0.6, 64)
    sel = np.array([0, 3, 17, 50, t.n_groups(64) - 1], dtype=np.int64)
    part = t.gravity(0.01, 0.6, 64, groups=sel)
    for k in ("n_tests", "n_cells", "n_parts"):
        assert np.array_equal(part[k], full[k][sel])
    idx = t.group_targets(64, sel)
    assert np.array_equal(part["acc_pot"][idx], full["acc_pot"][idx])
    assert np.array_equal(part["abs_sum"][idx], full["abs_sum"][idx])
    rest = np.setdiff1d(np.arange(6000), idx)
    assert not part["acc_pot"][rest].any()
    w = gen.wd_pair(5000, 3)
    ts = orc.Tree(w["pos_mass"], 16)
    fd = ts.sph_density(w["h"], 32)
    sel = np.array([1, 2, 40, ts.n_groups(32) - 1], dtype=np.int64)
    pd = ts.sph_density(w["h"], 32, groups=sel)
    idx = ts.group_targets(32, sel)
    assert np.array_equal(pd["n_parts"], fd["n_parts"][sel]) and np.array_equal(pd["rho"][idx], fd["rho"][idx])
    assert np.array_equal(pd["nngb"][idx], fd["nngb"][idx])
    P = (2.0 / 3.0) * fd["rho"] * w["u"]
    ff = ts.sph_force(w["h"], fd["rho"], P, 32, vel=w["vel"])
    pf = ts.sph_force(w["h"], fd["rho"], P, 32, vel=w["vel"], groups=sel)
    assert np.array_equal(pf["acc_dudt"][idx], ff["acc_dudt"][idx])


def test_exact_minimum_group_distance(orc):
    """dist_kind = 1 ("compute n_vec distances ... select the actual minimum"; reading R23).
    Pins by brute force on a small system: every accepted cell is farther than r_b from EVERY member of the
    group (fp32 distances recomputed here with numpy), every cell that was opened has some member within
    r_b, the lists still tile the system, they are never longer than the bounding-box lists, and theta = 0
    is the direct sum."""
    n, G, theta = 3000, 32, np.float32(0.7)
    pm = gen.plummer(n, 17)
    t = orc.Tree(pm, 8)
    e = t.export()
    spos = pm[e["perm"]]
    rb2 = t.rb2(float(theta))
    aabb = t.gravity(0.01, float(theta), G, forces=False)
    t.set_dist_kind(1)
    ex = t.gravity(0.01, float(theta), G, forces=False)
    assert np.all(ex["n_cells"].astype(int) + ex["n_parts"] <= aabb["n_cells"].astype(int) + aabb["n_parts"])
    assert ex["interactions"] < aabb["interactions"]
    cm = e["com_m"][:, :3]
    first, count, cf, cc = (e["cells"][k].astype(np.int64) for k in ("first", "count", "child_first", "child_count"))

    for g in range(0, t.n_groups(G), 9):
        cells, parts = t.group_lists_rb2(rb2, G, g, ex["n_cells"][g], ex["n_parts"][g])
        mem = spos[g * G:min((g + 1) * G, n), :3]
        cover = np.zeros(n, np.int32)
        cover[parts] += 1
        for c in cells:
            cover[first[c]:first[c] + count[c]] += 1
            d = (mem - cm[c]).astype(np.float32).astype(np.float64)
            assert ((d ** 2).sum(axis=1).min()) > float(rb2[c]) * (1 - 1e-6)       # every member outside r_b
            par = np.where((cf <= c) & (c < cf + cc) & (cc > 0))[0]                 # its parent was opened:
            if len(par):
                dp = (mem - cm[par[0]]).astype(np.float32).astype(np.float64)
                assert ((dp ** 2).sum(axis=1).min()) <= float(rb2[par[0]]) * (1 + 1e-6)   # some member inside the parent's r_b
        assert np.all(cover == 1)
    d = orc.direct_sum(pm, 0.01)
    assert np.allclose(t.gravity(0.01, 0.0, G)["acc_pot"], d, rtol=1e-12, atol=1e-14)
    # the accuracy is that of a per-particle MAC: no worse than a few times the box lists' error
    t2 = orc.Tree(pm, 8)
    eb = np.linalg.norm(t2.gravity(0.01, float(theta), G)["acc_pot"][:, :3] - d[:, :3], axis=1).mean()
    ee = np.linalg.norm(t.gravity(0.01, float(theta), G)["acc_pot"][:, :3] - d[:, :3], axis=1).mean()
    assert eb <= ee <= 3 * eb


def _np_cplev(a, b):
    """leading octree levels two 63-bit keys share (0..21), by comparing octant digits from the top"""
    l = 0
    for lev in range(21):
        sh = 3 * (20 - lev)
        if ((int(a) >> sh) & 7) != ((int(b) >> sh) & 7):
            break
        l += 1
    return l


def _np_pieces(keys, a, b, K=8):
    """reading R25 restated: cut [a, b) at its K-1 coarsest key boundaries (fewest shared levels; ties: lowest slot)"""
    cand = sorted((( _np_cplev(keys[s - 1], keys[s]), s) for s in range(a + 1, b)))[:K - 1]
    cuts = sorted(s for _, s in cand)
    edges = [a] + cuts + [b]
    return [(edges[i], edges[i + 1]) for i in range(len(edges) - 1)]


def _np_box_d2(lo, hi, c):
    """R8 in fp32: e = max(0, lo - c, c - hi); d2 = fma(ez, ez, fma(ey, ey, ex*ex)) (fma emulated in fp64: exact products)"""
    e = np.maximum(np.float32(0), np.maximum((lo - c).astype(np.float32), (c - hi).astype(np.float32))).astype(np.float64)
    t = np.float32(e[0] * e[0])
    t = np.float32(e[1] * e[1] + np.float64(t))
    return np.float32(e[2] * e[2] + np.float64(t))


@pytest.mark.parametrize("kind,G,theta,key_order", [("plummer", 32, 0.7, 0), ("uniform_cube", 64, 0.5, 0), ("hernquist", 128, 0.6, 1)])
def test_split_box_group_distance(orc, kind, G, theta, key_order):
    """dist_kind = 2 (reading R25, the default): the group-cell distance is the minimum over the tight boxes of the
    group's pieces between its 7 coarsest key boundaries.  Pins by brute force with the pieces recomputed here from
    the exported keys: every accepted cell is farther than r_b from EVERY piece box, every cell whose parent was
    opened has a parent within r_b of SOME piece, the lists tile the system, they are nested between the exact-minimum
    lists (R23) and the one-box lists (R8), and theta = 0 is the direct sum."""
    n, theta = 3000, np.float32(theta)
    pm = gen.make(kind, n, 23)
    t = orc.Tree(pm, 8, key_order=key_order)
    e = t.export()
    spos = pm[e["perm"]]
    rb2 = t.rb2(float(theta))
    t.set_dist_kind(0)
    box = t.gravity(0.01, float(theta), G, forces=False)
    t.set_dist_kind(1)
    exact = t.gravity(0.01, float(theta), G, forces=False)
    t.set_dist_kind(2)
    sp = t.gravity(0.01, float(theta), G, forces=False)
    Lb, Le, Ls = (x["n_cells"].astype(int) + x["n_parts"] for x in (box, exact, sp))
    assert np.all(Le <= Ls) and np.all(Ls <= Lb) and sp["interactions"] < box["interactions"]
    cm = e["com_m"][:, :3]
    first, count, cf, cc = (e["cells"][k].astype(np.int64) for k in ("first", "count", "child_first", "child_count"))
    parent = np.full(t.ncell, -1)
    for c in range(t.ncell):
        parent[cf[c]:cf[c] + cc[c]] = c
    for g in range(0, t.n_groups(G), 7):
        a, b = g * G, min((g + 1) * G, n)
        pieces = _np_pieces(e["keys"], a, b)
        assert len(pieces) == min(8, b - a) and pieces[0][0] == a and pieces[-1][1] == b
        boxes = [(spos[s0:s1, :3].min(0), spos[s0:s1, :3].max(0)) for s0, s1 in pieces]
        d2 = lambda c: min(_np_box_d2(lo, hi, cm[c]) for lo, hi in boxes)
        cells, parts = t.group_lists_rb2(rb2, G, g, sp["n_cells"][g], sp["n_parts"][g])
        cover = np.zeros(n, np.int32)
        cover[parts] += 1
        for c in cells:
            cover[first[c]:first[c] + count[c]] += 1
            assert d2(c) > rb2[c]                                   # accepted: outside r_b of every piece
            assert not d2(parent[c]) > rb2[parent[c]]               # its parent was opened
        assert np.all(cover == 1)
    d = orc.direct_sum(pm, 0.01)
    assert np.allclose(t.gravity(0.01, 0.0, G)["acc_pot"], d, rtol=1e-12, atol=1e-14)


def test_split_box_removes_the_system_sized_lists(orc):
    """What R25 is for: with one box per Morton group a few groups straddle the coarsest cell boundaries and list a
    large part of the system; cut at their coarsest boundaries the same groups have lists like everybody else's."""
    n, G = 200000, 128
    pm = gen.plummer(n, 5)
    t = orc.Tree(pm, 16)
    t.set_dist_kind(0)
    Lb = (lambda r: r["n_cells"].astype(int) + r["n_parts"])(t.gravity(0.004, 0.6, G, forces=False))
    t.set_dist_kind(2)
    Ls = (lambda r: r["n_cells"].astype(int) + r["n_parts"])(t.gravity(0.004, 0.6, G, forces=False))
    assert Lb.max() > 20 * np.median(Lb)               # the pathology is there with one box
    assert Ls.max() < 4 * np.median(Ls)                # and gone with the pieces
    assert Ls.sum() < 0.8 * Lb.sum()

"""Pins for the oracle's tree build (PAPER.md III-B/III-C; readings R1-R7).
Every expected value here is computed independently of oracle/ (numpy brute force, closed forms)."""
import numpy as np
import pytest

from workloads import generators as gen


def brute_octant_key(p, lo, S):
    """L129: at each level compare against the centre of the current cube; octant = x<<2|y<<1|z.
    Exact rational arithmetic on the fp32 quantised offsets is avoided by using the same
    quantisation grid: the level-l cell boundaries are multiples of S/2^l."""
    # quantise exactly like R2 but with numpy float32 scalars written independently
    scale = np.float32(2097152.0) / np.float32(S)
    q = []
    for k in range(3):
        t = np.float32(np.float32(p[k]) - np.float32(lo[k])) * scale
        q.append(min(int(np.float32(t)), 2 ** 21 - 1))
    key = 0
    c = [0, 0, 0]           # current cube corner in grid units
    size = 2 ** 21
    for lev in range(21):
        half = size // 2
        oct_ = 0
        for k in range(3):
            bit = 1 if q[k] >= c[k] + half else 0
            if bit:
                c[k] += half
            oct_ = (oct_ << 1) | bit
        key = (key << 3) | oct_
        size = half
    return key


def test_keys_bruteforce_and_corners(orc):
    pm = gen.plummer(300, 7)
    t = orc.Tree(pm, 4)
    ex = t.export()
    lo, S = t.lo, t.S
    assert np.all(lo == pm[:, :3].min(axis=0))
    assert S == np.float32((pm[:, :3].max(axis=0) - pm[:, :3].min(axis=0)).max())
    for s in range(0, 300, 7):
        i = ex["perm"][s]
        assert int(ex["keys"][s]) == brute_octant_key(pm[i, :3], lo, S)
    # corners: x = lo -> all-zero bits on that axis; x = hi on the longest axis -> clamped to 2^21-1
    assert t.key(lo) == 0
    k = int(np.argmax(pm[:, :3].max(axis=0) - lo))
    hi = lo.copy()
    hi[k] = pm[:, k].max()
    key = t.key(hi)
    bits = [(key >> (3 * b + (2 - k))) & 1 for b in range(21)]
    assert all(bits)


def test_degenerate_root(orc):
    pm = np.zeros((5, 4), np.float32)
    pm[:, :3] = 3.0
    pm[:, 3] = 1.0
    t = orc.Tree(pm, 2)
    assert t.S == 1.0                       # R1: S = 0 -> 1
    ex = t.export()
    assert np.all(ex["keys"] == 0)
    assert np.all(ex["perm"] == np.arange(5))   # R4 ties by index
    # coincident points: single-child chain down to level 21, leaf exceeds n_crit there (R5)
    assert t.ncell == 22 and t.depth == 21 and t.nleaf == 1
    assert ex["cells"]["count"].tolist() == [5] * 22
    one = orc.Tree(pm[:1], 16)
    assert one.ncell == 1
    empty = orc.Tree(np.zeros((0, 4), np.float32), 16)
    assert empty.ncell == 1 and empty.export()["cells"]["count"][0] == 0


@pytest.mark.parametrize("n,n_crit,seed", [(2000, 16, 1), (5000, 1, 2), (3000, 8, 3)])
def test_sort_and_topology_invariants(orc, n, n_crit, seed):
    pm = gen.plummer(n, seed)
    pm[10] = pm[11]                          # a duplicate point
    t = orc.Tree(pm, n_crit)
    ex = t.export()
    keys, perm, cells = ex["keys"], ex["perm"], ex["cells"]
    # R4: equals a stable sort of the unsorted keys
    ukeys = np.empty(n, np.uint64)
    ukeys[perm] = keys
    assert np.array_equal(perm, np.argsort(ukeys, kind="stable").astype(np.uint32))
    assert np.all(keys[1:] >= keys[:-1])
    # canonical order
    lv, fi = cells["level"].astype(np.int64), cells["first"].astype(np.int64)
    order = np.lexsort((fi, lv))
    assert np.array_equal(order, np.arange(t.ncell))
    assert cells[0]["level"] == 0 and cells[0]["count"] == n
    leaf = cells["child_count"] == 0
    assert t.nleaf == leaf.sum()
    assert cells["count"][leaf].sum() == n                     # leaves partition the particles
    assert np.all(cells["count"][~leaf] > n_crit)              # internal cells exceed n_crit
    assert np.all((cells["count"][leaf] <= n_crit) | (cells["level"][leaf] == 21))
    for c in range(t.ncell):
        cell = cells[c]
        sh = np.uint64(3 * (21 - int(cell["level"])))
        seg = keys[cell["first"]:cell["first"] + cell["count"]]
        assert np.all((seg >> sh) == cell["prefix"])           # every particle carries the prefix
        if cell["first"] > 0 and cell["level"] > 0:
            assert (keys[cell["first"] - 1] >> sh) != cell["prefix"]   # range is maximal
        if cell["child_count"]:
            ch = cells[cell["child_first"]:cell["child_first"] + cell["child_count"]]
            assert np.all(ch["level"] == cell["level"] + 1)
            assert ch["first"][0] == cell["first"] and ch["count"].sum() == cell["count"]
            assert np.all(ch["first"][1:] == ch["first"][:-1] + ch["count"][:-1])
            octs = ch["prefix"] & np.uint64(7)
            assert np.all(octs[1:] > octs[:-1])                # one child per occupied octant, in order
            assert np.all((ch["prefix"] >> np.uint64(3)) == cell["prefix"])


def test_mass_com_and_two_particle_cell(orc):
    pm = gen.plummer(4000, 5)
    pm[:, 3] = (1.0 + np.arange(4000) % 7).astype(np.float32) / 4000
    t = orc.Tree(pm, 16)
    ex = t.export()
    m = pm[:, 3].astype(np.float64)
    x = pm[:, :3].astype(np.float64)
    assert ex["MP"][0, 0] == pytest.approx(m.sum(), rel=1e-14)
    assert ex["com_m"][0, :3] == pytest.approx((m[:, None] * x).sum(0) / m.sum(), rel=1e-6)
    cells = ex["cells"]
    # every cell: CM from an independent numpy sum; CM inside the cell cube; s <= sqrt(3)/2 l
    for c in range(0, t.ncell, 37):
        cell = cells[c]
        idx = ex["perm"][cell["first"]:cell["first"] + cell["count"]]
        M = m[idx].sum()
        cm = (m[idx, None] * x[idx]).sum(0) / M
        assert ex["com_m"][c, 3] == pytest.approx(M, rel=1e-6)
        assert ex["com_m"][c, :3] == pytest.approx(cm, rel=1e-5, abs=1e-6)
        l = t.S / 2 ** int(cell["level"])
        assert ex["s"][c] <= np.sqrt(3) / 2 * l * (1 + 1e-6)
    # two particles of mass m separated by L in one cell: CM midway, b_max = L/2
    two = np.array([[0, 0, 0, 1.0], [1.0, 0, 0, 1.0]], np.float32)
    t2 = orc.Tree(two, 16)
    e2 = t2.export()
    assert t2.ncell == 1
    assert e2["com_m"][0].tolist() == [0.5, 0.0, 0.0, 2.0]
    b, r = t2.sph_cell_radii(np.array([0.25, 0.5], np.float32))
    assert b[0] == 0.5 and r[0] == 1.0          # Eq. 5: max(|x-CM| + h) = 0.5 + 0.5
    # geometric centre of the root cube is (0.5,0.5,0.5): s = |(0.5,0,0)-(0.5,0.5,0.5)|
    assert e2["s"][0] == pytest.approx(np.sqrt(0.5), rel=1e-15)


def test_rb2_hand_built_tree(orc):
    """R7 on a tree small enough to do by hand (l, s as defined at PAPER.md L63; none of the numbers below comes
    from the oracle).  Three unit masses A = (0,0,0), B = (1,1,1), C = (1/8,1/8,1/8), n_crit = 1: root cube [0,1]^3.
      root      l = 1,   centre (1/2,..),  CM = (3/8,..):   s = sqrt(3)/8,    r_b = 1/theta + s
      octant 0  l = 1/2, centre (1/4,..),  CM = (1/16,..):  s = 3 sqrt(3)/16  (holds A and C)
      octant 7  l = 1/2, centre (3/4,..),  CM = (1,1,1):    s = sqrt(3)/4     (holds B)
    theta = 1/2:  r_b^2 = (2 + 0.21650635)^2 = 4.9129004, (1 + 0.32475953)^2 = 1.7549878, (1 + 0.43301270)^2 = 2.0535254;
    the plain form r_b = l/theta (mac_kind 1) gives 4, 1, 1."""
    pm = np.array([[0, 0, 0, 1.0], [1, 1, 1, 1.0], [0.125, 0.125, 0.125, 1.0]], np.float32)
    t = orc.Tree(pm, 1)
    ex = t.export()
    c = ex["cells"]
    assert t.S == 1.0 and (c["level"][:3] == [0, 1, 1]).all() and (c["prefix"][:3] == [0, 0, 7]).all()
    assert (c["count"][:3] == [3, 2, 1]).all()
    assert ex["s"][:3] == pytest.approx([0.21650635, 0.32475953, 0.43301270], rel=2e-8)
    assert t.rb2(0.5)[:3] == pytest.approx([4.9129004, 1.7549878, 2.0535254], rel=2e-7)
    assert t.rb2(0.5, 1)[:3].tolist() == [4.0, 1.0, 1.0]
    assert t.rb2(1.0)[:3] == pytest.approx([1.4798877, 0.6802283, 0.8705127], rel=2e-7)   # (l + s)^2: 1 + 2s + s^2 with s^2 = 3/64, 27/256, 3/16
    assert np.all(np.isinf(t.rb2(0.0)))                                                    # theta = 0 opens everything
    # the deeper cells are the single-child chain down to the level where A and C separate (R5: chains are kept)
    assert t.depth == 3 and t.ncell == 6



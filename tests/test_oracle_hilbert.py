"""Pins of the oracle's Hilbert ordering (PAPER.md III-B step 2, L131; reading R20).  What a Hilbert curve
is fixes these: it is a bijection, consecutive keys are face-adjacent cells (no jumps -- the property the
paper wants it for, L131/L179), it is hierarchical (the top 3l bits of the key name the level-l octree
cell), and the tree built from it holds exactly the cells of the Morton tree."""
import numpy as np
import pytest

from workloads import generators as gen

B = 21


def test_bijection_adjacency_and_hierarchy_on_the_coarse_grid(orc):
    """all 16^3 cells of level 4 (coordinates in the top 4 of the 21 bits)"""
    lev, n = 4, 16
    sh = B - lev
    keys = {}
    for x in range(n):
        for y in range(n):
            for z in range(n):
                k = orc.hilbert_key([x << sh, y << sh, z << sh])
                keys[k >> (3 * sh)] = (x, y, z)
    assert sorted(keys) == list(range(n ** 3))                     # bijection onto 0 .. 4095
    path = np.array([keys[i] for i in range(n ** 3)])
    step = np.abs(np.diff(path, axis=0)).sum(axis=1)
    assert np.all(step == 1)                                       # consecutive keys: face neighbours
    for l in (1, 2, 3):                                            # hierarchy: a level-l prefix is one octree cell
        pre = np.arange(n ** 3) >> (3 * (lev - l))
        cell = (path >> (lev - l))
        for p in np.unique(pre):
            assert len(np.unique(cell[pre == p], axis=0)) == 1
        assert len(np.unique(np.c_[pre, cell], axis=0)) == 8 ** l


def test_inverse_and_fine_scale_adjacency(orc):
    rng = np.random.default_rng(7)
    for q in rng.integers(0, 1 << B, size=(200, 3), dtype=np.uint32):
        k = orc.hilbert_key(q)
        assert 0 <= k < 1 << 63
        assert np.array_equal(orc.hilbert_coords(k), q)
        if k + 1 < 1 << 63:                                        # the next key is a face neighbour at full depth
            d = np.abs(orc.hilbert_coords(k + 1).astype(np.int64) - q.astype(np.int64))
            assert d.sum() == 1
    # points in the same level-l octree cell share the top 3l key bits
    q0 = np.array([0x155555, 0x0F0F0F, 0x123456], dtype=np.uint32)
    for l in (1, 5, 13, 20):
        low = (1 << (B - l)) - 1
        a = orc.hilbert_key(q0 & ~np.uint32(low))
        b = orc.hilbert_key(q0 | np.uint32(low))
        assert a >> (3 * (B - l)) == b >> (3 * (B - l))


def test_hilbert_tree_has_the_cells_of_the_morton_tree(orc):
    pm = gen.plummer(6000, 31)
    pm[:, 3] = ((1 + np.arange(6000) % 5) / 6000.0).astype(np.float32)
    tm, th = orc.Tree(pm, 8), orc.Tree(pm, 8, key_order=1)
    assert (tm.ncell, tm.nleaf, tm.depth, tm.S) == (th.ncell, th.nleaf, th.depth, th.S)
    em, eh = tm.export(), th.export()

    def cellsets(e):
        out = {}
        for c in range(len(e["cells"])):
            f, n = int(e["cells"]["first"][c]), int(e["cells"]["count"][c])
            out[(int(e["cells"]["level"][c]), tuple(sorted(e["perm"][f:f + n].tolist())))] = c
        return out
    sm, sh_ = cellsets(em), cellsets(eh)
    assert set(sm) == set(sh_)                                     # same cells as sets of particles
    for k in list(sm)[::37]:
        a, b = sm[k], sh_[k]
        assert np.allclose(em["MP"][a], eh["MP"][b], rtol=1e-13, atol=1e-300)
        assert em["s"][a] == pytest.approx(eh["s"][b], rel=1e-9, abs=1e-15)    # same geometric centre
    # Hilbert-contiguous groups do not straddle octant boundaries with system-sized boxes (only the sparse ends
    # of the curve still have large boxes): fewer interactions and a shorter 90th-percentile list at the same theta
    rm, rh = tm.gravity(0.01, 0.6, 64, forces=False), th.gravity(0.01, 0.6, 64, forces=False)
    assert rh["interactions"] < rm["interactions"]
    lm, lh = rm["n_cells"].astype(np.int64) + rm["n_parts"], rh["n_cells"].astype(np.int64) + rh["n_parts"]
    assert np.percentile(lh, 90) < np.percentile(lm, 90)
    d = orc.direct_sum(pm, 0.01)
    assert np.allclose(th.gravity(0.01, 0.0, 64)["acc_pot"], d, rtol=1e-12, atol=1e-14)
    # every group's lists still tile the system
    rb2 = th.rb2(0.6)
    for g in (0, 17, th.n_groups(64) - 1):
        cells, parts = th.group_lists_rb2(rb2, 64, g, rh["n_cells"][g], rh["n_parts"][g])
        cover = np.zeros(6000, np.int32)
        cover[parts] += 1
        for c in cells:
            f, n = int(eh["cells"]["first"][c]), int(eh["cells"]["count"][c])
            cover[f:f + n] += 1
        assert np.all(cover == 1)

"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle on the same seeded
inputs.  Integer work (keys, permutation, cells, per-group counters) must match bit for bit;
floating point within the tolerances of DESIGN.md (R12, north_star: 1e-5)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from workloads import generators as gen  # noqa: E402


@pytest.fixture(scope="module")
def otoo():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1206_1199_b200 import binding
    o = binding.Otoo(max_particles=1 << 21, device=0)
    yield o
    o.close()


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


from tests.parity_rule import TOL, U32, FLOOR_FRAC_MAX_GRAVITY, FLOOR_FRAC_MAX_SPH, report, scalar_rel   # noqa: E402  (the one statement of the rule, R12)


def _label():
    import os
    return os.environ.get("PYTEST_CURRENT_TEST", "?").split("::")[-1].split(" ")[0]


def acc_err(got, want, abs_sum, pct=99.9, floor_frac_max=None, what="acc"):
    """R12 through tests/parity_rule.report (asserts the rule, prints and logs the audit numbers: un-floored max,
    p99.9, median, fraction of particles on the 8 u A floor).  Returns (|da| / bound scaled to 1e-5, plain
    relative error) for the callers' own assertions."""
    if floor_frac_max is None:
        floor_frac_max = FLOOR_FRAC_MAX_GRAVITY if what == "acc" else FLOOR_FRAC_MAX_SPH
    report(f"{_label()}:{what}", got[:, :3], want[:, :3], abs_sum, pct=pct, floor_frac_max=floor_frac_max)
    d = np.linalg.norm(got[:, :3].astype(np.float64) - want[:, :3], axis=1)
    an = np.linalg.norm(want[:, :3], axis=1)
    tol = np.maximum(1e-5 * an, 8 * U32 * abs_sum)
    return 1e-5 * d / np.maximum(tol, 1e-300), d / np.maximum(an, 1e-300)


def check_tree(otoo, orc, pm, n_crit, key_order=0):
    t = orc.Tree(pm, n_crit, key_order=key_order)
    otoo.otoo_set_option("key_order", key_order)
    try:
        otoo.otoo_build_tree(dev(pm), n_crit)
    finally:
        otoo.otoo_set_option("key_order", 0)
    ex = otoo.otoo_export_tree()
    eo = t.export()
    assert ex["N"] == t.N and ex["N_cell"] == t.ncell and ex["N_leaf"] == t.nleaf and ex["depth"] == t.depth
    assert np.array_equal(ex["lo"], t.lo) and ex["S"] == t.S
    assert np.array_equal(ex["keys"], eo["keys"])
    assert np.array_equal(ex["perm"], eo["perm"])
    for f in ("level", "prefix", "first", "count", "child_first", "child_count"):
        assert np.array_equal(ex["cells"][f], eo["cells"][f]), f
    assert np.array_equal(ex["com_m"].view(np.uint32), eo["com_m"].view(np.uint32))   # bit-exact cm, m (R6)
    return t


@pytest.mark.parametrize("kind,n,n_crit,seed", [("plummer", 16384, 16, 1206), ("plummer", 5000, 1, 1199),
                                                ("uniform_cube", 3001, 8, 2012), ("hernquist", 40000, 16, 3),
                                                ("plummer", 1, 16, 1), ("plummer", 7, 16, 2), ("uniform_sphere", 4097, 2, 5),
                                                ("plummer", 9000, 256, 6), ("plummer", 9000, 300, 7), ("plummer", 200, 256, 8)])
def test_tree_parity(otoo, orc, kind, n, n_crit, seed):
    check_tree(otoo, orc, gen.make(kind, n, seed), n_crit)


def test_tree_small_and_block_edge_sizes(otoo, orc):
    """N around 1, a warp, a block of 256 slots and the 64-slot look-ahead window of place_cells_kernel, with leaves of
    1 ... 100 particles: every cell tuple, key and moment against the oracle (leaves that straddle blocks and windows,
    blocks whose last warp is ragged, trees that are a single leaf)."""
    for n in (1, 2, 3, 5, 17, 31, 32, 33, 63, 64, 65, 255, 256, 257, 319, 320, 321, 511, 512, 513, 1000):
        for n_crit in (1, 3, 16, 100):
            pm = gen.plummer(n, 100 + n)
            check_tree(otoo, orc, pm, n_crit)
    pm = gen.uniform_cube(700, 5)
    pm[250:330] = pm[250]                 # 80 coincident points across the first block boundary and beyond its window
    check_tree(otoo, orc, pm, 4)
    check_tree(otoo, orc, pm, 4, key_order=1)


def test_tree_degenerate_inputs(otoo, orc):
    pm = np.zeros((300, 4), np.float32)
    pm[:, :3] = 2.5
    pm[:, 3] = 1.0
    check_tree(otoo, orc, pm, 4)            # all coincident: chain to level 21, leaf of 300
    pm2 = gen.plummer(2000, 4)
    pm2[100:140] = pm2[100]                 # a clump of duplicates inside a normal tree
    pm2[:, 3] = (1 + np.arange(2000) % 5) / 2000.0
    check_tree(otoo, orc, pm2, 8)
    pm3 = gen.uniform_cube(1000, 9)
    pm3[:, 2] = 0.25                        # planar: S from x/y only
    check_tree(otoo, orc, pm3, 16)


@pytest.mark.parametrize("kind,n,G,theta,eps", [("plummer", 16384, 64, 0.5, 0.01), ("plummer", 16384 + 37, 128, 0.6, 0.01),
                                                ("plummer", 20000, 256, 0.8, 0.004), ("hernquist", 30000, 32, 0.4, 0.002),
                                                ("uniform_cube", 50000, 128, 0.5, 0.001), ("plummer", 3000, 64, 0.0, 0.01),
                                                ("plummer", 3000, 128, 0.5, 0.0), ("uniform_sphere", 2500, 256, 0.0, 0.0),
                                                ("plummer", 40, 64, 0.5, 0.01), ("plummer", 6000 + 3, 4, 0.6, 0.01), ("hernquist", 9000 + 5, 8, 0.5, 0.002),
                                                ("uniform_cube", 12000 + 7, 16, 0.5, 0.001)])
@pytest.mark.parametrize("ws,dist", [(1, 2), (0, 2), (1, 0), (0, 0)])
def test_gravity_parity(otoo, orc, kind, n, G, theta, eps, ws, dist):
    """ws = 1: walker/evaluator warp pairs (default); ws = 0: the fused one-warp-does-both kernel.
    dist = 2: group-cell distance from the boxes of the group's pieces (R25, default); 0: from one box (R8)."""
    pm = gen.make(kind, n, 1206)
    t = check_tree(otoo, orc, pm, 16)
    theta32, eps32 = float(np.float32(theta)), float(np.float32(eps))
    t.set_dist_kind(dist)
    ref = t.gravity(eps32, theta32, G)
    otoo.otoo_set_option("warp_specialized", ws)
    otoo.otoo_set_option("group_distance", dist)
    try:
        out = otoo.otoo_gravity(eps32, theta32, G).cpu().numpy()
    finally:
        otoo.otoo_set_option("warp_specialized", 1)
        otoo.otoo_set_option("group_distance", 2)
    assert np.array_equal(otoo.otoo_export_tree()["rb2"].view(np.uint32), t.rb2(theta32).view(np.uint32))
    nt, nc, npart = otoo.otoo_export_group_stats()
    assert np.array_equal(nt, ref["n_tests"]) and np.array_equal(nc, ref["n_cells"]) and np.array_equal(npart, ref["n_parts"])
    st = otoo.otoo_last_stats()
    assert st["sum_interactions"] == ref["interactions"] and st["sum_tests"] == int(ref["n_tests"].sum())
    e, raw = acc_err(out, ref["acc_pot"], ref["abs_sum"])
    assert e.max() <= TOL, (e.max(), np.median(e), raw.max())
    assert np.percentile(raw, 99.9) <= TOL          # plain 1e-5 relative error for 99.9 % of the particles
    pe = np.abs(out[:, 3] - ref["acc_pot"][:, 3]) / np.abs(ref["acc_pot"][:, 3])
    assert pe.max() <= TOL, pe.max()


@pytest.mark.parametrize("kind,n,G,delta,m_limit,eps", [("plummer", 16384, 64, 0.01, 0.05, 0.01), ("plummer", 20000 + 5, 128, 0.1, np.inf, 0.004),
                                                        ("uniform_sphere", 30000, 32, 0.001, 0.025, 0.0), ("hernquist", 25000, 256, 1.0, 0.05, 0.002),
                                                        ("plummer", 3000, 64, 0.0, np.inf, 0.01)])
def test_gravity_delta_mac_parity(otoo, orc, kind, n, G, delta, m_limit, eps):
    """The paper's absolute-error MAC (Eq. 1-2, m_limit rule L157): rb^2 of every cell bit-exact,
    hence lists and counters exact; sums within the tolerances of the theta path."""
    pm = gen.make(kind, n, 1199)
    pm[:, 3] = ((1 + np.arange(n) % 3) / (2.0 * n)).astype(np.float32)        # unequal masses
    t = check_tree(otoo, orc, pm, 16)
    d32, ml32, eps32 = float(np.float32(delta)), float(np.float32(m_limit)), float(np.float32(eps))
    rb2 = t.rb2_delta(d32, ml32)
    ref = t.gravity(eps32, 0.0, G, rb2=rb2)
    out = otoo.otoo_gravity_delta(eps32, d32, ml32, G).cpu().numpy()
    assert np.array_equal(otoo.otoo_export_tree()["rb2"].view(np.uint32), rb2.view(np.uint32))
    nt, nc, npart = otoo.otoo_export_group_stats()
    assert np.array_equal(nt, ref["n_tests"]) and np.array_equal(nc, ref["n_cells"]) and np.array_equal(npart, ref["n_parts"])
    assert otoo.otoo_last_stats()["sum_interactions"] == ref["interactions"]
    e, raw = acc_err(out, ref["acc_pot"], ref["abs_sum"])
    assert e.max() <= TOL, (e.max(), raw.max())
    assert np.percentile(raw, 99.9) <= TOL
    pe = np.abs(out[:, 3] - ref["acc_pot"][:, 3]) / np.abs(ref["acc_pot"][:, 3])
    assert pe.max() <= TOL
    # an SPH call after it must not see the h = 0 radii of the Delta pass
    if n == 16384:
        h = np.full(n, 0.3, np.float32)
        rho, _ = otoo.otoo_sph_density(dev(h), 64)
        rref = t.sph_density(h, 64, groups=np.arange(4))
        idx = t.group_targets(64, np.arange(4))
        assert (np.abs(rho.cpu().numpy()[idx] - rref["rho"][idx]) / rref["rho"][idx]).max() <= TOL


@pytest.mark.parametrize("kind,n,n_crit,G", [("plummer", 16384, 16, 64), ("hernquist", 30000 + 7, 8, 128), ("uniform_cube", 40000, 16, 256),
                                             ("plummer", 9, 16, 32), ("uniform_sphere", 5000, 1, 32)])
def test_hilbert_order_parity(otoo, orc, kind, n, n_crit, G):
    """key_order = 1 (reading R20): keys, permutation, cells, moments bit-exact against the oracle's
    Hilbert tree; theta- and Delta-MAC walks exact; SPH density on the same tree."""
    pm = gen.make(kind, n, 2012)
    t = check_tree(otoo, orc, pm, n_crit, key_order=1)
    ref = t.gravity(0.01, float(np.float32(0.6)), G)
    out = otoo.otoo_gravity(0.01, float(np.float32(0.6)), G).cpu().numpy()
    nt, nc, npart = otoo.otoo_export_group_stats()
    assert np.array_equal(nt, ref["n_tests"]) and np.array_equal(nc, ref["n_cells"]) and np.array_equal(npart, ref["n_parts"])
    e, raw = acc_err(out, ref["acc_pot"], ref["abs_sum"])
    assert e.max() <= TOL
    rb2 = t.rb2_delta(float(np.float32(0.01)), float(np.float32(0.05)))
    refd = t.gravity(0.01, 0.0, G, rb2=rb2)
    outd = otoo.otoo_gravity_delta(0.01, 0.01, 0.05, G).cpu().numpy()
    assert np.array_equal(otoo.otoo_export_tree()["rb2"].view(np.uint32), rb2.view(np.uint32))
    nt, nc, npart = otoo.otoo_export_group_stats()
    assert np.array_equal(nt, refd["n_tests"]) and np.array_equal(nc, refd["n_cells"]) and np.array_equal(npart, refd["n_parts"])
    e, _ = acc_err(outd, refd["acc_pot"], refd["abs_sum"])
    assert e.max() <= TOL
    if n >= 1000:
        h = np.full(n, 0.1 * t.S / n ** (1 / 3) * 4, np.float32)
        rs = t.sph_density(h, G if G <= 128 else 128)
        rho, nngb = otoo.otoo_sph_density(dev(h), G if G <= 128 else 128)
        assert np.array_equal(nngb.cpu().numpy().view(np.uint32), rs["nngb"])
        assert (np.abs(rho.cpu().numpy() - rs["rho"]) / rs["rho"]).max() <= TOL


@pytest.mark.parametrize("kind,n,G,theta,key_order", [("plummer", 16384, 64, 0.5, 0), ("plummer", 20000 + 9, 128, 0.6, 0), ("hernquist", 30000, 32, 0.4, 1),
                                                       ("uniform_cube", 40000, 256, 0.5, 0), ("plummer", 3000, 128, 0.0, 0),
                                                       ("uniform_sphere", 8000 + 1, 4, 0.6, 1), ("plummer", 10000 + 3, 8, 0.5, 0)])
def test_exact_min_group_distance_parity(otoo, orc, kind, n, G, theta, key_order):
    """group_distance = 1: the paper's vector walk (reading R23) -- the MAC compares r_b with the
    actual minimum of the members' distances.  Lists (counters) exact, sums within tolerance, for both MACs."""
    pm = gen.make(kind, n, 1206)
    t = check_tree(otoo, orc, pm, 16, key_order=key_order)
    theta32 = float(np.float32(theta))
    t.set_dist_kind(0)
    aabb = t.gravity(0.01, theta32, G, forces=False)
    t.set_dist_kind(1)
    otoo.otoo_set_option("group_distance", 1)
    try:
        ref = t.gravity(0.01, theta32, G)
        out = otoo.otoo_gravity(0.01, theta32, G).cpu().numpy()
        nt, nc, npart = otoo.otoo_export_group_stats()
        assert np.array_equal(nt, ref["n_tests"]) and np.array_equal(nc, ref["n_cells"]) and np.array_equal(npart, ref["n_parts"])
        assert otoo.otoo_last_stats()["sum_interactions"] == ref["interactions"] <= aabb["interactions"]
        e, raw = acc_err(out, ref["acc_pot"], ref["abs_sum"])
        assert e.max() <= TOL and np.percentile(raw, 99.9) <= TOL
        rb2 = t.rb2_delta(float(np.float32(0.01)), float(np.float32(0.05)))
        refd = t.gravity(0.01, 0.0, G, rb2=rb2)
        outd = otoo.otoo_gravity_delta(0.01, 0.01, 0.05, G).cpu().numpy()
        nt, nc, npart = otoo.otoo_export_group_stats()
        assert np.array_equal(nt, refd["n_tests"]) and np.array_equal(nc, refd["n_cells"]) and np.array_equal(npart, refd["n_parts"])
        e, _ = acc_err(outd, refd["acc_pot"], refd["abs_sum"])
        assert e.max() <= TOL
        otoo.otoo_set_option("warp_specialized", 0)          # the one-warp kernel has no exact-minimum form: refused
        from paper_1206_1199_b200 import binding
        with pytest.raises(binding.OtooError):
            otoo.otoo_gravity(0.01, theta32, G)
    finally:
        otoo.otoo_set_option("warp_specialized", 1)
        otoo.otoo_set_option("group_distance", 2)


def test_walk_stack_spill(otoo, orc):
    """theta = 0 on a deep tree overflows the 512-entry shared stack: both overflow paths (task pool,
    private global spill) must give the same lists."""
    pm = gen.plummer(30000, 77)
    t = check_tree(otoo, orc, pm, 1)
    try:
        for theta, pool, ws in ((0.0, 0, 1), (0.0, 1, 1), (0.3, 0, 1), (0.0, 0, 0), (0.0, 1, 0)):
            otoo.otoo_set_option("task_pool", pool)
            otoo.otoo_set_option("warp_specialized", ws)
            ref = t.gravity(0.01, theta, 32)
            out = otoo.otoo_gravity(0.01, theta, 32).cpu().numpy()
            nt, nc, npart = otoo.otoo_export_group_stats()
            assert np.array_equal(nt, ref["n_tests"]) and np.array_equal(nc, ref["n_cells"]) and np.array_equal(npart, ref["n_parts"])
            e, _ = acc_err(out, ref["acc_pot"], ref["abs_sum"])
            assert e.max() <= TOL
    finally:
        otoo.otoo_set_option("task_pool", 1)
        otoo.otoo_set_option("warp_specialized", 1)


@pytest.mark.parametrize("ws,dist", [(0, 2), (1, 2), (0, 0), (1, 0)])
@pytest.mark.parametrize("n,G", [(20000, 64), (20000 + 11, 32), (8000, 128), (6000, 256), (5000 + 3, 4), (6000 + 1, 16)])
def test_sph_parity(otoo, orc, n, G, ws, dist):
    """ws = 0: one warp walks and sums in turn (default); ws = 1: walker/evaluator warp pairs.
    dist = 2: the SPH MAC per piece of the group (R26, default); 0: one box per group (R15)."""
    otoo.otoo_set_option("warp_specialized_sph", ws)
    otoo.otoo_set_option("group_distance", dist)
    try:
        _sph_parity(otoo, orc, n, G, dist)
    finally:
        otoo.otoo_set_option("warp_specialized_sph", 0)
        otoo.otoo_set_option("group_distance", 2)


def _sph_parity(otoo, orc, n, G, dist=2):
    w = gen.wd_pair(n, 1206)
    pm, h, u = w["pos_mass"], w["h"], w["u"]
    # the generator's rigid rotation has (v_i - v_j).(x_i - x_j) = 0 for every pair (du/dt would be
    # rounding noise): add a homologous contraction and a seeded perturbation for the du/dt check
    vel = w["vel"].copy()
    vel[:, :3] += -0.3 * pm[:, :3] + 0.05 * (gen.uniform01(99, np.arange(3 * n, dtype=np.uint64), 0).reshape(n, 3) - 0.5)
    vel = vel.astype(np.float32)
    t = check_tree(otoo, orc, pm, 16)
    t.set_dist_kind(dist)
    ref = t.sph_density(h, G)
    rho, nngb = otoo.otoo_sph_density(dev(h), G)
    b, r = otoo.otoo_export_sph_radii()
    bo, ro = t.sph_cell_radii(h)
    assert np.array_equal(b.view(np.uint32), bo.view(np.uint32)) and np.array_equal(r.view(np.uint32), ro.view(np.uint32))
    nt, _, npart = otoo.otoo_export_group_stats()
    assert np.array_equal(nt, ref["n_tests"]) and np.array_equal(npart, ref["n_parts"])
    assert otoo.otoo_last_stats()["sum_interactions"] == ref["candidates"]
    assert np.array_equal(nngb.cpu().numpy().view(np.uint32), ref["nngb"])
    rg = rho.cpu().numpy()
    assert (np.abs(rg - ref["rho"]) / ref["rho"]).max() <= TOL
    # stage 2 from the GPU's own density (R17): EOS on the device, oracle fed the same fp32 rho, P
    P = otoo.otoo_eos_ideal(rho, dev(u), 5.0 / 3.0)
    Pg = P.cpu().numpy()
    assert np.array_equal(Pg, (np.float32(5.0 / 3.0) - np.float32(1.0)) * rg * u)
    for v in (None, vel):
        rf = t.sph_force(h, rg.astype(np.float64), Pg.astype(np.float64), G, vel=v)
        reff = rf["acc_dudt"]
        otoo.otoo_set_option("sph_reuse_radii", 0 if v is None else 1)     # second pass: keep the radii of the first
        try:
            out = otoo.otoo_sph_force(dev(h), rho, P, G, vel=None if v is None else dev(v)).cpu().numpy()
        finally:
            otoo.otoo_set_option("sph_reuse_radii", 0)
        if v is not None:
            assert otoo.otoo_last_stats()["launches"] < launches_plain
        else:
            launches_plain = otoo.otoo_last_stats()["launches"]
        # pressure forces cancel pairwise: same bound as gravity, max(1e-5 |a|, 8 u sum_j |a_ij|) (R12)
        e, raw = acc_err(out, reff, rf["abs_sum"][:, 0], pct=99, what="a_sph")
        assert e.max() <= TOL, e.max()
        assert np.percentile(raw, 99) <= TOL
        if v is not None:
            report(f"{_label()}:dudt", out[:, 3], reff[:, 3], rf["abs_sum"][:, 1], pct=None)
        else:
            assert np.all(out[:, 3] == 0)


@pytest.mark.parametrize("pool", [1, 0])
@pytest.mark.parametrize("n,G,dist", [(20000, 64, 2), (20000 + 11, 32, 2), (8000, 128, 0), (6000, 256, 2), (6000 + 1, 16, 2)])
def test_sph_force_replays_the_leaves_of_the_density_walk(otoo, orc, n, G, dist, pool):
    """Option sph_reuse_walk (with sph_reuse_radii): the density walk records the leaves every group opens, the force walk
    starts from them instead of the root -- the same MAC (R15 / R26) opens them all again.  Against the oracle: per-group
    tests and particles of the force walk exact (the tests of the internal cells are counted, not repeated), forces and
    du/dt within the rule; against the plain force walk: the same counters, and fewer walk steps where every group could
    record (pool = 0: no part of a group's walk is handed to another warp; with the pool a group that donated walks again)."""
    w = gen.wd_pair(n, 77)
    pm, h, u = w["pos_mass"], w["h"], w["u"]
    vel = (w["vel"] - 0.3 * np.c_[pm[:, :3], np.zeros(n)]).astype(np.float32)
    t = check_tree(otoo, orc, pm, 16)
    t.set_dist_kind(dist)
    otoo.otoo_set_option("group_distance", dist)
    otoo.otoo_set_option("task_pool", pool)
    try:
        rho, _ = otoo.otoo_sph_density(dev(h), G)
        P = otoo.otoo_eos_ideal(rho, dev(u), 5.0 / 3.0)
        rg, Pg = rho.cpu().numpy(), P.cpu().numpy()
        plain = otoo.otoo_sph_force(dev(h), rho, P, G, vel=dev(vel)).cpu().numpy()
        st_plain = otoo.otoo_last_stats()
        nt_plain, _, np_plain = otoo.otoo_export_group_stats()
        otoo.otoo_set_option("sph_reuse_walk", 1)
        otoo.otoo_set_option("sph_reuse_radii", 1)
        rho2, _ = otoo.otoo_sph_density(dev(h), G)                       # records
        assert float((rho2 - rho).abs().max()) <= 1e-6 * float(rho.abs().max())      # (pool tasks add in another order)
        out = otoo.otoo_sph_force(dev(h), rho, P, G, vel=dev(vel)).cpu().numpy()   # replays
        st = otoo.otoo_last_stats()
        nt, _, npart = otoo.otoo_export_group_stats()
    finally:
        otoo.otoo_set_option("sph_reuse_walk", 0)
        otoo.otoo_set_option("sph_reuse_radii", 0)
        otoo.otoo_set_option("group_distance", 2)
        otoo.otoo_set_option("task_pool", 1)
    assert np.array_equal(nt, nt_plain) and np.array_equal(npart, np_plain)
    assert st["sum_tests"] == st_plain["sum_tests"] and st["sum_interactions"] == st_plain["sum_interactions"]
    if pool == 0 and G <= 64:                                           # (the replaying kernels exist for groups up to 64)
        assert st["sum_steps"] < 0.9 * st_plain["sum_steps"]            # the internal levels were not walked again
    if G > 64:
        assert st["sum_steps"] == st_plain["sum_steps"] or pool == 1    # larger groups walk from the root as before
    rf = t.sph_force(h, rg.astype(np.float64), Pg.astype(np.float64), G, vel=vel)
    rd = t.sph_density(h, G)                                            # (the oracle's walk is the same for both stages)
    assert np.array_equal(nt, rd["n_tests"]) and np.array_equal(npart, rd["n_parts"])
    e, raw = acc_err(out, rf["acc_dudt"], rf["abs_sum"][:, 0], pct=99, what="a_sph")
    assert e.max() <= TOL, e.max()
    report(f"{_label()}:dudt", out[:, 3], rf["acc_dudt"][:, 3], rf["abs_sum"][:, 1], pct=None)
    assert np.abs(out - plain).max() <= 1e-4 * np.abs(plain).max()      # (another order of the same leaves)


@pytest.mark.parametrize("kind,n,G,target,tol,h0", [("uniform_cube", 20000, 64, 40.0, 2.0, 0.03), ("wd", 16384 + 3, 32, 50.0, 3.0, None),
                                                      ("uniform_cube", 5000, 128, 32.0, 0.0, 0.2)])
def test_adaptive_h_parity(otoo, orc, kind, n, G, target, tol, h0):
    """otoo_sph_adapt_h (reading R21): the same number of updates, the same h bit for bit, the same counts."""
    if kind == "wd":
        w = gen.wd_pair(n, 77)
        pm, h = w["pos_mass"], (w["h"] * np.float32(0.6)).astype(np.float32)
    else:
        pm, h = gen.make(kind, n, 77), np.full(n, h0, np.float32)
    t = check_tree(otoo, orc, pm, 16)
    for max_iter in (2, 40):
        href, nref, itref = t.sph_adapt_h(h, target, tol, max_iter, G)
        d_h = dev(h.copy())
        nn, it = otoo.otoo_sph_adapt_h(d_h, target, tol, max_iter, G)
        assert it == itref
        assert np.array_equal(d_h.cpu().numpy().view(np.uint32), href.view(np.uint32))
        assert np.array_equal(nn.cpu().numpy().view(np.uint32), nref)
    if tol > 0:
        assert np.all(np.abs(nref.astype(float) - target) <= tol)


@pytest.mark.parametrize("n,G", [(20000, 64), (9000 + 5, 32), (6000, 128)])
def test_sph_stage1_divrot_parity(otoo, orc, n, G):
    """otoo_sph_stage1 (PAPER L252 step 4; reading R22): density and counts as otoo_sph_density, div v and rot v
    within max(1e-5 |x|, 8 u sum_j |x_ij|) (the velocity differences cancel like the pressure terms)."""
    w = gen.wd_pair(n, 31)
    pm, h = w["pos_mass"], w["h"]
    vel = w["vel"].copy()
    vel[:, :3] += -0.3 * pm[:, :3] + 0.05 * (gen.uniform01(5, np.arange(3 * n, dtype=np.uint64), 0).reshape(n, 3) - 0.5)
    vel = vel.astype(np.float32)
    t = check_tree(otoo, orc, pm, 16)
    ref = t.sph_divrot(h, vel, G)
    rho, nngb, dr = otoo.otoo_sph_stage1(dev(h), dev(vel), G)
    rho0, nn0 = otoo.otoo_sph_density(dev(h), G)
    assert np.array_equal(nngb.cpu().numpy(), nn0.cpu().numpy())
    rg = rho.cpu().numpy()
    assert (np.abs(rg - ref["rho"]) / ref["rho"]).max() <= TOL
    assert (np.abs(rg - rho0.cpu().numpy()) / rg).max() <= 4 * U32 * 8
    got = dr.cpu().numpy().astype(np.float64)
    report(f"{_label()}:div_v", got[:, 0], ref["divrot"][:, 0], ref["abs_sum"], pct=None)
    report(f"{_label()}:rot_v", got[:, 1:], ref["divrot"][:, 1:], ref["abs_sum"], pct=None)


@pytest.mark.parametrize("n,G", [(20000, 64), (7000 + 3, 32), (6000, 128)])
def test_sph_force_viscosity_parity(otoo, orc, n, G):
    """otoo_sph_force_visc (reading R24): the oracle fed the GPU's own fp32 rho, P; tolerance as the pressure force."""
    w = gen.wd_pair(n, 5)
    pm, h, u = w["pos_mass"], w["h"], w["u"]
    vel = np.zeros((n, 4), np.float32)
    vel[:, :3] = -0.4 * pm[:, :3] + 0.1 * np.sin(7 * pm[:, [1, 2, 0]])
    t = check_tree(otoo, orc, pm, 16)
    rho, _ = otoo.otoo_sph_density(dev(h), G)
    P = otoo.otoo_eos_ideal(rho, dev(u), 5.0 / 3.0)
    rg, Pg = rho.cpu().numpy(), P.cpu().numpy()
    visc = np.zeros((n, 4), np.float32)
    visc[:, 0] = np.sqrt((5.0 / 3.0) * Pg / rg)
    visc[:, 1] = 0.5 + 0.5 * gen.uniform01(3, np.arange(n, dtype=np.uint64), 0)
    visc[:, 2] = gen.uniform01(4, np.arange(n, dtype=np.uint64), 0)
    ref = t.sph_force(h, rg.astype(np.float64), Pg.astype(np.float64), G, vel=vel, visc=visc)
    base = t.sph_force(h, rg.astype(np.float64), Pg.astype(np.float64), G, vel=vel)
    assert np.abs(ref["acc_dudt"] - base["acc_dudt"]).max() > 1e-3 * np.abs(base["acc_dudt"]).max()   # the term is there
    out = otoo.otoo_sph_force_visc(dev(h), rho, P, dev(vel), dev(visc), G).cpu().numpy()
    e, raw = acc_err(out, ref["acc_dudt"], ref["abs_sum"][:, 0], pct=99, what="a_sph_visc")
    assert e.max() <= TOL, e.max()
    assert np.percentile(raw, 99) <= TOL
    report(f"{_label()}:dudt", out[:, 3], ref["acc_dudt"][:, 3], ref["abs_sum"][:, 1], pct=None)
    v0 = visc.copy()
    v0[:, 1] = 0.0                                                                                   # alpha = 0: the plain force
    out0 = otoo.otoo_sph_force_visc(dev(h), rho, P, dev(vel), dev(v0), G).cpu().numpy()
    plain = otoo.otoo_sph_force(dev(h), rho, P, G, vel=dev(vel)).cpu().numpy()
    assert np.allclose(out0, plain, rtol=1e-5, atol=1e-6 * np.abs(plain).max())
    # the paper's step (L252 steps 4, 6) with option sph_reuse_walk: stage 1 records the opened leaves, the viscous force
    # starts from them: the counters of the full walk, the same forces within the rule
    nt_full, _, np_full = otoo.otoo_export_group_stats()
    otoo.otoo_set_option("sph_reuse_walk", 1)
    otoo.otoo_set_option("sph_reuse_radii", 1)
    try:
        otoo.otoo_sph_stage1(dev(h), dev(vel), G)
        out_r = otoo.otoo_sph_force_visc(dev(h), rho, P, dev(vel), dev(visc), G).cpu().numpy()
        nt_r, _, np_r = otoo.otoo_export_group_stats()
    finally:
        otoo.otoo_set_option("sph_reuse_walk", 0)
        otoo.otoo_set_option("sph_reuse_radii", 0)
    assert np.array_equal(nt_r, nt_full) and np.array_equal(np_r, np_full)
    e, raw = acc_err(out_r, ref["acc_dudt"], ref["abs_sum"][:, 0], pct=99, what="a_sph_visc_replay")
    assert e.max() <= TOL, e.max()


@pytest.mark.parametrize("world,by_cost", [(3, False), (4, True)])
def test_target_sharding_ranges_add_up(otoo, orc, world, by_cost):
    """The paper's multi-device scheme (PAPER.md III-E, L179) on one GPU: the ranks' ranges are run one after the
    other on the same tree (no rank waits for another); every group's counters are those of the oracle, each
    target is written by exactly one range, and the ranges' outputs add up to the single-call result."""
    from paper_1206_1199_b200 import sharded
    n, G = 40000, 64
    pm = gen.plummer(n, 8)
    t = check_tree(otoo, orc, pm, 16)
    ref = t.gravity(0.01, 0.5, G)
    whole = otoo.otoo_gravity(0.01, 0.5, G).cpu().numpy()
    ng = t.n_groups(G)
    cost = (ref["n_cells"].astype(np.int64) + ref["n_parts"]) if by_cost else None
    ranges = sharded.group_ranges(ng, world, cost)
    total = np.zeros((n, 4), np.float64)
    written = np.zeros(n, np.int32)
    perm = t.export()["perm"].astype(np.int64)
    inter = 0
    try:
        for b, c in ranges:
            otoo.otoo_set_option("group_begin", b)
            otoo.otoo_set_option("group_count", c)
            part = otoo.otoo_gravity(0.01, 0.5, G).cpu().numpy()
            nt, nc, npart = otoo.otoo_export_group_stats()
            assert np.array_equal(nt[b:b + c], ref["n_tests"][b:b + c]) and np.array_equal(nc[b:b + c], ref["n_cells"][b:b + c])
            assert not nt[:b].any() and not nt[b + c:].any()
            inter += otoo.otoo_last_stats()["sum_interactions"]
            mine = perm[b * G:min((b + c) * G, n)]
            written[mine] += 1
            rest = np.setdiff1d(np.arange(n), mine)
            assert not part[rest].any()
            total += part
        otoo.otoo_set_option("group_begin", ng)                    # an empty range at the end is legal, one past it is not
        otoo.otoo_set_option("group_count", 0)
        assert not otoo.otoo_gravity(0.01, 0.5, G).cpu().numpy().any()
        otoo.otoo_set_option("group_count", 1)
        from paper_1206_1199_b200 import binding
        with pytest.raises(binding.OtooError):
            otoo.otoo_gravity(0.01, 0.5, G)
    finally:
        otoo.otoo_set_option("group_begin", 0)
        otoo.otoo_set_option("group_count", -1)
    assert np.all(written == 1) and inter == ref["interactions"]
    assert np.allclose(total, whole, rtol=2e-6, atol=1e-6 * np.abs(whole).max())
    e, _ = acc_err(total.astype(np.float32), ref["acc_pot"], ref["abs_sum"])
    assert e.max() <= TOL


def test_status_codes(otoo):
    from paper_1206_1199_b200 import binding
    fresh = binding.Otoo(max_particles=1000)
    out = torch.empty((10, 4), device="cuda")
    with pytest.raises(binding.OtooError) as e:
        fresh.otoo_gravity(0.01, 0.5, 64, out=out)
    assert e.value.status == binding.OTOO_ERR_NOT_BUILT
    pm = dev(gen.plummer(2000, 1))
    with pytest.raises(binding.OtooError) as e:
        fresh.otoo_build_tree(pm, 16)
    assert e.value.status == binding.OTOO_ERR_CAPACITY
    fresh.otoo_build_tree(pm[:500].contiguous(), 16)
    for bad in (dict(eps=0.01, delta=-1.0, m_limit=1.0, group_size=64), dict(eps=0.01, delta=0.1, m_limit=0.0, group_size=64),
                dict(eps=0.01, delta=float("nan"), m_limit=1.0, group_size=64)):
        with pytest.raises(binding.OtooError) as e:
            fresh.otoo_gravity_delta(**bad)
        assert e.value.status == binding.OTOO_ERR_INVALID_ARG
    for bad in (dict(eps=-1.0, theta=0.5, group_size=64), dict(eps=0.01, theta=-0.5, group_size=64),
                dict(eps=0.01, theta=0.5, group_size=48), dict(eps=0.01, theta=0.5, group_size=2)):
        with pytest.raises(binding.OtooError) as e:
            fresh.otoo_gravity(**bad)
        assert e.value.status == binding.OTOO_ERR_INVALID_ARG
    with pytest.raises(binding.OtooError) as e:
        fresh.otoo_build_tree(pm[:500].contiguous(), 0)
    assert e.value.status == binding.OTOO_ERR_INVALID_ARG
    fresh.otoo_build_tree(None, 16)          # N = 0: no-op, context not built
    with pytest.raises(binding.OtooError) as e:
        fresh.otoo_tree_info()
    assert e.value.status == binding.OTOO_ERR_NOT_BUILT
    fresh.close()


def test_host_entry_point(otoo, orc):
    pm = gen.plummer(10000, 5)
    out = otoo.otoo_gravity_host(pm, 16, 0.01, 0.5, 64)
    ref = orc.Tree(pm, 16).gravity(float(np.float32(0.01)), 0.5, 64)
    e, _ = acc_err(out, ref["acc_pot"], ref["abs_sum"])
    assert e.max() <= TOL


def test_config1_against_direct_sum(otoo, orc):
    """BASELINE config 1 (Plummer N = 16384, eps = 0.01, theta = 0.5, G = 64) against the O(N^2) direct sum: with
    theta = 0 the lists hold every particle and the CUDA sums are the direct sum to fp32 accuracy; with theta = 0.5
    the difference is the error of the monopole approximation."""
    cfg = gen.CONFIGS["C1"]
    n, G = cfg["n"], cfg["group"]
    pm = gen.make(cfg["kind"], n, 1206)
    eps = float(np.float32(cfg["eps"]))
    ref = orc.direct_sum(pm, eps)
    an = np.linalg.norm(ref[:, :3], axis=1)
    otoo.otoo_build_tree(dev(pm), cfg["n_crit"])
    out0 = otoo.otoo_gravity(eps, 0.0, G).cpu().numpy().astype(np.float64)
    assert otoo.otoo_last_stats()["sum_interactions"] == n * n
    e0 = np.linalg.norm(out0[:, :3] - ref[:, :3], axis=1) / an
    assert np.percentile(e0, 99.9) <= TOL and e0.max() <= 1e-4
    assert (np.abs(out0[:, 3] - ref[:, 3]) / np.abs(ref[:, 3])).max() <= TOL
    out = otoo.otoo_gravity(eps, float(np.float32(cfg["theta"])), G).cpu().numpy().astype(np.float64)
    e = np.linalg.norm(out[:, :3] - ref[:, :3], axis=1) / an
    assert 1e-6 < np.median(e) < 1e-3 and np.percentile(e, 99) < 1e-2
    assert np.median(np.abs(out[:, 3] - ref[:, 3]) / np.abs(ref[:, 3])) < 1e-3


def test_stats_phase_times_and_walk_only_flag(otoo, orc):
    """otoo_stats_t: per-phase device times of the last build and the last walk, and the record that a
    walk ran with `walk_only` (its outputs must not be mistaken for a result)."""
    pm = gen.plummer(200000, 3)
    otoo.otoo_build_tree(dev(pm), 16)
    otoo.otoo_gravity(0.01, 0.6, 128)
    st = otoo.otoo_last_stats()
    assert set(st["ms_build"]) == {"root_cube", "keys", "sort", "gather", "cells", "moments"}
    assert all(v > 0 for v in st["ms_build"].values())
    assert st["ms_build_total"] == pytest.approx(sum(st["ms_build"].values()), rel=1e-5)
    assert st["ms_walk_force"] > 0 and st["ms_walk_prep"] > 0
    assert st["ms_total"] == pytest.approx(st["ms_walk_prep"] + st["ms_walk_force"], rel=1e-5)
    assert st["ms_walk_force"] > st["ms_walk_prep"]                   # the fused walk + sum kernel dominates the call
    assert st["walk_only"] == 0 and st["error_flag"] == 0
    inter = st["sum_interactions"]
    otoo.otoo_set_option("walk_only", 1)
    try:
        otoo.otoo_gravity(0.01, 0.6, 128)
        st2 = otoo.otoo_last_stats()
        assert st2["walk_only"] == 1 and st2["sum_interactions"] == inter   # counters exact, outputs flagged
    finally:
        otoo.otoo_set_option("walk_only", 0)
    otoo.otoo_gravity(0.01, 0.6, 128)
    assert otoo.otoo_last_stats()["walk_only"] == 0


def test_build_leaves_rb2_and_reset_for_the_next_gravity_call(otoo, orc):
    """A build after a gravity call leaves rb^2 of that call's theta (R7) and a reset walk pool from inside its bottom-up
    pass: the next otoo_gravity with the same theta launches the walk kernel alone; another theta, or a second walk on
    the same tree, runs the r_b / reset kernel as before.  All three paths against the oracle, bit for bit on rb^2 and
    the counters."""
    pm = gen.plummer(30000 + 11, 21)
    t = orc.Tree(pm, 16)
    th1, th2, eps = float(np.float32(0.55)), float(np.float32(0.75)), float(np.float32(0.01))

    def check(theta, launches):
        out = otoo.otoo_gravity(eps, theta, 128).cpu().numpy()
        st = otoo.otoo_last_stats()
        assert st["launches"] == launches, (st["launches"], launches)
        ref = t.gravity(eps, theta, 128)
        assert np.array_equal(otoo.otoo_export_tree()["rb2"].view(np.uint32), t.rb2(theta).view(np.uint32))
        nt, nc, npart = otoo.otoo_export_group_stats()
        assert np.array_equal(nt, ref["n_tests"]) and np.array_equal(nc, ref["n_cells"]) and np.array_equal(npart, ref["n_parts"])
        assert st["sum_interactions"] == ref["interactions"]
        e, _ = acc_err(out, ref["acc_pot"], ref["abs_sum"])
        assert e.max() <= TOL

    otoo.otoo_build_tree(dev(pm), 16)
    check(th2, 2)                       # (whatever the fixture's last theta was: not th2 on this tree yet)
    otoo.otoo_build_tree(dev(pm), 16)
    check(th2, 1)                       # rb^2 of th2 and the reset came with the build
    check(th2, 2)                       # same tree, same theta: rb^2 stands, the pool needs its reset kernel
    check(th1, 2)                       # another theta: the r_b kernel (with the reset inside)
    otoo.otoo_build_tree(dev(pm), 16)
    check(th1, 1)
    otoo.otoo_build_tree(dev(pm), 16)
    check(th2, 2)                       # the build guessed th1


def test_spill_overflow_is_reported(otoo, orc):
    """Without the task pool and with a private spill area too small for theta = 0 on a deep tree the walk drops
    cells: the launch is flagged and the introspection calls return OTOO_ERR_CAPACITY instead of wrong numbers."""
    from paper_1206_1199_b200 import binding
    pm = gen.plummer(30000, 77)
    otoo.otoo_build_tree(dev(pm), 1)
    try:
        otoo.otoo_set_option("task_pool", 0)
        otoo.otoo_set_option("walk_spill", 0)
        otoo.otoo_gravity(0.01, 0.0, 32)
        with pytest.raises(binding.OtooError) as e:
            otoo.otoo_last_stats()
        assert e.value.status == binding.OTOO_ERR_CAPACITY
        with pytest.raises(binding.OtooError) as e:
            otoo.otoo_export_group_stats()
        assert e.value.status == binding.OTOO_ERR_CAPACITY
        otoo.otoo_set_option("walk_spill", 8192)
        otoo.otoo_gravity(0.01, 0.0, 32)
        assert otoo.otoo_last_stats()["error_flag"] == 0 and otoo.otoo_last_stats()["sum_interactions"] == 30000 * 30000
    finally:
        otoo.otoo_set_option("task_pool", 1)
        otoo.otoo_set_option("walk_spill", 8192)


def test_delta_host_entry_point(otoo, orc):
    pm = gen.plummer(10000, 5)
    out = otoo.otoo_gravity_delta_host(pm, 16, 0.01, 0.01, 0.05, 64)
    t = orc.Tree(pm, 16)
    ref = t.gravity(float(np.float32(0.01)), 0.0, 64, rb2=t.rb2_delta(float(np.float32(0.01)), float(np.float32(0.05))))
    e, _ = acc_err(out, ref["acc_pot"], ref["abs_sum"])
    assert e.max() <= TOL
    assert otoo.otoo_last_stats()["sum_interactions"] == ref["interactions"]


def test_binding_rejects_short_arrays(otoo):
    pm = gen.plummer(5000, 1)
    otoo.otoo_build_tree(dev(pm), 16)
    with pytest.raises(ValueError):
        otoo.otoo_gravity(0.01, 0.5, 64, out=torch.empty((4999, 4), dtype=torch.float32, device="cuda"))
    with pytest.raises(ValueError):
        otoo.otoo_sph_density(torch.full((100,), 0.1, device="cuda"), 64)


@pytest.mark.parametrize("world", [2, 3])
def test_sph_target_sharding_ranges_add_up(otoo, orc, world):
    """group_begin / group_count with the SPH entry points (PAPER III-E applied to stage 1 / stage 2): the ranges'
    outputs are zero outside their targets (no 0/0 from the div/rot normalisation), add up to the single-call
    result, and otoo_sph_adapt_h leaves the h of the other targets alone."""
    from paper_1206_1199_b200 import sharded
    n, G = 20000, 64
    w = gen.wd_pair(n, 11)
    pm, h = w["pos_mass"], w["h"]
    vel = np.zeros((n, 4), np.float32)
    vel[:, :3] = -0.4 * pm[:, :3] + 0.1 * np.sin(7 * pm[:, [1, 2, 0]])
    t = check_tree(otoo, orc, pm, 16)
    perm = t.export()["perm"].astype(np.int64)
    d_h, d_v = dev(h), dev(vel)
    rho_w, nn_w, dr_w = (x.cpu().numpy() for x in otoo.otoo_sph_stage1(d_h, d_v, G))
    ng = t.n_groups(G)
    h_adapt_whole = dev((h * np.float32(0.8)).astype(np.float32))
    otoo.otoo_sph_adapt_h(h_adapt_whole, 50.0, 3.0, 30, G)
    h_adapt_whole = h_adapt_whole.cpu().numpy()
    rho_s, dr_s, nn_s = np.zeros(n), np.zeros((n, 4)), np.zeros(n, np.int64)
    h_parts = (h * np.float32(0.8)).astype(np.float32)
    try:
        for b, c in sharded.group_ranges(ng, world):
            otoo.otoo_set_option("group_begin", b)
            otoo.otoo_set_option("group_count", c)
            rho, nn, dr = (x.cpu().numpy() for x in otoo.otoo_sph_stage1(d_h, d_v, G))
            mine = perm[b * G:min((b + c) * G, n)]
            rest = np.setdiff1d(np.arange(n), mine)
            assert np.isfinite(dr).all() and not dr[rest].any() and not rho[rest].any() and not nn[rest].any()
            rho_s += rho; dr_s += dr; nn_s += nn
            d_hp = dev(h_parts)
            otoo.otoo_sph_adapt_h(d_hp, 50.0, 3.0, 30, G)
            hp = d_hp.cpu().numpy()
            assert np.array_equal(hp[rest], h_parts[rest])            # others untouched
            assert np.array_equal(hp[mine].view(np.uint32), h_adapt_whole[mine].view(np.uint32))   # h_i depends on n_i(h_i) alone
    finally:
        otoo.otoo_set_option("group_begin", 0)
        otoo.otoo_set_option("group_count", -1)
    # (a group finished by several warps through the task pool adds its partial sums in another order)
    assert np.array_equal(nn_s, nn_w) and np.allclose(rho_s, rho_w, rtol=2e-6)
    assert np.allclose(dr_s, dr_w, rtol=1e-4, atol=1e-5 * np.abs(dr_w).max())


def test_sorted_output_and_unsort(otoo, orc):
    """option output_sorted + otoo_unsort (what sharded.ShardedGravity exchanges): a range's results are one contiguous
    run of rows in sorted order, zero elsewhere; the runs of all ranges side by side, unsorted, are the plain result."""
    from paper_1206_1199_b200 import sharded, binding
    n, G = 30000 + 17, 128
    pm = gen.plummer(n, 12)
    t = check_tree(otoo, orc, pm, 16)
    perm = t.export()["perm"].astype(np.int64)
    whole = otoo.otoo_gravity(0.01, 0.5, G)
    ng = t.n_groups(G)
    rows = torch.zeros((n, 4), dtype=torch.float32, device="cuda")
    try:
        otoo.otoo_set_option("output_sorted", 1)
        srt = otoo.otoo_gravity(0.01, 0.5, G)
        assert torch.allclose(srt, whole[torch.from_numpy(perm).cuda()], rtol=2e-6, atol=1e-6 * float(whole.abs().max()))
        for b, c in sharded.group_ranges(ng, 3, np.linspace(1, 5, ng)):
            otoo.otoo_set_option("group_begin", b)
            otoo.otoo_set_option("group_count", c)
            part = otoo.otoo_gravity(0.01, 0.5, G)
            lo, hi = b * G, min((b + c) * G, n)
            assert not part[:lo].any() and not part[hi:].any() and bool(part[lo:hi].any())
            rows[lo:hi] = part[lo:hi]
        with pytest.raises(binding.OtooError):                        # the SPH calls have no sorted-output form
            otoo.otoo_sph_density(torch.full((n,), 0.1, device="cuda"), 64)
    finally:
        otoo.otoo_set_option("group_begin", 0)
        otoo.otoo_set_option("group_count", -1)
        otoo.otoo_set_option("output_sorted", 0)
    back = otoo.otoo_unsort(rows)
    assert torch.allclose(back, whole, rtol=2e-6, atol=1e-6 * float(whole.abs().max()))
    sg = sharded.ShardedGravity(otoo)                                 # world 1: the same path end to end
    one = sg.gravity(dev(pm), 16, 0.01, 0.5, G)
    assert torch.allclose(one, whole, rtol=2e-6, atol=1e-6 * float(whole.abs().max()))
    assert sg.cost is not None and sg.cost.shape[0] == ng and sg.cost.is_cuda


def test_walk_profile_and_evaluated_counters(otoo, orc):
    """option walk_profile: the instrumented instantiation of the gravity kernel gives the same counters and fills the
    waiting-time fractions; sum_evaluated = interactions for gravity and <= the candidates for the culled SPH walks."""
    pm = gen.plummer(300000, 9)
    otoo.otoo_build_tree(dev(pm), 16)
    a = otoo.otoo_gravity(0.01, 0.6, 128)
    s0 = otoo.otoo_last_stats()
    assert s0["eval_wait_frac"] == 0 and s0["walker_wait_frac"] == 0 and s0["sum_evaluated"] == s0["sum_interactions"]
    otoo.otoo_set_option("walk_profile", 1)
    try:
        b = otoo.otoo_gravity(0.01, 0.6, 128)
        s1 = otoo.otoo_last_stats()
    finally:
        otoo.otoo_set_option("walk_profile", 0)
    assert s1["sum_interactions"] == s0["sum_interactions"] and s1["sum_tests"] == s0["sum_tests"]
    assert 0 < s1["eval_wait_frac"] < 0.5 and 0 < s1["walker_wait_frac"] < 1 and 0 <= s1["walker_idle_frac"] < 0.5
    assert 1000 < s1["walk_sm_mhz"] < 2500
    assert torch.allclose(a, b, rtol=2e-6, atol=1e-6 * float(a.abs().max()))
    w = gen.wd_pair(50000, 3)
    otoo.otoo_build_tree(dev(w["pos_mass"]), 16)
    otoo.otoo_sph_density(dev(w["h"]), 64)
    s2 = otoo.otoo_last_stats()
    assert 0 < s2["sum_evaluated"] < s2["sum_interactions"]

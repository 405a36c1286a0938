"""otoo_sort_pairs_static (include/otoo.h): the one entry point that allocates nothing -- its scratch is a file-scope
device array of the library -- against the existing path: the (key, id) sort inside otoo_build_tree, whose result
otoo_export_tree returns.  Integer work: bit-exact (tests/test_gpu_parity.py holds the tree build to the same bar).
Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests.

PAPER.md L133 (III-B step 3): "we sort an array of the pair of a key and a particle's id"; ties by original index (R4).
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from workloads import generators as gen

pytestmark = pytest.mark.gpu


def _existing_path(binding, kind, n, seed):
    """sorted keys and permutation of the existing path, and the particles' keys in their original order"""
    pm = gen.make(kind, n, seed)
    o = binding.Otoo(max_particles=n, device=0)
    o.otoo_build_tree(torch.from_numpy(pm).cuda(), 16)
    t = o.otoo_export_tree()
    skeys, perm = t["keys"].astype(np.uint64), t["perm"].astype(np.uint32)
    keys = np.empty(n, dtype=np.uint64)
    keys[perm] = skeys                      # key of particle perm[j] is the j-th sorted key
    return skeys, perm, keys


def test_static_sort_matches_the_build_sort_twice_in_a_row():
    from paper_1206_1199_b200 import binding
    dev = torch.device("cuda", 0)
    cap = 300_001
    # the caller's four buffers, created once (what a graph-capturing caller would do); reused by both calls
    k = torch.empty(cap, dtype=torch.int64, device=dev)
    v = torch.empty(cap, dtype=torch.int32, device=dev)
    k2 = torch.empty_like(k)
    v2 = torch.empty_like(v)
    # two calls in a row, the second smaller and on another distribution: the array keeps the first call's contents,
    # so stale histograms, tickets or status words would show here (74 tiles with a ragged tail, then 18)
    for kind, n, seed in (("plummer", 300_001, 1206), ("uniform_cube", 70_001, 1199)):
        skeys, perm, keys = _existing_path(binding, kind, n, seed)
        k[:n].copy_(torch.from_numpy(keys.view(np.int64)))
        v[:n].copy_(torch.arange(n, dtype=torch.int32))
        binding.otoo_sort_pairs_static(k, v, k2, v2, n=n)
        torch.cuda.synchronize()
        got_k = k[:n].cpu().numpy().view(np.uint64)
        got_v = v[:n].cpu().numpy().view(np.uint32)
        assert np.array_equal(got_k, skeys), (kind, n)
        assert np.array_equal(got_v, perm), (kind, n)          # stable: ties keep the original index order (R4)
    # and the same input again gives the same output (nothing carried from call to call)
    k[:n].copy_(torch.from_numpy(keys.view(np.int64)))
    v[:n].copy_(torch.arange(n, dtype=torch.int32))
    binding.otoo_sort_pairs_static(k, v, k2, v2, n=n)
    torch.cuda.synchronize()
    assert np.array_equal(k[:n].cpu().numpy().view(np.uint64), skeys)
    assert np.array_equal(v[:n].cpu().numpy().view(np.uint32), perm)


def test_static_sort_full_64_bit_keys_and_edges():
    """keys with the top bit set, all-equal keys (ties by id), n = 1, n = 0; against numpy's stable sort"""
    from paper_1206_1199_b200 import binding
    dev = torch.device("cuda", 0)
    rng = np.random.default_rng(2012)
    for n, mode in ((4097, "random"), (9000, "equal"), (1, "random"), (0, "random")):
        keys = rng.integers(0, 2 ** 64, size=n, dtype=np.uint64) if mode == "random" else np.full(n, 7, dtype=np.uint64)
        k = torch.from_numpy(keys.view(np.int64).copy()).to(dev)
        v = torch.arange(n, dtype=torch.int32, device=dev)
        binding.otoo_sort_pairs_static(k, v, torch.empty_like(k), torch.empty_like(v))
        torch.cuda.synchronize()
        order = np.argsort(keys, kind="stable")
        assert np.array_equal(k.cpu().numpy().view(np.uint64), keys[order])
        assert np.array_equal(v.cpu().numpy().view(np.uint32), order.astype(np.uint32))


def test_static_sort_rejects_sizes_beyond_its_scratch():
    from paper_1206_1199_b200 import binding
    dev = torch.device("cuda", 0)
    n = binding.SORT_STATIC_MAX_PAIRS + 1
    k = torch.zeros(n, dtype=torch.int64, device=dev)
    v = torch.zeros(n, dtype=torch.int32, device=dev)
    with pytest.raises(binding.OtooError) as e:
        binding.otoo_sort_pairs_static(k, v, torch.empty_like(k), torch.empty_like(v))
    assert e.value.status == 5 and "OTOO_SORT_STATIC_MAX_PAIRS" in str(e.value)      # OTOO_ERR_CAPACITY
    # the maximum itself is accepted
    n = binding.SORT_STATIC_MAX_PAIRS
    keys = np.random.default_rng(1).integers(0, 2 ** 63, size=n, dtype=np.uint64)
    k = torch.from_numpy(keys.view(np.int64).copy()).to(dev)
    v = torch.arange(n, dtype=torch.int32, device=dev)
    binding.otoo_sort_pairs_static(k, v, torch.empty_like(k), torch.empty_like(v))
    torch.cuda.synchronize()
    got = k.cpu().numpy().view(np.uint64)
    assert np.array_equal(got, np.sort(keys))

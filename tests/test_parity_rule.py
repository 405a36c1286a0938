"""CPU checks of the floating-point parity rule itself (tests/parity_rule.py, R12)."""
import numpy as np

from tests.parity_rule import TOL, U32, phi_tol


def test_phi_tol_is_1e5_for_every_list_of_the_default_walk():
    assert phi_tol(0) == TOL and phi_tol(28_000) == TOL and phi_tol(1_700_000) == TOL
    assert phi_tol(64 * (TOL / U32) ** 2) == TOL                       # the crossover: 1.8 M entries
    assert 2.0e-5 < phi_tol(8_265_352) < 2.3e-5                        # C3's system-sized group under group_distance = 0


def test_two_level_fp32_sum_of_like_signed_terms_stays_inside_phi_tol():
    """The arithmetic the bound is derived from, in numpy: 64-entry fp32 partial sums added one after the other to an
    fp32 total (the kernel's order, without its split over pool tasks, which only shortens the chains), against the
    fp64 sum, for a short list and for one as long as C3's worst.  The long one does not promise 1e-5."""
    rng = np.random.default_rng(1206)
    worst = {}
    for L in (28_672, 8_265_344):
        errs = []
        for _ in range(6):
            x = (rng.random(L, dtype=np.float32) + np.float32(0.25)) * np.float32(1e-3)
            partial = x.reshape(-1, 64).astype(np.float32).sum(axis=1, dtype=np.float32)
            total = np.cumsum(partial, dtype=np.float32)[-1]           # sequential fp32 accumulation
            exact = x.astype(np.float64).sum()
            errs.append(abs(float(total) - exact) / exact)
        worst[L] = max(errs)
        assert worst[L] <= phi_tol(L), (L, worst[L])
    assert worst[28_672] < 2e-6
    assert worst[8_265_344] > 1e-6                                     # three orders more additions: visibly worse

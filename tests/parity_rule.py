"""The floating-point parity rule of DESIGN.md section 7 (reading R12), in ONE place: the GPU parity tests and
__graft_entry__.smoke() both call it, and every call reports the numbers SURVEY 8(c) R12 asks for.

Per particle i, for a vector output x (acceleration, SPH force, (rot v)) or a scalar one (du/dt, div v):
    |dx_i| <= max(1e-5 |x_i|, 8 u A_i),   u = 2^-24,   A_i = sum_j |x_ij|  (the oracle's sum of pair-term
magnitudes over the same list -- pinned against numpy brute force in tests/test_oracle_abs_sum.py), and
    |dx_i| / |x_i| <= 1e-5  at the `pct`-th percentile (plain relative error, no floor; pct = None: not asserted).
Reported (printed, and appended to gpurun_out/parity_report.jsonl when that directory exists): the un-floored
maximum, p99.9 and median of |dx_i|/|x_i|; the maximum of |dx_i| over its bound; the fraction of particles whose
bound is the 8 u A_i floor (A_i/|x_i| > 1e-5/(8u) = 21); and the same error under SURVEY's own floor,
|dx_i| / max(|x_i|, 1e-2 x_rms).  `floor_frac_max` bounds the floor fraction and `above_tol_frac_max` the fraction
of particles whose plain relative error exceeds 1e-5: a test states how many particles it lets live on the floor."""
import json
import os

import numpy as np

TOL = 1e-5
U32 = 2.0 ** -24
FLOOR_RATIO = TOL / (8 * U32)        # A_i / |x_i| above which the floor is the bound (= 20.97)
# Measured on the B200 (profiles/r2_parity_audit.md): gravity has <= 0.4 % of the particles on the floor in every
# test (0.00 % at C5), the SPH pressure force <= 2.2 %, and <= 2 particles per test exceed plain 1e-5.  The tests
# assert these with a margin; a regression of the arithmetic shows up here before it reaches the bound.
FLOOR_FRAC_MAX_GRAVITY = 0.01
FLOOR_FRAC_MAX_SPH = 0.04
ABOVE_TOL_FRAC_MAX = 5e-4            # fraction of particles whose plain relative error may exceed 1e-5 (they are held by 8 u A)
_ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _norm(a):
    a = np.asarray(a, dtype=np.float64)
    return np.abs(a) if a.ndim == 1 else np.linalg.norm(a, axis=1)


def report(label, got, want, abs_sum, pct=99.9, floor_frac_max=FLOOR_FRAC_MAX_SPH, above_tol_frac_max=ABOVE_TOL_FRAC_MAX, check=True):
    """got, want: (n,) or (n,k) arrays; abs_sum: (n,).  Returns the statistics; asserts the rule if check."""
    got, want = np.asarray(got, dtype=np.float64), np.asarray(want, dtype=np.float64)
    d = _norm(got - want)
    xn = _norm(want)
    A = np.asarray(abs_sum, dtype=np.float64)
    bound = np.maximum(TOL * xn, 8 * U32 * A)
    rel = d / np.maximum(xn, 1e-300)
    rel = np.where((xn == 0) & (d == 0), 0.0, rel)
    rms = np.sqrt((xn ** 2).mean()) if len(xn) else 0.0
    st = dict(label=label, n=int(len(xn)),
              unfloored_max=float(rel.max()) if len(rel) else 0.0,
              p999=float(np.percentile(rel, 99.9)) if len(rel) else 0.0,
              p99=float(np.percentile(rel, 99)) if len(rel) else 0.0,
              median=float(np.median(rel)) if len(rel) else 0.0,
              max_over_bound=float((d / np.maximum(bound, 1e-300)).max()) if len(d) else 0.0,
              floor_frac=float((8 * U32 * A > TOL * xn).mean()) if len(xn) else 0.0,
              n_above_tol=int((rel > TOL).sum()),
              survey_floor_max=float((d / np.maximum(xn, 1e-2 * rms + 1e-300)).max()) if len(d) else 0.0)
    print("parity %(label)s: n=%(n)d un-floored max %(unfloored_max).2e p99.9 %(p999).2e median %(median).2e | "
          "max |dx|/bound %(max_over_bound).3f | on the 8uA floor %(floor_frac).4f | above 1e-5: %(n_above_tol)d | "
          "SURVEY floor (1e-2 rms) max %(survey_floor_max).2e" % st)
    out = os.path.join(_ROOT, "gpurun_out")
    if os.path.isdir(out):
        with open(os.path.join(out, "parity_report.jsonl"), "a") as f:
            f.write(json.dumps(st) + "\n")
    if check:
        assert st["max_over_bound"] <= 1.0, st
        if pct is not None:      # None: sums that cancel for most particles (div v, du/dt) are held by the bound alone
            assert float(np.percentile(rel, pct)) <= TOL, st
        assert st["floor_frac"] <= floor_frac_max, st
        assert st["n_above_tol"] <= max(2, above_tol_frac_max * st["n"]), st
    return st


def phi_tol(list_len):
    """Tolerance of the potential of a target whose interaction list has `list_len` entries (R12).
    phi is a sum of terms of one sign, so its error is pure rounding: plain 1e-5 relative, as long as fp32 arithmetic
    can promise it.  The kernel adds 64-entry partial sums to running totals (and the totals of a group's pool tasks
    to the output): L/64 fp32 additions of like-signed partials, each off by <= u/2 of the running total, a random walk
    of about u sqrt(L/64) at a few sigma.  That passes 1e-5 at L = 64 (1e-5/u)^2 = 1.8 M entries: the bound is
        max(1e-5, u sqrt(L/64)),
    1e-5 for every list of the default walk (longest: 28 k entries at C2) and 2.1e-5 for the ONE group of C3 that lists
    all 8.4 M particles under group_distance = 0 (measured on the B200 over 20 runs: 6.8e-6 ... 1.14e-5)."""
    L = np.asarray(list_len, dtype=np.float64)
    return np.maximum(TOL, U32 * np.sqrt(L / 64.0))


def scalar_rel(label, got, want, tol=TOL):
    """plain relative error of a positive-definite scalar sum (potential, density): max |dx|/|x| <= tol"""
    got, want = np.asarray(got, dtype=np.float64), np.asarray(want, dtype=np.float64)
    e = np.abs(got - want) / np.abs(want)
    print("parity %s: n=%d max rel %.2e median %.2e" % (label, len(e), e.max(), np.median(e)))
    assert e.max() <= tol, (label, float(e.max()))
    return float(e.max())

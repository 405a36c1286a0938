"""ctypes binding of the CPU oracle (oracle/otoo_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It imports nothing from the product package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = os.path.join(_HERE, "otoo_oracle.c")

CELL_DTYPE = np.dtype([("prefix", "<u8"), ("first", "<u4"), ("count", "<u4"), ("child_first", "<u4"),
                       ("level", "u1"), ("child_count", "u1")], align=True)
assert CELL_DTYPE.itemsize == 24


def build(force: bool = False) -> str:
    """Compile liboracle.so (gcc, -ffp-contract=off) if missing or stale."""
    hdr = os.path.join(_HERE, "otoo_oracle.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(_SRC), os.path.getmtime(hdr))):
        return _SO
    cmd = ["gcc", "-O2", "-std=c99", "-D_GNU_SOURCE", "-fopenmp", "-ffp-contract=off", "-fPIC",
           "-shared", "-o", _SO, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        L = _lib
        vp, i64, i32, dbl = C.c_void_p, C.c_int64, C.c_int, C.c_double
        L.orc_build.restype = vp
        L.orc_build.argtypes = [i64, vp, i32]
        L.orc_build_ord.restype = vp
        L.orc_build_ord.argtypes = [i64, vp, i32, i32]
        L.orc_hilbert_key.restype = C.c_uint64
        L.orc_hilbert_key.argtypes = [vp]
        L.orc_hilbert_coords.argtypes = [C.c_uint64, vp]
        L.orc_free.argtypes = [vp]
        L.orc_ncell.restype = i64
        L.orc_ncell.argtypes = [vp]
        L.orc_nleaf.restype = i64
        L.orc_nleaf.argtypes = [vp]
        L.orc_depth.restype = i32
        L.orc_depth.argtypes = [vp]
        L.orc_root.argtypes = [vp, vp, vp]
        L.orc_export.argtypes = [vp] * 7
        L.orc_key.restype = C.c_uint64
        L.orc_key.argtypes = [vp, vp]
        L.orc_rb2.argtypes = [vp, dbl, i32, vp]
        L.orc_direct_sum.argtypes = [i64, vp, dbl, i64, vp, vp]
        L.orc_gravity.restype = C.c_uint64
        L.orc_gravity.argtypes = [vp, dbl, dbl, i32, i32, i32, vp, vp, vp, vp, vp]
        L.orc_delta_cell_props.argtypes = [vp, vp, vp]
        L.orc_B2_direct.restype = dbl
        L.orc_B2_direct.argtypes = [vp, i64]
        L.orc_rb2_delta.argtypes = [vp, dbl, dbl, vp]
        L.orc_gravity_rb2.restype = C.c_uint64
        L.orc_gravity_rb2.argtypes = [vp, dbl, vp, i32, i32, vp, i64, vp, vp, vp, vp, vp]
        L.orc_gravity_sel.restype = C.c_uint64
        L.orc_gravity_sel.argtypes = [vp, dbl, dbl, i32, i32, i32, vp, i64, vp, vp, vp, vp, vp]
        L.orc_sph_density_sel.restype = C.c_uint64
        L.orc_sph_density_sel.argtypes = [vp, vp, i32, vp, i64, vp, vp, vp, vp]
        L.orc_sph_force_visc_sel.restype = C.c_uint64
        L.orc_sph_force_visc_sel.argtypes = [vp, vp, vp, vp, vp, vp, i32, vp, i64, vp, vp]
        L.orc_sph_force_sel.restype = C.c_uint64
        L.orc_sph_force_sel.argtypes = [vp, vp, vp, vp, vp, i32, vp, i64, vp, vp]
        L.orc_group_lists.argtypes = [vp, dbl, i32, i32, i64, vp, vp]
        L.orc_group_lists_rb2.argtypes = [vp, vp, i32, i64, vp, vp]
        L.orc_sph_cell_radii.argtypes = [vp, vp, vp, vp]
        L.orc_sph_density.restype = C.c_uint64
        L.orc_sph_density.argtypes = [vp, vp, i32, vp, vp, vp, vp]
        L.orc_sph_group_list.argtypes = [vp, vp, i32, i64, vp]
        L.orc_sph_divrot_sel.restype = C.c_uint64
        L.orc_sph_divrot_sel.argtypes = [vp, vp, vp, i32, vp, i64, vp, vp, vp]
        L.orc_sph_adapt_h.restype = i32
        L.orc_sph_adapt_h.argtypes = [vp, vp, dbl, dbl, i32, i32, vp]
        L.orc_sph_force.restype = C.c_uint64
        L.orc_sph_force.argtypes = [vp, vp, vp, vp, vp, i32, vp, vp]
        L.orc_W.restype = dbl
        L.orc_W.argtypes = [dbl, dbl]
        L.orc_dWdr.restype = dbl
        L.orc_dWdr.argtypes = [dbl, dbl]
        L.orc_set_dist_kind.argtypes = [vp, i32]
        L.orc_set_split_pieces.argtypes = [vp, i32]
        L.orc_max_threads.restype = i32
        L.orc_set_threads.argtypes = [i32]
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float32)
    if shape is not None:
        assert a.shape == shape, (a.shape, shape)
    return a


def max_threads() -> int:
    return lib().orc_max_threads()


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


def direct_sum(pos_mass, eps, targets=None):
    pm = _f32(pos_mass)
    n = pm.shape[0]
    if targets is None:
        out = np.empty((n, 4), dtype=np.float64)
        lib().orc_direct_sum(n, _p(pm), float(eps), 0, None, _p(out))
    else:
        tg = np.ascontiguousarray(targets, dtype=np.int64)
        out = np.empty((len(tg), 4), dtype=np.float64)
        lib().orc_direct_sum(n, _p(pm), float(eps), len(tg), _p(tg), _p(out))
    return out


def W(r, h):
    return lib().orc_W(float(r), float(h))


def dWdr(r, h):
    return lib().orc_dWdr(float(r), float(h))


def hilbert_key(q):
    """63-bit Hilbert key of 21-bit integer coordinates (x, y, z)"""
    a = np.ascontiguousarray(q, dtype=np.uint32)
    assert a.shape == (3,)
    return int(lib().orc_hilbert_key(_p(a)))


def hilbert_coords(key):
    out = np.zeros(3, dtype=np.uint32)
    lib().orc_hilbert_coords(C.c_uint64(int(key)), _p(out))
    return out


class Tree:
    """Oracle tree: PAPER.md III-B (build) + III-C (cell properties)."""

    def __init__(self, pos_mass, n_crit=16, key_order=0):
        """key_order 0: Morton keys (R3); 1: Hilbert keys (reading R20)"""
        self.pm = _f32(pos_mass)
        assert self.pm.ndim == 2 and self.pm.shape[1] == 4
        self.N = self.pm.shape[0]
        self.n_crit = int(n_crit)
        self.key_order = int(key_order)
        self._h = lib().orc_build_ord(self.N, _p(self.pm), self.n_crit, self.key_order)
        self.ncell = lib().orc_ncell(self._h)
        self.nleaf = lib().orc_nleaf(self._h)
        self.depth = lib().orc_depth(self._h)
        lo = np.empty(3, dtype=np.float32)
        S = np.empty(1, dtype=np.float32)
        lib().orc_root(self._h, _p(lo), _p(S))
        self.lo, self.S = lo, float(S[0])

    def __del__(self):
        try:
            if self._h:
                lib().orc_free(self._h)
                self._h = None
        except Exception:
            pass

    def export(self):
        perm = np.empty(self.N, dtype=np.uint32)
        keys = np.empty(self.N, dtype=np.uint64)
        cells = np.zeros(self.ncell, dtype=CELL_DTYPE)
        com_m = np.empty((self.ncell, 4), dtype=np.float32)
        s = np.empty(self.ncell, dtype=np.float64)
        MP = np.empty((self.ncell, 4), dtype=np.float64)
        lib().orc_export(self._h, _p(perm), _p(keys), _p(cells), _p(com_m), _p(s), _p(MP))
        return dict(perm=perm, keys=keys, cells=cells, com_m=com_m, s=s, MP=MP)

    def key(self, xyz):
        a = _f32(xyz, (3,))
        return int(lib().orc_key(self._h, _p(a)))

    def rb2(self, theta, mac_kind=0):
        out = np.empty(self.ncell, dtype=np.float32)
        lib().orc_rb2(self._h, float(theta), int(mac_kind), _p(out))
        return out

    def set_dist_kind(self, kind):
        """2 (default): boxes of the group's pieces (R25; SPH: R26); 0: one box per group (R8, R15);
        1: exact minimum over the group's members (R23; SPH walks then use one box)"""
        lib().orc_set_dist_kind(self._h, int(kind))

    def set_split_pieces(self, K):
        lib().orc_set_split_pieces(self._h, int(K))

    def delta_cell_props(self):
        """(B2, b_max) per cell in fp64: PAPER.md Eq. 2 (bottom-up, reading R19) and L63."""
        B2 = np.empty(self.ncell, dtype=np.float64)
        bm = np.empty(self.ncell, dtype=np.float64)
        lib().orc_delta_cell_props(self._h, _p(B2), _p(bm))
        return B2, bm

    def B2_direct(self, cell):
        return lib().orc_B2_direct(self._h, int(cell))

    def rb2_delta(self, delta, m_limit=np.inf):
        """rb^2 (fp32) of the paper's absolute-error MAC, Eq. 1, with the m_limit rule of L157."""
        out = np.empty(self.ncell, dtype=np.float32)
        lib().orc_rb2_delta(self._h, float(delta), float(m_limit), _p(out))
        return out

    def n_groups(self, G):
        return (self.N + G - 1) // G

    def gravity(self, eps, theta, group_size, mac_kind=0, walk_kind=0, forces=True, groups=None, rb2=None):
        """groups: optional array of group indices; then only those are walked, the counters are indexed
        by position in `groups`, and acc_pot / abs_sum (still N rows) are filled for their targets only."""
        sel = None if groups is None else np.ascontiguousarray(groups, dtype=np.int64)
        ng = self.n_groups(group_size) if sel is None else len(sel)
        acc = np.zeros((self.N, 4), dtype=np.float64) if forces else None
        nt = np.zeros(ng, dtype=np.uint32)
        nc = np.zeros(ng, dtype=np.uint32)
        npart = np.zeros(ng, dtype=np.uint32)
        asum = np.zeros(self.N, dtype=np.float64) if forces else None
        if rb2 is not None:       # any MAC of the form "accept iff d > r_b": theta is ignored
            rb2 = np.ascontiguousarray(rb2, dtype=np.float32)
            assert rb2.shape == (self.ncell,)
            tot = lib().orc_gravity_rb2(self._h, float(eps), _p(rb2), int(group_size), int(walk_kind), _p(sel),
                                        0 if sel is None else len(sel), _p(acc), _p(nt), _p(nc), _p(npart), _p(asum))
        else:
            tot = lib().orc_gravity_sel(self._h, float(eps), float(theta), int(group_size), int(mac_kind),
                                        int(walk_kind), _p(sel), 0 if sel is None else len(sel),
                                        _p(acc), _p(nt), _p(nc), _p(npart), _p(asum))
        return dict(acc_pot=acc, n_tests=nt, n_cells=nc, n_parts=npart, interactions=int(tot), abs_sum=asum)

    def group_targets(self, group_size, groups):
        """original particle indices of the members of the given groups (sorted slots -> perm)"""
        perm = self.export()["perm"] if not hasattr(self, "_perm") else self._perm
        self._perm = perm
        out = []
        for g in np.asarray(groups, dtype=np.int64):
            out.append(perm[g * group_size:min((g + 1) * group_size, self.N)])
        return np.concatenate(out).astype(np.int64)

    def group_lists(self, theta, group_size, g, n_cells, n_parts, mac_kind=0):
        """theta-MAC lists of one group (for other MACs use group_lists_rb2)"""
        cells = np.empty(max(int(n_cells), 1), dtype=np.uint32)
        parts = np.empty(max(int(n_parts), 1), dtype=np.uint32)
        lib().orc_group_lists(self._h, float(theta), int(group_size), int(mac_kind), int(g),
                              _p(cells), _p(parts))
        return cells[:int(n_cells)], parts[:int(n_parts)]

    def group_lists_rb2(self, rb2, group_size, g, n_cells, n_parts):
        rb2 = np.ascontiguousarray(rb2, dtype=np.float32)
        cells = np.empty(max(int(n_cells), 1), dtype=np.uint32)
        parts = np.empty(max(int(n_parts), 1), dtype=np.uint32)
        lib().orc_group_lists_rb2(self._h, _p(rb2), int(group_size), int(g), _p(cells), _p(parts))
        return cells[:int(n_cells)], parts[:int(n_parts)]

    def sph_cell_radii(self, h):
        h = _f32(h, (self.N,))
        b = np.empty(self.ncell, dtype=np.float32)
        r = np.empty(self.ncell, dtype=np.float32)
        lib().orc_sph_cell_radii(self._h, _p(h), _p(b), _p(r))
        return b, r

    def sph_density(self, h, group_size, sums=True, groups=None):
        h = _f32(h, (self.N,))
        sel = None if groups is None else np.ascontiguousarray(groups, dtype=np.int64)
        ng = self.n_groups(group_size) if sel is None else len(sel)
        rho = np.zeros(self.N, dtype=np.float64) if sums else None
        nngb = np.zeros(self.N, dtype=np.uint32)
        nt = np.zeros(ng, dtype=np.uint32)
        npart = np.zeros(ng, dtype=np.uint32)
        tot = lib().orc_sph_density_sel(self._h, _p(h), int(group_size), _p(sel), 0 if sel is None else len(sel),
                                        _p(rho), _p(nngb), _p(nt), _p(npart))
        return dict(rho=rho, nngb=nngb, n_tests=nt, n_parts=npart, candidates=int(tot))

    def sph_divrot(self, h, vel, group_size, groups=None):
        """SPH stage 1 with velocity derivatives (reading R22): rho, (div v, rot v) per particle, caller's order"""
        h = _f32(h, (self.N,))
        v = _f32(vel, (self.N, 4))
        sel = None if groups is None else np.ascontiguousarray(groups, dtype=np.int64)
        rho = np.zeros(self.N, dtype=np.float64)
        out = np.zeros((self.N, 4), dtype=np.float64)
        asum = np.zeros(self.N, dtype=np.float64)
        tot = lib().orc_sph_divrot_sel(self._h, _p(h), _p(v), int(group_size), _p(sel), 0 if sel is None else len(sel),
                                       _p(rho), _p(out), _p(asum))
        return dict(rho=rho, divrot=out, abs_sum=asum, candidates=int(tot))

    def sph_adapt_h(self, h, n_target, tol, max_iter, group_size):
        """reading R21: returns (h after the iteration, neighbour counts of that h, iterations done)"""
        h = _f32(h, (self.N,)).copy()
        nngb = np.zeros(self.N, dtype=np.uint32)
        it = lib().orc_sph_adapt_h(self._h, _p(h), float(n_target), float(tol), int(max_iter), int(group_size), _p(nngb))
        return h, nngb, int(it)

    def sph_group_list(self, h, group_size, g, n_parts):
        h = _f32(h, (self.N,))
        parts = np.empty(max(int(n_parts), 1), dtype=np.uint32)
        lib().orc_sph_group_list(self._h, _p(h), int(group_size), int(g), _p(parts))
        return parts[:int(n_parts)]

    def sph_force(self, h, rho, P, group_size, vel=None, groups=None, visc=None):
        """visc: optional (N,4) fp32 (sound speed c, alpha, Balsara f, -): artificial viscosity, reading R24 (needs vel)"""
        h = _f32(h, (self.N,))
        rho = np.ascontiguousarray(rho, dtype=np.float64)
        P = np.ascontiguousarray(P, dtype=np.float64)
        v = None if vel is None else _f32(vel, (self.N, 4))
        out = np.zeros((self.N, 4), dtype=np.float64)
        asum = np.zeros((self.N, 2), dtype=np.float64)
        sel = None if groups is None else np.ascontiguousarray(groups, dtype=np.int64)
        if visc is not None:
            assert v is not None
            q = _f32(visc, (self.N, 4))
            tot = lib().orc_sph_force_visc_sel(self._h, _p(h), _p(rho), _p(P), _p(v), _p(q), int(group_size), _p(sel),
                                               0 if sel is None else len(sel), _p(out), _p(asum))
        else:
            tot = lib().orc_sph_force_sel(self._h, _p(h), _p(rho), _p(P), _p(v), int(group_size), _p(sel),
                                          0 if sel is None else len(sel), _p(out), _p(asum))
        return dict(acc_dudt=out, candidates=int(tot), abs_sum=asum)

"""Thin Python binding of libotoo.so (include/otoo.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; torch is used for device memory
and streams.  There is no CPU fallback: if the library is missing, import fails loudly.
Function names mirror the C-ABI.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libotoo.so")
if not os.path.exists(_LIB_PATH):
    raise ImportError(f"{_LIB_PATH} is missing: run `python -m paper_1206_1199_b200.build` "
                      "(nvcc, sm_100a). There is no CPU fallback.")
_lib = C.CDLL(_LIB_PATH)

OTOO_OK, OTOO_ERR_INVALID_ARG, OTOO_ERR_OOM, OTOO_ERR_CUDA, OTOO_ERR_NOT_BUILT, OTOO_ERR_CAPACITY = range(6)
STATUS_NAMES = ["OTOO_OK", "OTOO_ERR_INVALID_ARG", "OTOO_ERR_OOM", "OTOO_ERR_CUDA", "OTOO_ERR_NOT_BUILT",
                "OTOO_ERR_CAPACITY"]

EXPORTS = ["otoo_version", "otoo_create", "otoo_destroy", "otoo_last_error", "otoo_build_tree", "otoo_gravity",
           "otoo_sph_density", "otoo_sph_force", "otoo_eos_ideal", "otoo_tree_info", "otoo_export_tree",
           "otoo_export_sph_radii", "otoo_export_group_stats", "otoo_last_stats", "otoo_set_option",
           "otoo_gravity_host", "otoo_gravity_delta_host", "otoo_gravity_delta", "otoo_measure_fp32_peak", "otoo_probe", "otoo_unsort", "otoo_sph_adapt_h", "otoo_sph_stage1", "otoo_sph_force_visc",
           "otoo_sort_pairs_static"]


class TreeInfo(C.Structure):
    _fields_ = [("N", C.c_int64), ("N_cell", C.c_int64), ("N_leaf", C.c_int64), ("depth", C.c_int32),
                ("lo", C.c_float * 3), ("S", C.c_float)]


class Stats(C.Structure):
    _fields_ = [("sum_tests", C.c_uint64), ("sum_interactions", C.c_uint64), ("sum_cells", C.c_uint64),
                ("sum_parts", C.c_uint64), ("n_groups", C.c_int64), ("group_size", C.c_int32),
                ("launches", C.c_int32), ("sum_steps", C.c_uint64), ("sum_tasks", C.c_uint64),
                ("sum_flushes", C.c_uint64), ("sum_evaluated", C.c_uint64), ("ms_build", C.c_float * 8), ("ms_build_total", C.c_float),
                ("ms_walk_prep", C.c_float), ("ms_walk_force", C.c_float), ("ms_total", C.c_float),
                ("walk_sm_mhz", C.c_float), ("eval_wait_frac", C.c_float), ("walker_wait_frac", C.c_float),
                ("walker_idle_frac", C.c_float), ("walk_only", C.c_int32), ("error_flag", C.c_int32)]


BUILD_PHASES = ["root_cube", "keys", "sort", "gather", "cells", "moments"]


CELL_DTYPE = np.dtype([("prefix", "<u8"), ("first", "<u4"), ("count", "<u4"), ("child_first", "<u4"),
                       ("level", "u1"), ("child_count", "u1")], align=True)

_vp, _i64, _i32, _f = C.c_void_p, C.c_int64, C.c_int, C.c_float
_lib.otoo_version.restype = _i32
_lib.otoo_create.argtypes = [C.POINTER(_vp), _i32, _i64]
_lib.otoo_destroy.argtypes = [_vp]
_lib.otoo_destroy.restype = None
_lib.otoo_last_error.argtypes = [_vp]
_lib.otoo_last_error.restype = C.c_char_p
_lib.otoo_build_tree.argtypes = [_vp, _vp, _i64, _i32, _vp]
_lib.otoo_gravity.argtypes = [_vp, _f, _f, _i32, _vp, _vp]
_lib.otoo_gravity_delta.argtypes = [_vp, _f, _f, _f, _i32, _vp, _vp]
_lib.otoo_sph_density.argtypes = [_vp, _vp, _i32, _vp, _vp, _vp]
_lib.otoo_sph_force_visc.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _i32, _vp, _vp]
_lib.otoo_sph_stage1.argtypes = [_vp, _vp, _vp, _i32, _vp, _vp, _vp, _vp]
_lib.otoo_sph_adapt_h.argtypes = [_vp, _vp, _f, _f, _i32, _i32, _vp, C.POINTER(C.c_int), _vp]
_lib.otoo_sph_force.argtypes = [_vp, _vp, _vp, _vp, _vp, _i32, _vp, _vp]
_lib.otoo_eos_ideal.argtypes = [_vp, _vp, _vp, _f, _i64, _vp, _vp]
_lib.otoo_tree_info.argtypes = [_vp, C.POINTER(TreeInfo)]
_lib.otoo_export_tree.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp]
_lib.otoo_export_sph_radii.argtypes = [_vp, _vp, _vp]
_lib.otoo_export_group_stats.argtypes = [_vp, _vp, _vp, _vp]
_lib.otoo_last_stats.argtypes = [_vp, C.POINTER(Stats)]
_lib.otoo_set_option.argtypes = [_vp, C.c_char_p, _i64]
_lib.otoo_measure_fp32_peak.argtypes = [_vp, C.POINTER(C.c_double), _vp]
_lib.otoo_unsort.argtypes = [_vp, _vp, _vp, _vp]
_lib.otoo_probe.argtypes = [_vp, C.c_char_p, C.c_char_p, _i64, _vp]
_lib.otoo_gravity_host.argtypes = [_vp, _vp, _i64, _i32, _f, _f, _i32, _vp]
_lib.otoo_gravity_delta_host.argtypes = [_vp, _vp, _i64, _i32, _f, _f, _f, _i32, _vp]
_lib.otoo_sort_pairs_static.argtypes = [_vp, _vp, _vp, _vp, _i64, _vp, C.c_char_p, _i64]
SORT_STATIC_MAX_PAIRS = 2097152      # OTOO_SORT_STATIC_MAX_PAIRS of include/otoo.h


class OtooError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < 6 else status}: {msg}")
        self.status = status


def _ptr(t, dtype=None, shape_last=None, rows=None, device=None):
    """data_ptr() of a contiguous CUDA tensor after the checks the C side cannot make: dtype, (N, k) shape, the row
    count the kernels will read or write, and the device of the context."""
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda or not t.is_contiguous():
        raise TypeError("expected a contiguous CUDA torch.Tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    if shape_last is not None and (t.ndim != 2 or t.shape[1] != shape_last):
        raise TypeError(f"expected shape (N,{shape_last})")
    if rows is not None and t.shape[0] != rows:
        raise ValueError(f"expected {rows} rows, got {t.shape[0]}")
    if device is not None and t.device.index != device:
        raise ValueError(f"tensor on cuda:{t.device.index}, context on cuda:{device}")
    return t.data_ptr()


class Otoo:
    """One context per GPU (otoo_create / otoo_destroy)."""

    def __init__(self, max_particles: int, device: int = 0):
        self._h = _vp()
        self.device = device
        st = _lib.otoo_create(C.byref(self._h), int(device), int(max_particles))
        if st != OTOO_OK:
            raise OtooError(st, "otoo_create failed")
        self.N = 0

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            _lib.otoo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st):
        if st != OTOO_OK:
            raise OtooError(st, _lib.otoo_last_error(self._h).decode())

    def _dev(self):
        return torch.device("cuda", self.device)

    def _stream(self, stream):
        if stream is None:
            return torch.cuda.current_stream(self.device).cuda_stream
        return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)

    def _p(self, t, dtype=None, shape_last=None):
        """a per-particle argument: N rows on this context's device (before a build the C side answers NOT_BUILT)"""
        return _ptr(t, dtype, shape_last, rows=self.N if self.N else None, device=self.device)

    # ---- the hot path
    def otoo_build_tree(self, pos_mass, n_crit=16, stream=None):
        n = 0 if pos_mass is None else pos_mass.shape[0]
        self._check(_lib.otoo_build_tree(self._h, _ptr(pos_mass, torch.float32, 4, device=self.device) if n else None, n, int(n_crit),
                                         self._stream(stream)))
        self.N = n

    def otoo_gravity(self, eps, theta, group_size, out=None, stream=None):
        if out is None:
            out = torch.empty((self.N, 4), dtype=torch.float32, device=self._dev())
        self._check(_lib.otoo_gravity(self._h, float(eps), float(theta), int(group_size),
                                      self._p(out, torch.float32, 4), self._stream(stream)))
        return out

    def otoo_gravity_delta(self, eps, delta, m_limit, group_size, out=None, stream=None):
        if out is None:
            out = torch.empty((self.N, 4), dtype=torch.float32, device=self._dev())
        self._check(_lib.otoo_gravity_delta(self._h, float(eps), float(delta), float(m_limit), int(group_size),
                                            self._p(out, torch.float32, 4), self._stream(stream)))
        return out

    def otoo_sph_density(self, h, group_size, want_nngb=True, stream=None):
        rho = torch.empty(self.N, dtype=torch.float32, device=self._dev())
        nngb = torch.empty(self.N, dtype=torch.int32, device=self._dev()) if want_nngb else None
        self._check(_lib.otoo_sph_density(self._h, self._p(h, torch.float32), int(group_size), self._p(rho),
                                          self._p(nngb), self._stream(stream)))
        return rho, nngb

    def otoo_sph_force_visc(self, h, rho, P, vel, visc, group_size, stream=None):
        """pressure force + artificial viscosity + du/dt; visc = (N,4) fp32 (c, alpha, Balsara f, -)"""
        out = torch.empty((self.N, 4), dtype=torch.float32, device=self._dev())
        self._check(_lib.otoo_sph_force_visc(self._h, self._p(h, torch.float32), self._p(rho, torch.float32), self._p(P, torch.float32),
                                             self._p(vel, torch.float32, 4), self._p(visc, torch.float32, 4), int(group_size),
                                             out.data_ptr(), self._stream(stream)))
        return out

    def otoo_sph_stage1(self, h, vel, group_size, stream=None):
        """density, neighbour counts and (div v, rot v): returns (rho, nngb, divrot)"""
        rho = torch.empty(self.N, dtype=torch.float32, device=self._dev())
        nngb = torch.empty(self.N, dtype=torch.int32, device=self._dev())
        dr = torch.empty((self.N, 4), dtype=torch.float32, device=self._dev())
        self._check(_lib.otoo_sph_stage1(self._h, self._p(h, torch.float32), self._p(vel, torch.float32, 4), int(group_size),
                                         rho.data_ptr(), nngb.data_ptr(), dr.data_ptr(), self._stream(stream)))
        return rho, nngb, dr

    def otoo_sph_adapt_h(self, h, n_target, tol, max_iter, group_size, stream=None):
        """h (N floats on the device) is updated in place; returns (nngb of the final h, updates made)"""
        nngb = torch.empty(self.N, dtype=torch.int32, device=self._dev())
        it = C.c_int(0)
        self._check(_lib.otoo_sph_adapt_h(self._h, self._p(h, torch.float32), float(n_target), float(tol), int(max_iter),
                                          int(group_size), nngb.data_ptr(), C.byref(it), self._stream(stream)))
        return nngb, int(it.value)

    def otoo_sph_force(self, h, rho, P, group_size, vel=None, stream=None):
        out = torch.empty((self.N, 4), dtype=torch.float32, device=self._dev())
        self._check(_lib.otoo_sph_force(self._h, self._p(h, torch.float32), self._p(rho, torch.float32),
                                        self._p(P, torch.float32), self._p(vel, torch.float32, 4) if vel is not None else None,
                                        int(group_size), self._p(out), self._stream(stream)))
        return out

    def otoo_unsort(self, sorted_rows, out=None, stream=None):
        """rows (N,4) in sorted order -> the caller's particle order"""
        if out is None:
            out = torch.empty((self.N, 4), dtype=torch.float32, device=self._dev())
        self._check(_lib.otoo_unsort(self._h, self._p(sorted_rows, torch.float32, 4), self._p(out, torch.float32, 4), self._stream(stream)))
        return out

    def otoo_eos_ideal(self, rho, u, gamma=5.0 / 3.0, stream=None):
        P = torch.empty_like(rho)
        self._check(_lib.otoo_eos_ideal(self._h, _ptr(rho, torch.float32), _ptr(u, torch.float32), float(gamma),
                                        rho.numel(), _ptr(P), self._stream(stream)))
        return P

    def otoo_gravity_host(self, pos_mass: np.ndarray, n_crit, eps, theta, group_size, out: np.ndarray = None):
        pm = np.ascontiguousarray(pos_mass, dtype=np.float32)
        n = pm.shape[0]
        if out is None:
            out = np.empty((n, 4), dtype=np.float32)
        self._check(_lib.otoo_gravity_host(self._h, pm.ctypes.data, n, int(n_crit), float(eps), float(theta),
                                           int(group_size), out.ctypes.data))
        self.N = n
        return out

    def otoo_gravity_delta_host(self, pos_mass: np.ndarray, n_crit, eps, delta, m_limit, group_size, out: np.ndarray = None):
        pm = np.ascontiguousarray(pos_mass, dtype=np.float32)
        n = pm.shape[0]
        if out is None:
            out = np.empty((n, 4), dtype=np.float32)
        self._check(_lib.otoo_gravity_delta_host(self._h, pm.ctypes.data, n, int(n_crit), float(eps), float(delta),
                                                 float(m_limit), int(group_size), out.ctypes.data))
        self.N = n
        return out

    # ---- introspection
    def otoo_tree_info(self):
        ti = TreeInfo()
        self._check(_lib.otoo_tree_info(self._h, C.byref(ti)))
        return dict(N=ti.N, N_cell=ti.N_cell, N_leaf=ti.N_leaf, depth=ti.depth,
                    lo=np.array(list(ti.lo), dtype=np.float32), S=float(ti.S))

    def otoo_export_tree(self):
        info = self.otoo_tree_info()
        n, nc, dev = info["N"], info["N_cell"], self._dev()
        perm = torch.empty(n, dtype=torch.int32, device=dev)
        keys = torch.empty(n, dtype=torch.int64, device=dev)
        cells = torch.empty(nc * CELL_DTYPE.itemsize, dtype=torch.uint8, device=dev)
        com_m = torch.empty((nc, 4), dtype=torch.float32, device=dev)
        rb2 = torch.empty(nc, dtype=torch.float32, device=dev)
        self._check(_lib.otoo_export_tree(self._h, perm.data_ptr(), keys.data_ptr(), cells.data_ptr(),
                                          com_m.data_ptr(), rb2.data_ptr()))
        return dict(perm=perm.cpu().numpy().view(np.uint32), keys=keys.cpu().numpy().view(np.uint64),
                    cells=cells.cpu().numpy().view(CELL_DTYPE), com_m=com_m.cpu().numpy(), rb2=rb2.cpu().numpy(),
                    **info)

    def otoo_export_sph_radii(self):
        nc = self.otoo_tree_info()["N_cell"]
        b = torch.empty(nc, dtype=torch.float32, device=self._dev())
        r = torch.empty(nc, dtype=torch.float32, device=self._dev())
        self._check(_lib.otoo_export_sph_radii(self._h, b.data_ptr(), r.data_ptr()))
        return b.cpu().numpy(), r.cpu().numpy()

    def otoo_export_group_stats(self, on_device=False):
        """(n_tests, n_cells, n_parts) per group of the last walk: numpy uint32 arrays, or int32 CUDA tensors"""
        st = self.otoo_last_stats()
        ng = st["n_groups"]
        a = [torch.empty(ng, dtype=torch.int32, device=self._dev()) for _ in range(3)]
        self._check(_lib.otoo_export_group_stats(self._h, a[0].data_ptr(), a[1].data_ptr(), a[2].data_ptr()))
        if on_device:
            return tuple(a)
        return tuple(x.cpu().numpy().view(np.uint32) for x in a)

    def otoo_last_stats(self):
        s = Stats()
        self._check(_lib.otoo_last_stats(self._h, C.byref(s)))
        d = {k: getattr(s, k) for k, _ in Stats._fields_}
        d["ms_build"] = dict(zip(BUILD_PHASES, [float(x) for x in s.ms_build]))
        return d

    def otoo_measure_fp32_peak(self, stream=None) -> float:
        v = C.c_double(0.0)
        self._check(_lib.otoo_measure_fp32_peak(self._h, C.byref(v), self._stream(stream)))
        return float(v.value)

    def otoo_probe(self, which: str, stream=None):
        """microbenchmark table of the library (list of dicts); invalidates the tree"""
        import json
        buf = C.create_string_buffer(1 << 16)
        self._check(_lib.otoo_probe(self._h, which.encode(), buf, len(buf), self._stream(stream)))
        self.N = 0
        return json.loads(buf.value.decode())

    def otoo_set_option(self, name: str, value: int):
        self._check(_lib.otoo_set_option(self._h, name.encode(), int(value)))


def otoo_sort_pairs_static(keys, vals, keys_alt, vals_alt, n=None, stream=None):
    """otoo_sort_pairs_static of include/otoo.h: stable sort of (int64-typed u64 key, int32-typed u32 value) pairs in
    place on the tensors' device, no allocation inside the library (the four buffers are the caller's: create them
    before a graph capture).  Argument marshalling only; raises OtooError with the library's message."""
    n = int(keys.shape[0] if n is None else n)
    dev = keys.device
    for t, dt in ((keys, torch.int64), (vals, torch.int32), (keys_alt, torch.int64), (vals_alt, torch.int32)):
        _ptr(t, dt, device=dev.index)
        if t.ndim != 1 or t.shape[0] < n:
            raise ValueError(f"expected 1-d tensors of at least {n} elements")
    err = C.create_string_buffer(512)
    with torch.cuda.device(dev):                 # the entry point works on the current device
        st = torch.cuda.current_stream(dev).cuda_stream if stream is None else (
            stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))
        status = _lib.otoo_sort_pairs_static(keys.data_ptr(), vals.data_ptr(), keys_alt.data_ptr(), vals_alt.data_ptr(),
                                             n, st, err, len(err))
    if status != 0:
        raise OtooError(status, err.value.decode())
    return keys, vals

def raw():
    """The ctypes library handle (tests check exported symbols and error statuses)."""
    return _lib

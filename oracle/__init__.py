"""ctypes binding of the serial C++ oracle (oracle/sdm_oracle.cpp).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package (paper_2103_17238_b200) never
imports this module, and this module never imports the product package.

All arrays are numpy host arrays; `coalescence_step` updates `xi` and `v` in place.
"""
from __future__ import annotations

import ctypes as C
import importlib.util
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))


def _load():
    spec = importlib.util.spec_from_file_location("_oracle_build", os.path.join(_HERE, "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return C.CDLL(mod.build())


class KernelParams(C.Structure):
    _fields_ = [("kind", C.c_int32), ("_pad", C.c_int32), ("b", C.c_double), ("E", C.c_double),
                ("n_r", C.c_int32), ("n_p", C.c_int32), ("radius", C.c_void_p), ("table", C.c_void_p)]


GOLOVIN = 0
GEOMETRIC = 1
GEOMETRIC_TABLE = 2

_lib = _load()

_i64p = np.ctypeslib.ndpointer(np.int64, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")
_i32p = np.ctypeslib.ndpointer(np.int32, flags="C_CONTIGUOUS")
_u32p = np.ctypeslib.ndpointer(np.uint32, flags="C_CONTIGUOUS")

_lib.oracle_philox4x32_10.argtypes = [_u32p, _u32p, _u32p]
_lib.oracle_philox4x32_10.restype = None
_lib.oracle_uniform_from_words.argtypes = [C.c_uint32, C.c_uint32]
_lib.oracle_uniform_from_words.restype = C.c_double
_lib.oracle_sd_random.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.POINTER(C.c_uint32), C.POINTER(C.c_double)]
_lib.oracle_sd_random.restype = None
_lib.oracle_sd_random_batch.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.c_int64, _u32p, _f64p]
_lib.oracle_sd_random_batch.restype = None
_lib.oracle_det_cbrt.argtypes = [C.c_double]
_lib.oracle_det_cbrt.restype = C.c_double
_lib.oracle_terminal_velocity.argtypes = [C.c_double]
_lib.oracle_terminal_velocity.restype = C.c_double
_lib.oracle_radius.argtypes = [C.c_double]
_lib.oracle_radius.restype = C.c_double
_lib.oracle_efficiency.argtypes = [C.POINTER(KernelParams), C.c_double, C.c_double]
_lib.oracle_efficiency.restype = C.c_double
_lib.oracle_kernel.argtypes = [C.POINTER(KernelParams), C.c_double, C.c_double]
_lib.oracle_kernel.restype = C.c_double
_lib.oracle_gamma_from_p.argtypes = [C.c_double, C.c_double]
_lib.oracle_gamma_from_p.restype = C.c_int64
_lib.oracle_pair_update.argtypes = [C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_double),
                                    C.POINTER(C.c_double), C.c_int64]
_lib.oracle_pair_update.restype = C.c_int64
_lib.oracle_coalescence_step.argtypes = [
    _i64p, _f64p, _i32p, C.c_int64, C.c_int32, C.c_double, C.c_double, C.POINTER(KernelParams),
    C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.oracle_coalescence_step.restype = C.c_int
_lib.oracle_coalescence_step_shard.argtypes = [
    _i64p, _f64p, _i32p, C.c_int64, C.c_int32, C.c_double, C.c_double, C.POINTER(KernelParams),
    C.c_uint64, C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.oracle_coalescence_step_shard.restype = C.c_int
_lib.oracle_remove_zero_multiplicity.argtypes = [_i64p, _f64p, _i32p, C.c_int64]
_lib.oracle_remove_zero_multiplicity.restype = C.c_int64
_lib.oracle_cell_stats.argtypes = [_i64p, _f64p, _i32p, C.c_int64, C.c_int32, _i32p, _i64p, _f64p, _f64p]
_lib.oracle_cell_stats.restype = C.c_int
_lib.oracle_volume_spectrum.argtypes = [_i64p, _f64p, C.c_int64, _f64p, C.c_int32, _i64p, _i64p, _f64p]
_lib.oracle_volume_spectrum.restype = C.c_int
_lib.oracle_total_xi_v_int128.argtypes = [_i64p, _f64p, C.c_int64, C.POINTER(C.c_int64), C.POINTER(C.c_uint64)]
_lib.oracle_total_xi_v_int128.restype = None
_lib.oracle_run.argtypes = [_i64p, _f64p, _i32p, C.c_int64, C.c_int32, C.c_double, C.c_double,
                            C.POINTER(KernelParams), C.c_uint64, C.c_uint64, C.c_int64, C.c_int64]
_lib.oracle_run.restype = C.c_int64


_lib.oracle_wrap_periodic.argtypes = [C.c_double, C.c_int32]
_lib.oracle_wrap_periodic.restype = C.c_double
_lib.oracle_cell_of.argtypes = [C.c_double, C.c_double, C.c_int32, C.c_int32]
_lib.oracle_cell_of.restype = C.c_int32
_lib.oracle_cell_id_from_positions.argtypes = [_f64p, _f64p, C.c_int64, C.c_int32, C.c_int32, _i32p]
_lib.oracle_cell_id_from_positions.restype = C.c_int
_lib.oracle_displace.argtypes = [_f64p, _f64p, _i32p, C.c_int64, C.c_int32, C.c_int32, _f64p, _f64p, C.c_double]
_lib.oracle_displace.restype = C.c_int


def kernel_params(kind: int, b: float = 0.0, E: float = 1.0) -> KernelParams:
    return KernelParams(kind=kind, _pad=0, b=b, E=E, n_r=0, n_p=0, radius=None, table=None)


def geometric_table(radius, table) -> KernelParams:
    """Geometric kernel with a tabulated collision efficiency E(r_big, r_small / r_big) (R39): `radius` strictly
    ascending [n_r], `table` [n_r][n_p] over the ratios j / (n_p - 1).  The arrays are kept alive by the result."""
    r = np.ascontiguousarray(radius, np.float64)
    t = np.ascontiguousarray(table, np.float64)
    if r.ndim != 1 or t.ndim != 2 or t.shape[0] != r.shape[0] or r.shape[0] < 2 or t.shape[1] < 2:
        raise ValueError("table shape")
    if not np.all(np.diff(r) > 0) or not np.all(np.isfinite(t)) or np.any(t < 0):
        raise ValueError("table values")
    kp = KernelParams(kind=GEOMETRIC_TABLE, _pad=0, b=0.0, E=0.0, n_r=r.shape[0], n_p=t.shape[1],
                      radius=r.ctypes.data, table=t.ctypes.data)
    kp._keep = (r, t)
    return kp


def efficiency(kp: KernelParams, r_big: float, p: float) -> float:
    return float(_lib.oracle_efficiency(C.byref(kp), r_big, p))


def golovin(b: float) -> KernelParams:
    return kernel_params(GOLOVIN, b=b, E=0.0)


def geometric(E: float = 1.0) -> KernelParams:
    return kernel_params(GEOMETRIC, b=0.0, E=E)


def philox4x32_10(ctr, key) -> np.ndarray:
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32)
    key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    _lib.oracle_philox4x32_10(ctr, key, out)
    return out


def uniform_from_words(w2: int, w3: int) -> float:
    return float(_lib.oracle_uniform_from_words(w2, w3))


def sd_random(seed: int, step: int, i: int):
    k = C.c_uint32()
    u = C.c_double()
    _lib.oracle_sd_random(seed, step, i, C.byref(k), C.byref(u))
    return int(k.value), float(u.value)


def sd_random_batch(seed: int, step: int, i0: int, n: int):
    keys = np.zeros(n, np.uint32)
    us = np.zeros(n, np.float64)
    _lib.oracle_sd_random_batch(seed, step, i0, n, keys, us)
    return keys, us


def det_cbrt(x: float) -> float:
    return float(_lib.oracle_det_cbrt(x))


def terminal_velocity(r: float) -> float:
    return float(_lib.oracle_terminal_velocity(r))


def radius(v: float) -> float:
    return float(_lib.oracle_radius(v))


def kernel(kp: KernelParams, vj: float, vk: float) -> float:
    return float(_lib.oracle_kernel(C.byref(kp), vj, vk))


def gamma_from_p(p: float, u: float) -> int:
    return int(_lib.oracle_gamma_from_p(p, u))


def pair_update(xi_j: int, xi_k: int, v_j: float, v_k: float, g: int):
    a, b = C.c_int64(xi_j), C.c_int64(xi_k)
    c, d = C.c_double(v_j), C.c_double(v_k)
    gt = _lib.oracle_pair_update(C.byref(a), C.byref(b), C.byref(c), C.byref(d), g)
    return int(gt), int(a.value), int(b.value), float(c.value), float(d.value)


def coalescence_step(xi, v, cell_id, n_cell, dt, dV, kp, seed, step, n_sd=None, debug=False, index_base=0):
    """One step, in place.  With debug=True returns dict(perm, gamma, gamma_clamped, cell_start).
    index_base: Philox counter of entry i is index_base + i (a shard of a larger array, R34)."""
    n = int(len(xi) if n_sd is None else n_sd)
    out = None
    ptrs = [None, None, None, None]
    if debug:
        out = dict(perm=np.zeros(n, np.int32), gamma=np.zeros(n, np.int64),
                   gamma_clamped=np.zeros(n, np.int64), cell_start=np.zeros(n_cell + 1, np.int32))
        ptrs = [out[k].ctypes.data for k in ("perm", "gamma", "gamma_clamped", "cell_start")]
    rc = _lib.oracle_coalescence_step_shard(xi, v, cell_id, n, n_cell, dt, dV, C.byref(kp), seed, step, int(index_base),
                                            *ptrs)
    if rc != 0:
        raise ValueError(f"oracle_coalescence_step failed: {rc}")
    return out


def remove_zero_multiplicity(xi, v, cell_id, n_sd=None) -> int:
    n = int(len(xi) if n_sd is None else n_sd)
    return int(_lib.oracle_remove_zero_multiplicity(xi, v, cell_id, n))


def cell_stats(xi, v, cell_id, n_cell, n_sd=None):
    n = int(len(xi) if n_sd is None else n_sd)
    count = np.zeros(n_cell, np.int32)
    sum_xi = np.zeros(n_cell, np.int64)
    sum_xi_v = np.zeros(n_cell, np.float64)
    sum_xi_v2 = np.zeros(n_cell, np.float64)
    rc = _lib.oracle_cell_stats(xi, v, cell_id, n, n_cell, count, sum_xi, sum_xi_v, sum_xi_v2)
    if rc != 0:
        raise ValueError(f"oracle_cell_stats failed: {rc}")
    return count, sum_xi, sum_xi_v, sum_xi_v2


def volume_spectrum(xi, v, volume_edges, n_sd=None):
    """O7: per-bin (count, sum xi, sum xi*v) over bins edges[b] <= v < edges[b+1] of VOLUME edges."""
    n = int(len(xi) if n_sd is None else n_sd)
    edges = np.ascontiguousarray(volume_edges, np.float64)
    nb = len(edges) - 1
    count = np.zeros(max(nb, 0), np.int64)
    sum_xi = np.zeros(max(nb, 0), np.int64)
    sum_xi_v = np.zeros(max(nb, 0), np.float64)
    rc = _lib.oracle_volume_spectrum(xi, v, n, edges, len(edges), count, sum_xi, sum_xi_v)
    if rc != 0:
        raise ValueError(f"oracle_volume_spectrum failed: {rc}")
    return count, sum_xi, sum_xi_v


def total_xi_v_exact(xi, v, n_sd=None) -> int:
    """Exact sum of xi*v for integer-valued v, as a Python int (128-bit accumulate)."""
    n = int(len(xi) if n_sd is None else n_sd)
    hi, lo = C.c_int64(), C.c_uint64()
    _lib.oracle_total_xi_v_int128(xi, v, n, C.byref(hi), C.byref(lo))
    return (int(hi.value) << 64) | int(lo.value)


def run(xi, v, cell_id, n_cell, dt, dV, kp, seed, step0, n_steps, compact_every=0, n_sd=None) -> int:
    n = int(len(xi) if n_sd is None else n_sd)
    r = int(_lib.oracle_run(xi, v, cell_id, n, n_cell, dt, dV, C.byref(kp), seed, step0, n_steps, compact_every))
    if r < 0:
        raise ValueError(f"oracle_run failed: {r}")
    return r


def wrap_periodic(q: float, n: int) -> float:
    return float(_lib.oracle_wrap_periodic(q, n))


def cell_of(x: float, z: float, nx: int, nz: int) -> int:
    return int(_lib.oracle_cell_of(x, z, nx, nz))


def cell_id_from_positions(x, z, nx, nz) -> np.ndarray:
    """O8: cell_id = floor(z) * nx + floor(x) for positions in grid units."""
    out = np.zeros(len(x), np.int32)
    rc = _lib.oracle_cell_id_from_positions(x, z, len(x), nx, nz, out)
    if rc != 0:
        raise ValueError(f"oracle_cell_id_from_positions failed: {rc}")
    return out


def displace(x, z, cell_id, nx, nz, u_cell, w_cell, dt):
    """O8: one explicit-Euler displacement step on the periodic nx x nz grid, in place; rewrites cell_id."""
    rc = _lib.oracle_displace(x, z, cell_id, len(x), nx, nz, np.ascontiguousarray(u_cell, np.float64),
                              np.ascontiguousarray(w_cell, np.float64), dt)
    if rc != 0:
        raise ValueError(f"oracle_displace failed: {rc}")

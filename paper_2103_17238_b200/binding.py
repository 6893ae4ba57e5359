"""ctypes binding of include/sdm.h -- same names, argument marshalling only.

`SDMContext` owns a torch-allocated workspace and forwards torch tensors' data pointers and the
current CUDA stream to the C ABI.  Nothing is computed here.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libsdm_b200.so")

GOLOVIN = 0
GEOMETRIC = 1
GEOMETRIC_TABLE = 2
PATH_AUTO = 0
PATH_GENERAL = 1
PATH_CELL_SORTED = 2
PATH_HYBRID = 3
PATH_BOX = 4
PATH_BUCKET = 5
OPT_NARROW_KEY_BITS = 0
OPT_TRACK_ZEROS = 1
OPT_INDEX_BASE = 2
OPT_SKIP_KEY_DIGITS = 3
OPT_FUSED_WORDS_PER_LANE = 4
OPT_BUCKET_BITS = 5
OPT_BOX_CLUSTER = 6

SDM_OK = 0

EXPORTS = [
    "sdm_workspace_bytes", "sdm_init", "sdm_coalescence_step", "sdm_coalescence_steps", "sdm_remove_zero_multiplicity",
    "sdm_cell_stats", "sdm_debug_outputs", "sdm_set_path", "sdm_last_path", "sdm_host_staging_bytes",
    "sdm_bind_host_staging", "sdm_coalescence_step_host", "sdm_poll_error", "sdm_launch_count",
    "sdm_philox_fill", "sdm_kernel_eval", "sdm_strerror", "sdm_destroy", "sdm_profile_enable",
    "sdm_profile_read", "sdm_set_option", "sdm_volume_spectrum", "sdm_displace", "sdm_cell_id_from_positions",
    "sdm_set_collision_efficiency", "sdm_static_max_n_sd", "sdm_static_setup", "sdm_remove_zero_multiplicity_static",
]

PROF_CLASSES = ["keys_hist", "cell_scan", "radix_pass", "pair", "count_zero", "compact", "cell_stats", "other",
                "cell_bounds", "cell_fused", "cell_digit_hist", "tie_repair", "volume_spectrum", "displace", "cell_classes", "box_step", "bucket", "resident_move"]


class SDMError(RuntimeError):
    def __init__(self, status: int, what: str):
        super().__init__(f"{what}: status {status} ({_strerror(status)})")
        self.status = status


class KernelParams(C.Structure):
    _fields_ = [("kind", C.c_int32), ("_pad", C.c_int32), ("b", C.c_double), ("E", C.c_double)]


def golovin(b: float) -> KernelParams:
    return KernelParams(kind=GOLOVIN, _pad=0, b=float(b), E=0.0)


def geometric(E: float = 1.0) -> KernelParams:
    return KernelParams(kind=GEOMETRIC, _pad=0, b=0.0, E=float(E))


def geometric_table() -> KernelParams:
    """Geometric kernel with the collision-efficiency table installed by SDMContext.set_collision_efficiency."""
    return KernelParams(kind=GEOMETRIC_TABLE, _pad=0, b=0.0, E=0.0)


_lib = None


def library_path() -> str:
    return _LIB_PATH


def load_library():
    """Loads libsdm_b200.so; raises (never falls back) when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise SDMError(-3, f"{_LIB_PATH} is missing -- build it with `python -m paper_2103_17238_b200._build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(_LIB_PATH)
    vp, i64, i32, u64, dbl = C.c_void_p, C.c_int64, C.c_int32, C.c_uint64, C.c_double
    kpp = C.POINTER(KernelParams)
    lib.sdm_workspace_bytes.argtypes = [i64, i32]
    lib.sdm_workspace_bytes.restype = C.c_size_t
    lib.sdm_init.argtypes = [C.POINTER(vp), C.c_int, i64, i32, vp, C.c_size_t, vp]
    lib.sdm_init.restype = C.c_int
    lib.sdm_coalescence_step.argtypes = [vp, vp, vp, vp, i64, i32, dbl, dbl, kpp, u64, u64]
    lib.sdm_coalescence_step.restype = C.c_int
    lib.sdm_coalescence_steps.argtypes = [vp, vp, vp, vp, i64, i32, dbl, dbl, kpp, u64, u64, i64, i64, C.POINTER(i64)]
    lib.sdm_coalescence_steps.restype = C.c_int
    lib.sdm_remove_zero_multiplicity.argtypes = [vp, vp, vp, vp, i64, C.POINTER(i64)]
    lib.sdm_remove_zero_multiplicity.restype = C.c_int
    lib.sdm_cell_stats.argtypes = [vp, vp, vp, vp, i64, i32, vp, vp, vp, vp]
    lib.sdm_cell_stats.restype = C.c_int
    lib.sdm_debug_outputs.argtypes = [vp, vp, vp, vp, vp]
    lib.sdm_debug_outputs.restype = C.c_int
    lib.sdm_set_path.argtypes = [vp, C.c_int]
    lib.sdm_set_path.restype = C.c_int
    lib.sdm_set_option.argtypes = [vp, C.c_int, i64]
    lib.sdm_set_option.restype = C.c_int
    lib.sdm_last_path.argtypes = [vp]
    lib.sdm_last_path.restype = C.c_int
    lib.sdm_host_staging_bytes.argtypes = [i64]
    lib.sdm_host_staging_bytes.restype = C.c_size_t
    lib.sdm_bind_host_staging.argtypes = [vp, vp, C.c_size_t]
    lib.sdm_bind_host_staging.restype = C.c_int
    lib.sdm_coalescence_step_host.argtypes = [vp, vp, vp, vp, i64, i32, dbl, dbl, kpp, u64, u64, C.c_int,
                                              C.POINTER(i64)]
    lib.sdm_profile_enable.argtypes = [vp, C.c_int]
    lib.sdm_profile_enable.restype = C.c_int
    lib.sdm_profile_read.argtypes = [vp, C.POINTER(dbl), C.POINTER(i64)]
    lib.sdm_profile_read.restype = C.c_int
    lib.sdm_coalescence_step_host.restype = C.c_int
    lib.sdm_volume_spectrum.argtypes = [vp, vp, vp, i64, C.POINTER(C.c_double), i32, vp, vp, vp]
    lib.sdm_volume_spectrum.restype = C.c_int
    lib.sdm_displace.argtypes = [vp, vp, vp, vp, i64, i32, i32, vp, vp, dbl]
    lib.sdm_displace.restype = C.c_int
    lib.sdm_cell_id_from_positions.argtypes = [vp, vp, vp, i64, i32, i32, vp]
    lib.sdm_cell_id_from_positions.restype = C.c_int
    lib.sdm_set_collision_efficiency.argtypes = [vp, C.POINTER(C.c_double), i32, i32, C.POINTER(C.c_double)]
    lib.sdm_set_collision_efficiency.restype = C.c_int
    lib.sdm_poll_error.argtypes = [vp]
    lib.sdm_poll_error.restype = C.c_int
    lib.sdm_launch_count.argtypes = [vp]
    lib.sdm_launch_count.restype = i64
    lib.sdm_philox_fill.argtypes = [vp, u64, u64, u64, i64, vp, vp]
    lib.sdm_philox_fill.restype = C.c_int
    lib.sdm_kernel_eval.argtypes = [vp, kpp, vp, vp, i64, vp]
    lib.sdm_kernel_eval.restype = C.c_int
    lib.sdm_static_max_n_sd.argtypes = []
    lib.sdm_static_max_n_sd.restype = i64
    lib.sdm_static_setup.argtypes = []
    lib.sdm_static_setup.restype = C.c_int
    lib.sdm_remove_zero_multiplicity_static.argtypes = [vp, vp, vp, i64, vp, vp]
    lib.sdm_remove_zero_multiplicity_static.restype = C.c_int
    lib.sdm_strerror.argtypes = [C.c_int]
    lib.sdm_strerror.restype = C.c_char_p
    lib.sdm_destroy.argtypes = [vp]
    lib.sdm_destroy.restype = None
    _lib = lib
    return lib


def _strerror(status: int) -> str:
    try:
        return load_library().sdm_strerror(status).decode()
    except Exception:  # library missing: still give a readable message
        return "library not loaded"


def workspace_bytes(max_n_sd: int, max_n_cell: int) -> int:
    return int(load_library().sdm_workspace_bytes(max_n_sd, max_n_cell))


def host_staging_bytes(max_n_sd: int) -> int:
    return int(load_library().sdm_host_staging_bytes(max_n_sd))


def static_max_n_sd() -> int:
    """Largest n_sd the allocation-free entry point takes (its scratch is a fixed device array inside the library)."""
    return int(load_library().sdm_static_max_n_sd())


def remove_zero_multiplicity_static(multiplicity, volume, cell_id, n_sd_out, n_sd=None, stream=None) -> None:
    """sdm_remove_zero_multiplicity_static: no context, no workspace, no allocation, no synchronisation.  `n_sd_out`
    is a DEVICE int64 tensor of one element that receives the number of survivors.  Runs on the tensors' device, on
    `stream` (default: torch's current stream there).  Calls that overlap on the GPU race on the shared scratch."""
    import torch

    lib = load_library()
    n = int(multiplicity.shape[0] if n_sd is None else n_sd)
    if n_sd_out.dtype != torch.int64 or n_sd_out.numel() < 1 or not n_sd_out.is_cuda:
        raise TypeError("n_sd_out must be a CUDA int64 tensor of at least one element")
    with torch.cuda.device(n_sd_out.device):
        st = stream if stream is not None else torch.cuda.current_stream(n_sd_out.device)
        rc = lib.sdm_remove_zero_multiplicity_static(_ptr(multiplicity, torch.int64), _ptr(volume, torch.float64),
                                                     _ptr(cell_id, torch.int32), n, n_sd_out.data_ptr(), st.cuda_stream)
    _check(rc, "sdm_remove_zero_multiplicity_static")


def _ptr(t, dtype=None):
    if t is None:
        return None
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    return t.data_ptr()


def _check(status: int, what: str):
    if status != SDM_OK:
        raise SDMError(status, what)


class SDMContext:
    """sdm_init / sdm_destroy plus one method per C entry point (same names without the prefix)."""

    def __init__(self, max_n_sd: int, max_n_cell: int, device=None, stream=None, host_staging: bool = False):
        import torch

        self._torch = torch
        self._lib = load_library()
        if not torch.cuda.is_available():
            raise SDMError(-3, "no CUDA device: the SDM step has no CPU fallback")
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self.max_n_sd = int(max_n_sd)
        self.max_n_cell = int(max_n_cell)
        nbytes = workspace_bytes(self.max_n_sd, self.max_n_cell)
        if nbytes == 0:
            raise SDMError(-1, "sdm_workspace_bytes")
        with torch.cuda.device(self.device):
            self._workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self._stream = torch.cuda.current_stream(self.device) if stream is None else stream
            handle = C.c_void_p()
            rc = self._lib.sdm_init(C.byref(handle), self.device.index, self.max_n_sd, self.max_n_cell,
                                    self._workspace.data_ptr(), nbytes, self._stream.cuda_stream)
        _check(rc, "sdm_init")
        self._h = handle
        self._staging = None
        self._debug = None
        if host_staging:
            sb = host_staging_bytes(self.max_n_sd)
            self._staging = torch.empty(sb, dtype=torch.uint8, device=self.device)
            _check(self._lib.sdm_bind_host_staging(self._h, self._staging.data_ptr(), sb), "sdm_bind_host_staging")

    # -- lifetime ---------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None) is not None:
            self._torch.cuda.synchronize(self.device)
            self._lib.sdm_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- the calls --------------------------------------------------------------------------
    def coalescence_step(self, multiplicity, volume, cell_id, n_cell, dt, dV, kp, seed, step, n_sd=None):
        t = self._torch
        n = int(multiplicity.shape[0] if n_sd is None else n_sd)
        rc = self._lib.sdm_coalescence_step(self._h, _ptr(multiplicity, t.int64), _ptr(volume, t.float64),
                                            _ptr(cell_id, t.int32), n, int(n_cell), float(dt), float(dV),
                                            C.byref(kp), int(seed), int(step))
        _check(rc, "sdm_coalescence_step")

    def coalescence_steps(self, multiplicity, volume, cell_id, n_cell, dt, dV, kp, seed, step0, n_steps,
                          compact_every=0, n_sd=None) -> int:
        """sdm_coalescence_steps: n_steps steps (+ a compaction every `compact_every` steps) in one call; returns
        the final number of super-droplets."""
        t = self._torch
        n = int(multiplicity.shape[0] if n_sd is None else n_sd)
        out = C.c_int64(n)
        rc = self._lib.sdm_coalescence_steps(self._h, _ptr(multiplicity, t.int64), _ptr(volume, t.float64),
                                             _ptr(cell_id, t.int32), n, int(n_cell), float(dt), float(dV), C.byref(kp),
                                             int(seed), int(step0), int(n_steps), int(compact_every), C.byref(out))
        _check(rc, "sdm_coalescence_steps")
        return int(out.value)

    def remove_zero_multiplicity(self, multiplicity, volume, cell_id, n_sd=None) -> int:
        t = self._torch
        n = int(multiplicity.shape[0] if n_sd is None else n_sd)
        out = C.c_int64(0)
        rc = self._lib.sdm_remove_zero_multiplicity(self._h, _ptr(multiplicity, t.int64), _ptr(volume, t.float64),
                                                    _ptr(cell_id, t.int32), n, C.byref(out))
        _check(rc, "sdm_remove_zero_multiplicity")
        return int(out.value)

    def cell_stats(self, multiplicity, volume, cell_id, n_cell, n_sd=None):
        t = self._torch
        n = int(multiplicity.shape[0] if n_sd is None else n_sd)
        count = t.empty(n_cell, dtype=t.int32, device=self.device)
        sum_xi = t.empty(n_cell, dtype=t.int64, device=self.device)
        sum_xi_v = t.empty(n_cell, dtype=t.float64, device=self.device)
        sum_xi_v2 = t.empty(n_cell, dtype=t.float64, device=self.device)
        rc = self._lib.sdm_cell_stats(self._h, _ptr(multiplicity, t.int64), _ptr(volume, t.float64),
                                      _ptr(cell_id, t.int32), n, int(n_cell), count.data_ptr(), sum_xi.data_ptr(),
                                      sum_xi_v.data_ptr(), sum_xi_v2.data_ptr())
        _check(rc, "sdm_cell_stats")
        return count, sum_xi, sum_xi_v, sum_xi_v2

    def debug_outputs(self, n_sd: int | None, n_cell: int | None = None):
        """Allocates and registers the parity outputs (or switches them off with n_sd=None)."""
        t = self._torch
        if n_sd is None:
            self._debug = None
            _check(self._lib.sdm_debug_outputs(self._h, None, None, None, None), "sdm_debug_outputs")
            return None
        d = dict(perm=t.zeros(max(n_sd, 1), dtype=t.int32, device=self.device),
                 gamma=t.zeros(max(n_sd, 1), dtype=t.int64, device=self.device),
                 gamma_clamped=t.zeros(max(n_sd, 1), dtype=t.int64, device=self.device),
                 cell_start=t.zeros((n_cell or 1) + 1, dtype=t.int32, device=self.device))
        self._debug = d
        _check(self._lib.sdm_debug_outputs(self._h, d["perm"].data_ptr(), d["gamma"].data_ptr(),
                                           d["gamma_clamped"].data_ptr(), d["cell_start"].data_ptr()),
               "sdm_debug_outputs")
        return d

    def set_path(self, path: int):
        _check(self._lib.sdm_set_path(self._h, int(path)), "sdm_set_path")

    def volume_spectrum(self, multiplicity, volume, volume_edges, n_sd=None):
        """sdm_volume_spectrum: (count int64[nb], sum_xi int64[nb], sum_xi_v float64[nb]) device tensors."""
        t = self._torch
        n = int(multiplicity.shape[0] if n_sd is None else n_sd)
        edges = [float(e) for e in volume_edges]
        arr = (C.c_double * len(edges))(*edges)
        nb = max(len(edges) - 1, 0)
        count = t.empty(nb, dtype=t.int64, device=self.device)
        sum_xi = t.empty(nb, dtype=t.int64, device=self.device)
        sum_xi_v = t.empty(nb, dtype=t.float64, device=self.device)
        rc = self._lib.sdm_volume_spectrum(self._h, _ptr(multiplicity, t.int64), _ptr(volume, t.float64), n, arr,
                                           len(edges), count.data_ptr(), sum_xi.data_ptr(), sum_xi_v.data_ptr())
        _check(rc, "sdm_volume_spectrum")
        return count, sum_xi, sum_xi_v

    def displace(self, x, z, cell_id, nx, nz, u_cell, w_cell, dt, n_sd=None):
        """sdm_displace: one explicit-Euler step on the periodic nx x nz grid; x, z, cell_id updated in place."""
        t = self._torch
        n = int(x.shape[0] if n_sd is None else n_sd)
        rc = self._lib.sdm_displace(self._h, _ptr(x, t.float64), _ptr(z, t.float64), _ptr(cell_id, t.int32), n, int(nx),
                                    int(nz), _ptr(u_cell, t.float64), _ptr(w_cell, t.float64), float(dt))
        _check(rc, "sdm_displace")

    def cell_id_from_positions(self, x, z, nx, nz, cell_id=None, n_sd=None):
        t = self._torch
        n = int(x.shape[0] if n_sd is None else n_sd)
        if cell_id is None:
            cell_id = t.empty(max(n, 1), dtype=t.int32, device=self.device)
        rc = self._lib.sdm_cell_id_from_positions(self._h, _ptr(x, t.float64), _ptr(z, t.float64), n, int(nx), int(nz),
                                                  _ptr(cell_id, t.int32))
        _check(rc, "sdm_cell_id_from_positions")
        return cell_id

    def set_collision_efficiency(self, radius, table):
        """sdm_set_collision_efficiency: `radius` [n_r] ascending (m), `table` [n_r][n_p] (nested sequences or a
        2-D array); None, None removes the table."""
        if radius is None and table is None:
            _check(self._lib.sdm_set_collision_efficiency(self._h, None, 0, 0, None), "sdm_set_collision_efficiency")
            return
        rows = [[float(e) for e in row] for row in table]
        n_r, n_p = len(rows), (len(rows[0]) if rows else 0)
        if any(len(row) != n_p for row in rows) or len(radius) != n_r:
            raise ValueError("table shape")
        r = (C.c_double * n_r)(*[float(x) for x in radius])
        t = (C.c_double * (n_r * n_p))(*[e for row in rows for e in row])
        _check(self._lib.sdm_set_collision_efficiency(self._h, r, n_r, n_p, t), "sdm_set_collision_efficiency")

    def set_option(self, option: int, value: int):
        _check(self._lib.sdm_set_option(self._h, int(option), int(value)), "sdm_set_option")

    def last_path(self) -> int:
        return int(self._lib.sdm_last_path(self._h))

    def coalescence_step_host(self, multiplicity, volume, cell_id, n_cell, dt, dV, kp, seed, step, n_sd=None,
                              compact=False) -> int:
        """Host (ideally pinned) torch CPU tensors in and out; copies are inside the call.  Returns n_sd
        after the optional compaction."""
        t = self._torch
        n = int(multiplicity.shape[0] if n_sd is None else n_sd)
        for x in (multiplicity, volume, cell_id):
            if x.device.type != "cpu":
                raise ValueError("coalescence_step_host takes CPU tensors")
        n_out = C.c_int64(n)
        rc = self._lib.sdm_coalescence_step_host(self._h, _ptr(multiplicity, t.int64), _ptr(volume, t.float64),
                                                 _ptr(cell_id, t.int32), n, int(n_cell), float(dt), float(dV),
                                                 C.byref(kp), int(seed), int(step), int(bool(compact)),
                                                 C.byref(n_out))
        _check(rc, "sdm_coalescence_step_host")
        return int(n_out.value)

    def profile_enable(self, on: bool):
        _check(self._lib.sdm_profile_enable(self._h, int(bool(on))), "sdm_profile_enable")

    def profile_read(self):
        """dict kernel class -> (milliseconds, launches) since the last read."""
        ms = (C.c_double * len(PROF_CLASSES))()
        cnt = (C.c_int64 * len(PROF_CLASSES))()
        _check(self._lib.sdm_profile_read(self._h, ms, cnt), "sdm_profile_read")
        return {name: (float(ms[i]), int(cnt[i])) for i, name in enumerate(PROF_CLASSES)}

    def poll_error(self) -> int:
        return int(self._lib.sdm_poll_error(self._h))

    def launch_count(self) -> int:
        return int(self._lib.sdm_launch_count(self._h))

    def philox_fill(self, seed, step, i0, n):
        t = self._torch
        key = t.empty(n, dtype=t.int32, device=self.device)   # uint32 bit patterns
        u = t.empty(n, dtype=t.float64, device=self.device)
        _check(self._lib.sdm_philox_fill(self._h, int(seed), int(step), int(i0), int(n), key.data_ptr(),
                                         u.data_ptr()), "sdm_philox_fill")
        return key, u

    def kernel_eval(self, kp, vj, vk):
        t = self._torch
        out = t.empty_like(vj)
        _check(self._lib.sdm_kernel_eval(self._h, C.byref(kp), _ptr(vj, t.float64), _ptr(vk, t.float64),
                                         int(vj.shape[0]), out.data_ptr()), "sdm_kernel_eval")
        return out

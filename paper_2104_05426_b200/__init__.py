"""Thin ctypes binding of libjefi.so (include/jefi.h): argument marshalling only.

Every step of the path (pre-pass, pairwise kernel, reduce/scale epilogue) runs in the CUDA
kernels behind the C ABI; PyTorch is used by callers only to allocate device memory and to
supply streams.  There is no CPU fallback: if the shared library has not been built
(``python paper_2104_05426_b200/build.py``) importing this package raises.
The functions carry the names of the C entry points; ``Jefi`` is a small owner object around
them for tests and the bench.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libjefi.so"

JEFI_OK, JEFI_ERR_INVALID_ARG, JEFI_ERR_CUDA, JEFI_ERR_OOM = 0, 1, 2, 3
JEFI_ERR_NO_HISTORY, JEFI_ERR_TIME_RANGE, JEFI_ERR_UNSUPPORTED = 4, 5, 6
JEFI_F32, JEFI_F64 = 0, 1

EXPORTS = (                                   # include/jefi.h: the product ABI
    "jefi_create", "jefi_upload_history", "jefi_upload_history_host", "jefi_fields",
    "jefi_fields_at_time", "jefi_fields_host", "jefi_set_kernel",
    "jefi_device_bytes", "jefi_destroy", "jefi_status_string", "jefi_last_error",
    "jefi_flops_per_pair", "jefi_shard_obs",
    "jefi_append_step", "jefi_append_step_host", "jefi_fields_series", "jefi_fields_series_host",
    "jefi_fields_noalloc", "jefi_reserve_series", "jefi_shard_src",
)
JEFI_NOALLOC_SCRATCH_BYTES, JEFI_NOALLOC_MAX_OBS = 8 * 1024 * 1024, 131072
INSTRUMENT_EXPORTS = (                        # include/jefi_instrument.h: bench / test instrumentation
    "jefi_launch_count", "jefi_measure_alu_peak", "jefi_measure_ffma_operand_rates", "jefi_debug_pair_lags", "jefi_debug_launch_limits",
)


class jefi_grid_desc(C.Structure):
    _fields_ = [("n", C.c_int32 * 3), ("origin", C.c_double * 3), ("spacing", C.c_double * 3)]


class jefi_obs_desc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("grid", jefi_grid_desc), ("npoints", C.c_int64),
                ("points_dev", C.c_void_p)]


class jefi_time_desc(C.Structure):
    _fields_ = [("t0", C.c_double), ("dt", C.c_double), ("c", C.c_double), ("nsteps", C.c_int32),
                ("deriv_mode", C.c_int32), ("past_mode", C.c_int32)]


class JefiError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        name = jefi_status_string(status)
        super().__init__(f"{where}: {name}" + (f" ({detail})" if detail else ""))


if not LIB_PATH.exists():
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python paper_2104_05426_b200/build.py` "
        "(nvcc, sm_100a).  There is no fallback path.")

_lib = C.CDLL(str(LIB_PATH))
_P = C.c_void_p
_lib.jefi_create.argtypes = [C.POINTER(jefi_grid_desc), C.POINTER(jefi_obs_desc),
                             C.POINTER(jefi_time_desc), C.c_int, C.c_int, C.POINTER(_P)]
_lib.jefi_upload_history.argtypes = [_P, _P, _P, _P]
_lib.jefi_upload_history_host.argtypes = [_P, _P, _P, _P]
_lib.jefi_append_step.argtypes = [_P, _P, _P, _P]
_lib.jefi_append_step_host.argtypes = [_P, _P, _P, _P]
_lib.jefi_fields.argtypes = [_P, C.c_int32, C.c_int64, C.c_int64, _P, _P, _P]
_lib.jefi_fields_series.argtypes = [_P, C.c_int32, C.c_int32, C.c_int64, C.c_int64, _P, _P, _P]
_lib.jefi_fields_series_host.argtypes = [_P, C.c_int32, C.c_int32, C.c_int64, C.c_int64, _P, _P, _P]
_lib.jefi_fields_at_time.argtypes = [_P, C.c_double, C.c_int64, C.c_int64, _P, _P, _P]
_lib.jefi_fields_host.argtypes = [_P, C.c_int32, C.c_int64, C.c_int64, _P, _P, _P]
_lib.jefi_set_kernel.argtypes = [_P, C.c_int32]
_lib.jefi_reserve_series.argtypes = [_P, C.c_int32, C.c_int64, C.c_int32]
_lib.jefi_fields_noalloc.argtypes = [C.POINTER(jefi_grid_desc), C.POINTER(jefi_obs_desc), C.POINTER(jefi_time_desc),
                                     C.c_int, C.c_int32, _P, _P, C.c_int64, C.c_int64, _P, _P, _P, C.c_char_p,
                                     C.c_int32]
_lib.jefi_launch_count.argtypes = [_P]
_lib.jefi_launch_count.restype = C.c_int64
_lib.jefi_device_bytes.argtypes = [_P]
_lib.jefi_device_bytes.restype = C.c_int64
_lib.jefi_destroy.argtypes = [_P]
_lib.jefi_status_string.argtypes = [C.c_int]
_lib.jefi_status_string.restype = C.c_char_p
_lib.jefi_last_error.argtypes = [_P]
_lib.jefi_last_error.restype = C.c_char_p
_lib.jefi_flops_per_pair.argtypes = []
_lib.jefi_measure_alu_peak.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double)]
_lib.jefi_shard_obs.argtypes = [C.POINTER(jefi_obs_desc), C.c_int32, C.c_int32, C.POINTER(C.c_int64),
                                C.POINTER(C.c_int64)]
_lib.jefi_shard_src.argtypes = [C.POINTER(jefi_grid_desc), C.c_int32, C.c_int32, C.POINTER(jefi_grid_desc),
                                C.POINTER(C.c_int64)]
_lib.jefi_measure_ffma_operand_rates.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
_lib.jefi_debug_pair_lags.argtypes = [_P, C.c_int32, C.c_int64, _P, _P, _P, _P]
_lib.jefi_debug_launch_limits.argtypes = [_P, C.c_int64, C.c_int64]
for _n in EXPORTS + INSTRUMENT_EXPORTS:
    if _n not in ("jefi_launch_count", "jefi_device_bytes", "jefi_status_string", "jefi_last_error"):
        getattr(_lib, _n).restype = C.c_int


def _ptr(x):
    """Device/host address of a torch tensor or numpy array, or a raw int / None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError(f"cannot take the address of {type(x)!r}")


def _stream(s):
    if s is None:
        return None
    return s if isinstance(s, int) else int(s.cuda_stream)


def make_grid(n, origin, spacing) -> jefi_grid_desc:
    g = jefi_grid_desc()
    g.n[:] = [int(v) for v in n]
    g.origin[:] = [float(v) for v in origin]
    g.spacing[:] = [float(v) for v in spacing]
    return g


# ------------------------------------------------------------------ the C entry points
def jefi_status_string(status: int) -> str:
    return _lib.jefi_status_string(int(status)).decode()


def jefi_last_error(ctx) -> str:
    return _lib.jefi_last_error(ctx).decode() if ctx else ""


def jefi_flops_per_pair() -> int:
    return int(_lib.jefi_flops_per_pair())


def jefi_create(src: jefi_grid_desc, obs: jefi_obs_desc, time: jefi_time_desc, dtype: int, device: int):
    out = _P()
    st = _lib.jefi_create(C.byref(src) if src is not None else None,
                          C.byref(obs) if obs is not None else None,
                          C.byref(time) if time is not None else None, int(dtype), int(device), C.byref(out))
    if st != JEFI_OK:
        raise JefiError(st, "jefi_create")
    return out


def _check(st, ctx, where):
    if st != JEFI_OK:
        raise JefiError(st, where, jefi_last_error(ctx))


def jefi_upload_history(ctx, rho_dev, J_dev, stream=None):
    _check(_lib.jefi_upload_history(ctx, _ptr(rho_dev), _ptr(J_dev), _stream(stream)), ctx, "jefi_upload_history")


def jefi_upload_history_host(ctx, rho_host, J_host, stream=None):
    _check(_lib.jefi_upload_history_host(ctx, _ptr(rho_host), _ptr(J_host), _stream(stream)), ctx,
           "jefi_upload_history_host")


def jefi_append_step(ctx, rho_new_dev, J_new_dev, stream=None):
    _check(_lib.jefi_append_step(ctx, _ptr(rho_new_dev), _ptr(J_new_dev), _stream(stream)), ctx, "jefi_append_step")


def jefi_append_step_host(ctx, rho_new_host, J_new_host, stream=None):
    _check(_lib.jefi_append_step_host(ctx, _ptr(rho_new_host), _ptr(J_new_host), _stream(stream)), ctx,
           "jefi_append_step_host")


def jefi_fields(ctx, step, obs_begin, obs_count, E_out_dev, B_out_dev, stream=None):
    _check(_lib.jefi_fields(ctx, int(step), int(obs_begin), int(obs_count), _ptr(E_out_dev), _ptr(B_out_dev),
                            _stream(stream)), ctx, "jefi_fields")


def jefi_fields_series(ctx, step_begin, step_count, obs_begin, obs_count, E_out_dev, B_out_dev, stream=None):
    _check(_lib.jefi_fields_series(ctx, int(step_begin), int(step_count), int(obs_begin), int(obs_count),
                                   _ptr(E_out_dev), _ptr(B_out_dev), _stream(stream)), ctx, "jefi_fields_series")


def jefi_fields_series_host(ctx, step_begin, step_count, obs_begin, obs_count, E_out_host, B_out_host, stream=None):
    _check(_lib.jefi_fields_series_host(ctx, int(step_begin), int(step_count), int(obs_begin), int(obs_count),
                                        _ptr(E_out_host), _ptr(B_out_host), _stream(stream)), ctx,
           "jefi_fields_series_host")


def jefi_reserve_series(ctx, max_steps, max_obs, host_staging=False):
    _check(_lib.jefi_reserve_series(ctx, int(max_steps), int(max_obs), 1 if host_staging else 0), ctx,
           "jefi_reserve_series")


def jefi_fields_at_time(ctx, t, obs_begin, obs_count, E_out_dev, B_out_dev, stream=None):
    _check(_lib.jefi_fields_at_time(ctx, float(t), int(obs_begin), int(obs_count), _ptr(E_out_dev),
                                    _ptr(B_out_dev), _stream(stream)), ctx, "jefi_fields_at_time")


def jefi_fields_host(ctx, step, obs_begin, obs_count, E_out_host, B_out_host, stream=None):
    _check(_lib.jefi_fields_host(ctx, int(step), int(obs_begin), int(obs_count), _ptr(E_out_host),
                                 _ptr(B_out_host), _stream(stream)), ctx, "jefi_fields_host")


def jefi_fields_noalloc(src: jefi_grid_desc, obs: jefi_obs_desc, time: jefi_time_desc, dtype: int, step: int,
                        rho_dev, J_dev, obs_begin, obs_count, E_out_dev, B_out_dev, stream=None):
    """E, B of one step on the current device without a context and without any device
    allocation (for hosts that cannot cudaMalloc: all memory already pooled by the application,
    or a loop that must not stall).  The caller passes the raw history and the outputs; at most
    JEFI_NOALLOC_MAX_OBS points per call; calls that overlap on the GPU race on the library's
    one fixed scratch array.  See include/jefi.h."""
    msg = C.create_string_buffer(512)
    st = _lib.jefi_fields_noalloc(C.byref(src) if src is not None else None,
                                  C.byref(obs) if obs is not None else None,
                                  C.byref(time) if time is not None else None, int(dtype), int(step),
                                  _ptr(rho_dev), _ptr(J_dev), int(obs_begin), int(obs_count), _ptr(E_out_dev),
                                  _ptr(B_out_dev), _stream(stream), msg, len(msg))
    if st != JEFI_OK:
        raise JefiError(st, "jefi_fields_noalloc", msg.value.decode())


def jefi_set_kernel(ctx, which: int):
    _check(_lib.jefi_set_kernel(ctx, int(which)), ctx, "jefi_set_kernel")


def jefi_launch_count(ctx) -> int:
    return int(_lib.jefi_launch_count(ctx))


def jefi_device_bytes(ctx) -> int:
    return int(_lib.jefi_device_bytes(ctx))


def jefi_destroy(ctx):
    st = _lib.jefi_destroy(ctx)
    if st != JEFI_OK:
        raise JefiError(st, "jefi_destroy")


def jefi_measure_alu_peak(device: int, dtype: int) -> float:
    v = C.c_double()
    st = _lib.jefi_measure_alu_peak(int(device), int(dtype), C.byref(v))
    if st != JEFI_OK:
        raise JefiError(st, "jefi_measure_alu_peak")
    return v.value


def jefi_measure_ffma_operand_rates(device: int):
    """(two fresh registers + one reused, three fresh registers) FFMA rates in TFLOP/s."""
    a, b = C.c_double(), C.c_double()
    st = _lib.jefi_measure_ffma_operand_rates(int(device), C.byref(a), C.byref(b))
    if st != JEFI_OK:
        raise JefiError(st, "jefi_measure_ffma_operand_rates")
    return a.value, b.value


def jefi_debug_pair_lags(ctx, which: int, n_pairs: int, obs_index_dev, cell_index_dev, lag_out_dev, stream=None):
    _check(_lib.jefi_debug_pair_lags(ctx, int(which), int(n_pairs), _ptr(obs_index_dev), _ptr(cell_index_dev),
                                     _ptr(lag_out_dev), _stream(stream)), ctx, "jefi_debug_pair_lags")


def jefi_debug_launch_limits(ctx, scratch_elems: int = 0, chunk_bytes: int = 0):
    _check(_lib.jefi_debug_launch_limits(ctx, int(scratch_elems), int(chunk_bytes)), ctx, "jefi_debug_launch_limits")


def jefi_shard_obs(obs: jefi_obs_desc, rank: int, world: int):
    """(begin, count) of the observation slice rank `rank` of `world` evaluates."""
    b, n = C.c_int64(), C.c_int64()
    st = _lib.jefi_shard_obs(C.byref(obs) if obs is not None else None, int(rank), int(world), C.byref(b),
                             C.byref(n))
    if st != JEFI_OK:
        raise JefiError(st, "jefi_shard_obs")
    return b.value, n.value


def jefi_shard_src(src: jefi_grid_desc, rank: int, world: int):
    """(slab descriptor, cell_begin) of the source z-layers rank `rank` of `world` owns."""
    slab, cb = jefi_grid_desc(), C.c_int64()
    st = _lib.jefi_shard_src(C.byref(src) if src is not None else None, int(rank), int(world), C.byref(slab),
                             C.byref(cb))
    if st != JEFI_OK:
        raise JefiError(st, "jefi_shard_src")
    return slab, cb.value


def make_obs_grid(n, origin, spacing) -> jefi_obs_desc:
    obs = jefi_obs_desc()
    obs.kind = 0
    obs.grid = make_grid(n, origin, spacing)
    return obs


# ------------------------------------------------------------------ owner object
class Jefi:
    """Owns one jefi_ctx.  ``n_src``/``origin_src``/``spacing_src`` describe the source grid,
    the observation set is a regular grid (``n_obs``, ``origin_obs``, ``spacing_obs``) or, with
    ``points_dev`` (a device tensor [n,3] of the context dtype), an explicit list."""

    def __init__(self, n_src, origin_src, spacing_src, *, dt, c, nsteps, dtype, n_obs=None, origin_obs=None,
                 spacing_obs=None, points_dev=None, t0=0.0, deriv_mode=0, device=0):
        self.dtype = {"f32": JEFI_F32, "f64": JEFI_F64}.get(dtype, dtype)
        src = make_grid(n_src, origin_src, spacing_src)
        obs = jefi_obs_desc()
        if points_dev is None:
            obs.kind = 0
            obs.grid = make_grid(n_obs, origin_obs, spacing_obs)
            self.n_points = int(n_obs[0]) * int(n_obs[1]) * int(n_obs[2])
        else:
            obs.kind = 1
            obs.grid = make_grid((1, 1, 1), (0, 0, 0), (1, 1, 1))
            obs.npoints = int(points_dev.shape[0])
            obs.points_dev = _ptr(points_dev)
            self._keep = points_dev
            self.n_points = obs.npoints
        tm = jefi_time_desc(float(t0), float(dt), float(c), int(nsteps), int(deriv_mode), 0)
        self.ctx = jefi_create(src, obs, tm, self.dtype, device)

    def upload_history(self, rho_dev, J_dev, stream=None):
        jefi_upload_history(self.ctx, rho_dev, J_dev, stream)

    def upload_history_host(self, rho_host, J_host, stream=None):
        jefi_upload_history_host(self.ctx, rho_host, J_host, stream)

    def append_step(self, rho_new_dev, J_new_dev, stream=None):
        jefi_append_step(self.ctx, rho_new_dev, J_new_dev, stream)

    def append_step_host(self, rho_new_host, J_new_host, stream=None):
        jefi_append_step_host(self.ctx, rho_new_host, J_new_host, stream)

    def fields(self, step, E_out_dev, B_out_dev, obs_begin=0, obs_count=None, stream=None):
        n = self.n_points - obs_begin if obs_count is None else obs_count
        jefi_fields(self.ctx, step, obs_begin, n, E_out_dev, B_out_dev, stream)

    def fields_series(self, step_begin, step_count, E_out_dev, B_out_dev, obs_begin=0, obs_count=None, stream=None):
        n = self.n_points - obs_begin if obs_count is None else obs_count
        jefi_fields_series(self.ctx, step_begin, step_count, obs_begin, n, E_out_dev, B_out_dev, stream)

    def fields_series_host(self, step_begin, step_count, E_out_host, B_out_host, obs_begin=0, obs_count=None,
                           stream=None):
        n = self.n_points - obs_begin if obs_count is None else obs_count
        jefi_fields_series_host(self.ctx, step_begin, step_count, obs_begin, n, E_out_host, B_out_host, stream)

    def reserve_series(self, max_steps, max_obs=None, host_staging=False):
        jefi_reserve_series(self.ctx, max_steps, self.n_points if max_obs is None else max_obs, host_staging)

    def fields_host(self, step, E_out_host, B_out_host, obs_begin=0, obs_count=None, stream=None):
        n = self.n_points - obs_begin if obs_count is None else obs_count
        jefi_fields_host(self.ctx, step, obs_begin, n, E_out_host, B_out_host, stream)

    def set_kernel(self, which):
        jefi_set_kernel(self.ctx, which)

    @property
    def launches(self):
        return jefi_launch_count(self.ctx)

    def close(self):
        if self.ctx is not None:
            ctx, self.ctx = self.ctx, None
            jefi_destroy(ctx)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

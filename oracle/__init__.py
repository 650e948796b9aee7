"""fp64 CPU oracle for the discretised Jefimenko sums (Eq. (4)-(6)).

TEST INFRASTRUCTURE, NOT PRODUCT.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package.  It
shares nothing with the CUDA path (``paper_2104_05426_b200``) and neither imports the other.

The arithmetic lives in ``jefi_oracle.c`` (plain C, triple loop, libc only); this module only
compiles it with gcc and marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "jefi_oracle.c"
_LIB = _HERE / "libjefi_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile the C oracle (-O2, no fast-math: IEEE semantics are part of the definition)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fno-fast-math", "-ffp-contract=off",
             "-o", str(tmp), str(_SRC), "-lm", "-lpthread"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        lib.jefi_oracle_fields.restype = ctypes.c_int
        lib.jefi_oracle_fields.argtypes = [
            ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double),
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int,
            ctypes.c_double, ctypes.c_double, ctypes.c_int, ctypes.c_int,
            ctypes.c_long, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int,
        ]
        lib.jefi_oracle_lag.restype = ctypes.c_long
        lib.jefi_oracle_lag.argtypes = [ctypes.c_double] * 8
        _lib = lib
    return _lib


def host_cores() -> int:
    return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)


def fields(n_src, origin_src, spacing_src, rho, J, *, dt, c, step, obs_xyz,
           deriv_mode: int = 0, nthreads: int | None = None):
    """E, B (each ``[3][n_obs]`` float64) at the explicit points ``obs_xyz[n_obs][3]``.

    ``rho``: ``[T, nz, ny, nx]`` (or ``[T, N_s]``), ``J``: ``[T, 3, nz, ny, nx]``; float64, or
    float32 (promoted element-wise to double inside the oracle: an fp32 run's inputs are the
    fp32-rounded values, nothing else is rounded).  ``origin_src`` is the centre of cell (0,0,0).
    """
    lib = _load()
    rho = np.ascontiguousarray(rho)
    J = np.ascontiguousarray(J)
    if rho.dtype != J.dtype or rho.dtype not in (np.float32, np.float64):
        raise TypeError("rho and J must both be float32 or both float64")
    nx, ny, nz = (int(v) for v in n_src)
    Ns = nx * ny * nz
    T = int(rho.shape[0])
    if rho.size != T * Ns or J.size != T * 3 * Ns or J.shape[0] != T:
        raise ValueError("rho must be [T][N_s] and J [T][3][N_s]")
    obs = np.ascontiguousarray(obs_xyz, dtype=np.float64).reshape(-1, 3)
    n_obs = obs.shape[0]
    E = np.zeros((3, n_obs), dtype=np.float64)
    B = np.zeros((3, n_obs), dtype=np.float64)
    n_arr = (ctypes.c_int * 3)(nx, ny, nz)
    o_arr = (ctypes.c_double * 3)(*[float(v) for v in origin_src])
    h_arr = (ctypes.c_double * 3)(*[float(v) for v in spacing_src])
    if nthreads is None:
        nthreads = host_cores()
    rc = lib.jefi_oracle_fields(
        n_arr, o_arr, h_arr, rho.ctypes.data, J.ctypes.data, int(rho.dtype == np.float32), T,
        float(dt), float(c), int(deriv_mode), int(step), n_obs,
        obs.ctypes.data, E.ctypes.data, B.ctypes.data, int(nthreads),
    )
    if rc != 0:
        raise ValueError("jefi_oracle_fields: invalid arguments")
    return E, B


def lag(r, s, *, dt, c) -> int:
    """k = floor(|r-s|/(c dt) + 0.5) in fp64 (reading Q3)."""
    return int(_load().jefi_oracle_lag(*[float(v) for v in r], *[float(v) for v in s], float(dt), float(c)))

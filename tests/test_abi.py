"""The C-ABI library loads and exports every symbol include/jefi.h declares, and rejects bad
arguments before touching the device (no compute calls: runs without a GPU)."""
import ctypes as C
import os
import re

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)


@pytest.fixture(scope="module")
def jb():
    import __graft_entry__
    __graft_entry__.build()          # loads build.py by path (the package raises without its .so)
    import paper_2104_05426_b200 as jb
    return jb


def _declared_symbols(header="jefi.h"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(jefi_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported(jb):
    names = _declared_symbols()
    assert len(names) >= 12
    lib = C.CDLL(str(jb.LIB_PATH))
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/jefi.h but not exported"
    assert set(names) == set(jb.EXPORTS)
    # measurement / test instrumentation lives in its own header, outside the product ABI
    extra = _declared_symbols("jefi_instrument.h")
    for n in extra:
        assert hasattr(lib, n), f"{n} declared in include/jefi_instrument.h but not exported"
    assert set(extra) == set(jb.INSTRUMENT_EXPORTS) and not set(extra) & set(names)


def test_binding_has_same_names(jb):
    for n in _declared_symbols() + _declared_symbols("jefi_instrument.h"):
        assert callable(getattr(jb, n)), n


def test_flops_per_pair_and_status_strings(jb):
    assert jb.jefi_flops_per_pair() == 52
    assert jb.jefi_status_string(0) == "JEFI_OK"
    assert jb.jefi_status_string(jb.JEFI_ERR_TIME_RANGE) == "JEFI_ERR_TIME_RANGE"
    assert jb.jefi_last_error(None) == ""


def _descs(jb, n=(4, 4, 4), h=(0.1, 0.1, 0.1), dt=0.05, c=1.0, T=8):
    src = jb.make_grid(n, (0, 0, 0), h)
    obs = jb.jefi_obs_desc()
    obs.kind = 0
    obs.grid = jb.make_grid(n, (0, 0, 0), h)
    tm = jb.jefi_time_desc(0.0, dt, c, T, 0, 0)
    return src, obs, tm


@pytest.mark.parametrize("mutate,status", [
    (lambda s, o, t: s.n.__setitem__(1, 0), 1),
    (lambda s, o, t: s.spacing.__setitem__(2, -0.1), 1),
    (lambda s, o, t: s.origin.__setitem__(0, float("nan")), 1),
    (lambda s, o, t: setattr(o, "kind", 7), 1),
    (lambda s, o, t: o.grid.n.__setitem__(0, -3), 1),
    (lambda s, o, t: setattr(t, "dt", 0.0), 1),
    (lambda s, o, t: setattr(t, "c", -1.0), 1),
    (lambda s, o, t: setattr(t, "nsteps", 0), 1),
    (lambda s, o, t: setattr(t, "deriv_mode", 2), 1),
    (lambda s, o, t: setattr(t, "past_mode", 1), 6),
])
def test_create_rejects_bad_descriptors_before_any_cuda_call(jb, mutate, status):
    src, obs, tm = _descs(jb)
    mutate(src, obs, tm)
    with pytest.raises(jb.JefiError) as e:
        jb.jefi_create(src, obs, tm, jb.JEFI_F32, 0)
    assert e.value.status == status


def test_create_rejects_null_and_bad_dtype(jb):
    src, obs, tm = _descs(jb)
    for args in ((None, obs, tm, 0, 0), (src, None, tm, 0, 0), (src, obs, None, 0, 0), (src, obs, tm, 5, 0),
                 (src, obs, tm, 0, -1)):
        with pytest.raises(jb.JefiError) as e:
            jb.jefi_create(*args)
        assert e.value.status == jb.JEFI_ERR_INVALID_ARG


def test_create_refuses_sizes_beyond_the_index_range(jb):
    """2^31 source cells exceed the 32-bit cell index of the kernels: refused before any
    allocation (JEFI_ERR_UNSUPPORTED), as is an observation set of 2^40 points."""
    src, obs, tm = _descs(jb, n=(2048, 2048, 512))
    obs.grid = jb.make_grid((4, 4, 4), (0, 0, 0), (0.1, 0.1, 0.1))
    with pytest.raises(jb.JefiError) as e:
        jb.jefi_create(src, obs, tm, jb.JEFI_F32, 0)
    assert e.value.status == jb.JEFI_ERR_UNSUPPORTED
    src, obs, tm = _descs(jb)
    pts = jb.jefi_obs_desc()
    pts.kind, pts.npoints, pts.points_dev = 1, 1 << 40, 16
    pts.grid = jb.make_grid((1, 1, 1), (0, 0, 0), (1, 1, 1))
    with pytest.raises(jb.JefiError) as e:
        jb.jefi_create(src, pts, tm, jb.JEFI_F32, 0)
    assert e.value.status == jb.JEFI_ERR_UNSUPPORTED


def test_append_and_shard_reject_null_arguments(jb):
    lib = C.CDLL(str(jb.LIB_PATH))
    lib.jefi_append_step.argtypes = [C.c_void_p] * 4
    lib.jefi_append_step_host.argtypes = [C.c_void_p] * 4
    assert lib.jefi_append_step(None, None, None, None) == jb.JEFI_ERR_INVALID_ARG
    assert lib.jefi_append_step_host(None, None, None, None) == jb.JEFI_ERR_INVALID_ARG
    lib.jefi_shard_obs.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
    assert lib.jefi_shard_obs(None, 0, 1, None, None) == jb.JEFI_ERR_INVALID_ARG


def test_null_context_is_an_error_not_a_crash(jb):
    lib = C.CDLL(str(jb.LIB_PATH))
    lib.jefi_fields.argtypes = [C.c_void_p, C.c_int32, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
    assert lib.jefi_fields(None, 0, 0, 0, None, None, None) == jb.JEFI_ERR_INVALID_ARG
    lib.jefi_upload_history.argtypes = [C.c_void_p] * 4
    assert lib.jefi_upload_history(None, None, None, None) == jb.JEFI_ERR_INVALID_ARG
    lib.jefi_destroy.argtypes = [C.c_void_p]
    assert lib.jefi_destroy(None) == jb.JEFI_ERR_INVALID_ARG
    lib.jefi_measure_alu_peak.argtypes = [C.c_int, C.c_int, C.c_void_p]
    assert lib.jefi_measure_alu_peak(0, 0, None) == jb.JEFI_ERR_INVALID_ARG


def test_series_and_instrument_entry_points_reject_null_arguments(jb):
    lib = C.CDLL(str(jb.LIB_PATH))
    P = C.c_void_p
    lib.jefi_fields_series.argtypes = [P, C.c_int32, C.c_int32, C.c_int64, C.c_int64, P, P, P]
    lib.jefi_fields_series_host.argtypes = [P, C.c_int32, C.c_int32, C.c_int64, C.c_int64, P, P, P]
    assert lib.jefi_fields_series(None, 0, 4, 0, 0, None, None, None) == jb.JEFI_ERR_INVALID_ARG
    assert lib.jefi_fields_series_host(None, 0, 4, 0, 0, None, None, None) == jb.JEFI_ERR_INVALID_ARG
    lib.jefi_debug_pair_lags.argtypes = [P, C.c_int32, C.c_int64, P, P, P, P]
    assert lib.jefi_debug_pair_lags(None, 2, 1, None, None, None, None) == jb.JEFI_ERR_INVALID_ARG
    lib.jefi_debug_launch_limits.argtypes = [P, C.c_int64, C.c_int64]
    assert lib.jefi_debug_launch_limits(None, 1, 1) == jb.JEFI_ERR_INVALID_ARG
    lib.jefi_measure_ffma_operand_rates.argtypes = [C.c_int, P, P]
    assert lib.jefi_measure_ffma_operand_rates(0, None, None) == jb.JEFI_ERR_INVALID_ARG
    lib.jefi_launch_count.argtypes = [P]
    lib.jefi_launch_count.restype = C.c_int64
    assert lib.jefi_launch_count(None) == 0
    lib.jefi_set_kernel.argtypes = [P, C.c_int32]
    assert lib.jefi_set_kernel(None, 3) == jb.JEFI_ERR_INVALID_ARG
    lib.jefi_reserve_series.argtypes = [P, C.c_int32, C.c_int64, C.c_int32]
    assert lib.jefi_reserve_series(None, 1, 1, 0) == jb.JEFI_ERR_INVALID_ARG


def test_create_rejects_a_point_list_without_positions(jb):
    src, obs, tm = _descs(jb)
    pts = jb.jefi_obs_desc()
    pts.kind, pts.npoints, pts.points_dev = 1, 100, None
    pts.grid = jb.make_grid((1, 1, 1), (0, 0, 0), (1, 1, 1))
    with pytest.raises(jb.JefiError) as e:
        jb.jefi_create(src, pts, tm, jb.JEFI_F32, 0)
    assert e.value.status == jb.JEFI_ERR_INVALID_ARG
    pts.npoints = -1
    with pytest.raises(jb.JefiError) as e:
        jb.jefi_create(src, pts, tm, jb.JEFI_F32, 0)
    assert e.value.status == jb.JEFI_ERR_INVALID_ARG


def test_product_does_not_import_the_oracle():
    """The product path must never route through oracle/ (or workloads' arithmetic-free data)."""
    pkg = os.path.join(ROOT, "paper_2104_05426_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "jefi_oracle" not in text, f

"""Parity of the time-blocked kernel (csrc/pairwise_series.cu: NS
consecutive output steps per (observation point, source cell) pair, raw 16-byte records,
time differences formed in registers) against the fp64 CPU oracle, step by step, through
jefi_fields_series.  jefi_set_kernel(3) = time-blocked kernel or JEFI_ERR_UNSUPPORTED, so a
silent fallback to the one-step kernel cannot pass these tests.  Same bars as everywhere:
rel-L2 per component <= 1e-5 (fp64) / 2e-4 (fp32) plus the pointwise bound of check()."""
import numpy as np
import pytest

import workloads as wl
from gpu_util import gpu_fields, gpu_fields_series, make_ctx, oracle_fields, upload
from test_parity_gpu import c4_oracle_plan, check

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def jb():
    import __graft_entry__
    __graft_entry__.build()
    import paper_2104_05426_b200 as jb
    return jb


def series_case(jb, w, step_begin, step_count, deriv_mode=0, obs_begin=0, obs_count=None, limits=None, what="",
                comp_floor=1e-12):
    ctx = make_ctx(w, jb, deriv_mode)
    try:
        ctx.set_kernel(3)
        if limits:
            jb.jefi_debug_launch_limits(ctx.ctx, *limits)
        upload(ctx, w)
        E, B = gpu_fields_series(ctx, w, step_begin, step_count, obs_begin, obs_count)
        n = w.N_o - obs_begin if obs_count is None else obs_count
        idx = np.arange(obs_begin, obs_begin + n)
        for k in range(step_count):
            Eo, Bo = oracle_fields(w, step_begin + k, idx, deriv_mode)
            check(w, E[k], B[k], Eo, Bo, None, f"{what} series step {step_begin + k} mode {deriv_mode}", comp_floor)
        return E, B
    finally:
        ctx.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
@pytest.mark.parametrize("deriv_mode", [0, 1])
def test_series_from_step_zero_every_step(jb, dtype, deriv_mode):
    """All T steps of a white-noise history in one call, from step 0: the early blocks have most
    of the light cone before the stored history (m < 0 -> zero, Q4: the EDGE path in centred mode,
    the zero slots in backward mode), the first records use the one-sided difference (ghost
    slot), the last block ends on the newest step (ghost slot at the other end); T = 37 is not a
    multiple of the block length, so the last block is ragged."""
    w = wl.random_history((6, 5, 4), 37, seed=81, dtype=dtype, n_obs=(7, 6, 5), dt=0.05)
    series_case(jb, w, 0, 37, deriv_mode, what=f"from zero {dtype}")


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_series_ragged_anisotropic_grids_with_c_and_subranges(jb, dtype):
    w = wl.random_history((13, 5, 7), 40, seed=77, dtype=dtype, spacing=(0.1, 0.15, 0.07),
                          n_obs=(9, 11, 3), spacing_obs=(0.12, 0.05, 0.2), origin_obs=(-0.31, -0.22, 0.13),
                          dt=0.02, c=1.7)
    for mode in (0, 1):
        series_case(jb, w, 11, 23, mode, what="ragged")
        series_case(jb, w, 30, 10, mode, obs_begin=37, obs_count=201, what="ragged sub-range")
    # a plane-shaped observation set (the plane tile) and a single row
    w2 = wl.random_history((6, 5, 4), 30, seed=83, dtype=dtype, n_obs=(19, 13, 1), dt=0.05)
    series_case(jb, w2, 3, 27, what="plane")
    w3 = wl.random_history((6, 5, 4), 30, seed=85, dtype=dtype, n_obs=(5, 1, 1), dt=0.05)
    series_case(jb, w3, 0, 30, what="row")


def test_series_single_stored_step_and_overlapping_grid(jb):
    """T = 1 (derivative 0: both ghost slots equal f[0]); obs == source centres (self cell at
    R = 0, the screening rule inside a block)."""
    w = wl.random_history((1, 1, 1), 1, seed=9, dtype="f64", n_obs=(3, 2, 2), spacing_obs=(0.01, 0.01, 0.01),
                          origin_obs=(0.2, 0.0, 0.0), dt=10.0)
    ctx = make_ctx(w, jb)
    try:
        upload(ctx, w)                       # a 1-step series is below the block threshold: one-step kernel
        E, B = gpu_fields_series(ctx, w, 0, 1)
        Eo, Bo = oracle_fields(w, 0)
        check(w, E[0], B[0], Eo, Bo)
    finally:
        ctx.close()
    w = wl.random_history((2, 1, 1), 2, seed=10, dtype="f64", n_obs=(3, 2, 2), spacing_obs=(0.03, 0.03, 0.03),
                          origin_obs=(0.2, 0.0, 0.0), dt=10.0)
    series_case(jb, w, 0, 2, 0, what="T=2")
    series_case(jb, w, 0, 2, 1, what="T=2")
    w = wl.random_history((6, 6, 6), 24, seed=5, dtype="f64", spacing=(0.1, 0.1, 0.1), dt=0.05)
    series_case(jb, w, 2, 22, what="overlapping")
    w = wl.random_history((6, 6, 6), 24, seed=5, dtype="f32", spacing=(0.1, 0.1, 0.1), dt=0.05)
    series_case(jb, w, 0, 24, what="overlapping f32")


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_series_batches_and_accumulating_launches(jb, dtype):
    """Scratch capped so that (a) the steps go in several batches and (b) the source chunks of
    a batch are spread over accumulating launches."""
    w = wl.random_history((12, 10, 9), 60, seed=71, dtype=dtype, n_obs=(9, 8, 10), dt=0.05)
    series_case(jb, w, 20, 40, limits=(17 * 6 * w.N_o, 24 * 1024), what="batches+accumulate")


def test_series_long_windows(jb):
    """dx/(c dt) = 20: ~250-step windows plus the block; history shorter than the longest lag."""
    w = wl.random_history((5, 4, 3), 300, seed=51, dtype="f32", n_obs=(10, 8, 8), dt=0.005)
    series_case(jb, w, 280, 20, what="long windows")
    series_case(jb, w, 0, 9, 1, what="long windows, start")


def test_series_matches_single_step_calls_and_errors(jb):
    import torch
    w = wl.random_history((8, 6, 5), 20, seed=31, dtype="f32", n_obs=(7, 5, 3), dt=0.05)
    ctx = make_ctx(w, jb)
    try:
        upload(ctx, w)
        Es, Bs = gpu_fields_series(ctx, w, 4, 16)
        for k in (0, 7, 15):
            E1, B1 = gpu_fields(ctx, w, 4 + k)
            np.testing.assert_allclose(Es[k], E1, rtol=0, atol=2e-5 * np.abs(E1).max())
            np.testing.assert_allclose(Bs[k], B1, rtol=0, atol=2e-5 * np.abs(B1).max())
        E = torch.empty((20, 3, w.N_o), dtype=torch.float32, device="cuda")
        with pytest.raises(jb.JefiError) as e:
            ctx.fields_series(10, 11, E, torch.empty_like(E))
        assert e.value.status == jb.JEFI_ERR_TIME_RANGE
        # host-buffer entry point: the same values, through the context's staging (grown on demand)
        for begin, count in ((4, 16), (0, 20), (7, 3)):
            Eh = torch.empty((count, 3, w.N_o), dtype=torch.float32).pin_memory()
            Bh = torch.empty_like(Eh).pin_memory()
            ctx.fields_series_host(begin, count, Eh, Bh)
            torch.cuda.synchronize()
            Ed, Bd = gpu_fields_series(ctx, w, begin, count)
            np.testing.assert_array_equal(Eh.numpy().astype(np.float64), Ed)
            np.testing.assert_array_equal(Bh.numpy().astype(np.float64), Bd)
        with pytest.raises(jb.JefiError) as e:
            jb.jefi_fields_series_host(ctx.ctx, 0, 4, 0, w.N_o, None, Bh)
        assert e.value.status == jb.JEFI_ERR_INVALID_ARG
        # after an append the series layout is rebuilt
        ctx.append_step(torch.from_numpy(w.rho[3]).cuda(), torch.from_numpy(w.J[3]).cuda())
        Es2, _ = gpu_fields_series(ctx, w, 4, 16)
        E1, _ = gpu_fields(ctx, w, 19)
        np.testing.assert_allclose(Es2[15], E1, rtol=0, atol=2e-5 * np.abs(E1).max())
        assert not np.allclose(Es2[15], Es[15])
    finally:
        ctx.close()
    pts = np.zeros((5, 3)); pts[:, 0] = 1.0 + np.arange(5)
    ctx = make_ctx(w, jb, points=pts)
    try:
        ctx.set_kernel(3)
        upload(ctx, w)
        E = torch.empty((8, 3, 5), dtype=torch.float32, device="cuda")
        ctx.fields_series(0, 8, E, torch.empty_like(E))       # point lists: one-step per-point kernel
        torch.cuda.synchronize()
        assert torch.isfinite(E).all()
    finally:
        ctx.close()


def test_reserve_series_makes_the_series_calls_allocation_free(jb):
    """include/jefi.h: after jefi_reserve_series the series entry points within the reserved limits
    neither allocate nor free (jefi_device_bytes, which counts every buffer of the context, is constant),
    and the results are those of an unreserved context.  Without the reserve call the first series
    call grows the context (the documented lazy behaviour)."""
    import torch
    w = wl.random_history((9, 8, 7), 48, seed=77, dtype="f32", n_obs=(12, 11, 10), dt=0.05)
    ref_ctx = make_ctx(w, jb)
    ctx = make_ctx(w, jb)
    try:
        upload(ref_ctx, w)
        upload(ctx, w)
        before = jb.jefi_device_bytes(ref_ctx.ctx)
        Er, Br = gpu_fields_series(ref_ctx, w, 0, 48)
        assert jb.jefi_device_bytes(ref_ctx.ctx) > before            # lazy: layout (+ scratch) on first use

        with pytest.raises(jb.JefiError) as e:
            ctx.reserve_series(49)
        assert e.value.status == jb.JEFI_ERR_INVALID_ARG
        ctx.reserve_series(48, host_staging=True)
        reserved = jb.jefi_device_bytes(ctx.ctx)
        assert reserved > before
        E = torch.empty((48, 3, w.N_o), dtype=torch.float32, device="cuda")
        B = torch.empty_like(E)
        Eh = torch.empty((48, 3, w.N_o), dtype=torch.float32).pin_memory()
        Bh = torch.empty_like(Eh).pin_memory()
        ctx.fields_series(0, 48, E, B)
        ctx.fields_series(5, 17, E, B, 100, 333)
        ctx.fields_series_host(0, 48, Eh, Bh)
        torch.cuda.synchronize()
        assert jb.jefi_device_bytes(ctx.ctx) == reserved
        np.testing.assert_array_equal(Eh.numpy().astype(np.float64), Er)
        np.testing.assert_array_equal(Bh.numpy().astype(np.float64), Br)
        ctx.reserve_series(10, 5)                                     # smaller limits: nothing shrinks or grows
        assert jb.jefi_device_bytes(ctx.ctx) == reserved
    finally:
        ctx.close()
        ref_ctx.close()


# ------------------------------------------------------------------ config 4, all 128 output steps
def test_series_config4_all_128_steps(jb):
    """BASELINE.json configs[3]: the 128-step time series of the detached plane in ONE call,
    every step against the oracle (four steps on every point, the rest on the seeded subset;
    the oracle results are the ones test_config4_detached_plane_time_series computed)."""
    w = wl.config4_detached()
    full, idx = c4_oracle_plan(w)
    ctx = make_ctx(w, jb)
    try:
        ctx.set_kernel(3)
        upload(ctx, w)
        E, B = gpu_fields_series(ctx, w, w.steps[0], len(w.steps))
        for k, n in enumerate(w.steps):
            if n in full:
                Eo, Bo = oracle_fields(w, n, None)
                check(w, E[k], B[k], Eo, Bo, None, f"c4 series step {n} (every point)")
            else:
                Eo, Bo = oracle_fields(w, n, idx)
                check(w, E[k][:, idx], B[k][:, idx], Eo, Bo, None, f"c4 series step {n}")
    finally:
        ctx.close()


# ------------------------------------------------------------------ seeded fuzz
def test_series_fuzz_random_geometries_fp64(jb):
    rng = np.random.default_rng(20210406)
    ran = 0
    for case in range(60):
        n_src = tuple(int(v) for v in rng.integers(1, 11, 3))
        n_obs = tuple(int(v) for v in rng.integers(1, 17, 3))
        sp_src = tuple(float(v) for v in rng.uniform(0.05, 0.3, 3))
        sp_obs = tuple(float(v) for v in rng.uniform(0.05, 0.3, 3))
        origin_obs = tuple(float(-(n - 1) / 2 * h + rng.uniform(-0.5, 0.5)) for n, h in zip(n_obs, sp_obs))
        c = float(rng.uniform(0.5, 2.0))
        dt = float(min(sp_src) / (c * rng.uniform(0.5, 12.0)))
        T = int(rng.integers(2, 61))
        w = wl.random_history(n_src, T, seed=5000 + case, dtype="f64", spacing=sp_src, n_obs=n_obs,
                              spacing_obs=sp_obs, origin_obs=origin_obs, dt=dt, c=c)
        count = int(rng.integers(2, min(T, 14) + 1))
        begin = int(rng.integers(0, T - count + 1))
        ob = int(rng.integers(0, w.N_o))
        oc = int(rng.integers(1, w.N_o - ob + 1))
        mode = int(rng.integers(0, 2))
        try:
            series_case(jb, w, begin, count, mode, ob, oc, what=f"fuzz {case}: src {n_src} obs {n_obs} T {T}")
            ran += 1
        except jb.JefiError as e:                          # window beyond shared memory
            assert e.status == jb.JEFI_ERR_UNSUPPORTED
    assert ran >= 48


def test_series_fuzz_random_lattices_fp32(jb):
    rng = np.random.default_rng(5427)
    ran = 0
    while ran < 40:
        n_src = tuple(int(v) for v in rng.integers(1, 11, 3))
        n_obs = tuple(int(v) for v in rng.integers(1, 17, 3))
        if sum((a - b) % 2 for a, b in zip(n_src, n_obs)) == 1:
            continue                                       # exactly one half-cell offset: R can equal rcut
        ratio = int(rng.choice([1, 2, 4]))
        T = int(rng.integers(4, 61))
        w = wl.random_history(n_src, T, seed=7000 + ran, dtype="f32", n_obs=n_obs, dt=0.1 / ratio)
        count = int(rng.integers(4, min(T, 20) + 1))
        begin = int(rng.integers(0, T - count + 1))
        mode = int(rng.integers(0, 2))
        series_case(jb, w, begin, count, mode, what=f"fp32 fuzz {ran}: src {n_src} obs {n_obs} T {T} ratio {ratio}",
                    comp_floor=1e-3)
        ran += 1

"""Parity of the CUDA path (through the C ABI) against the fp64 CPU oracle on the same seeded
inputs.  Bar (BASELINE.json north_star): relative L2 error per field component <= 1e-5 in fp64
mode and <= 2e-4 in fp32 mode; a component that is identically zero in the oracle is measured
against the whole field's norm (Q10).  All tests need a GPU."""
import numpy as np
import pytest

import workloads as wl
from conftest import rel_l2
from gpu_util import gpu_fields, make_ctx, oracle_fields, tol_for, upload

pytestmark = pytest.mark.gpu

KERNELS = [1, 0]        # 1 = per-point kernel, 0 = automatic (tiled where supported)


@pytest.fixture(scope="module")
def jb():
    import __graft_entry__
    __graft_entry__.build()            # no-op when libjefi.so is newer than its sources
    import paper_2104_05426_b200 as jb
    return jb


def check(w, E, B, Eo, Bo, tol=None, what=""):
    tol = tol_for(w) if tol is None else tol
    assert np.isfinite(E).all() and np.isfinite(B).all(), what
    eE, eB = rel_l2(E, Eo, field_ref=Eo), rel_l2(B, Bo, field_ref=Bo)
    assert max(eE) <= tol and max(eB) <= tol, f"{what}: rel-L2 E {eE} B {eB} tol {tol}"
    return eE, eB


def run_case(jb, w, idx, kernel, deriv_mode=0, steps=None, tol=None):
    ctx = make_ctx(w, jb, deriv_mode)
    try:
        ctx.set_kernel(kernel)
        upload(ctx, w)
        for n in (w.steps if steps is None else steps):
            E, B = gpu_fields(ctx, w, n)
            Eo, Bo = oracle_fields(w, n, idx, deriv_mode)
            sel = slice(None) if idx is None else idx
            check(w, E[:, sel], B[:, sel], Eo, Bo, tol, f"{w.name} step {n} kernel {kernel}")
        return E, B
    finally:
        ctx.close()


# ------------------------------------------------------------------ config 1
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("deriv_mode", [0, 1])
def test_config1_tiny_fp64_full(jb, kernel, deriv_mode):
    run_case(jb, wl.config1_tiny(), None, kernel, deriv_mode)


# ------------------------------------------------------------------ config 2
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config2a_coulomb(jb, kernel, dtype):
    w = wl.config2a_coulomb(dtype)
    E, B = run_case(jb, w, w.obs_subset(2048), kernel)
    assert np.all(B == 0.0)                      # J = 0: every B term is an exact zero


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config2b_biot_savart(jb, kernel, dtype):
    w = wl.config2b_wire(dtype)
    E, B = run_case(jb, w, w.obs_subset(2048), kernel)
    assert np.all(E == 0.0)
    assert np.all(B[2] == 0.0)                   # J || z


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_config2c_white_noise_history(jb, kernel, dtype):
    """White in time: one wrong retarded index is an O(1) error in that term."""
    w = wl.config2c_noise(dtype)
    run_case(jb, w, w.obs_subset(2048), kernel)


# ------------------------------------------------------------------ config 3 (the bench workload, full size)
@pytest.mark.parametrize("kernel", KERNELS)
def test_config3_collision_full_size_sampled(jb, kernel):
    w = wl.config3_collision()
    assert w.T == 221 and w.N_s == 64 ** 3
    run_case(jb, w, w.obs_subset(1024), kernel)


# ------------------------------------------------------------------ config 4
def test_config4_detached_plane_time_series(jb):
    w = wl.config4_detached()
    assert w.T == 622 and w.steps[0] == 494 and len(w.steps) == 128
    idx = w.obs_subset(1536)
    ctx = make_ctx(w, jb)
    try:
        upload(ctx, w)
        checked = {w.steps[0], w.steps[-1], w.steps[37]}
        for n in w.steps:
            E, B = gpu_fields(ctx, w, n)
            assert np.isfinite(E).all() and np.isfinite(B).all()
            if n in checked:
                Eo, Bo = oracle_fields(w, n, idx)
                check(w, E[:, idx], B[:, idx], Eo, Bo, None, f"c4 step {n}")
    finally:
        ctx.close()


# ------------------------------------------------------------------ config 5
@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_config5_large_sampled(jb, dtype):
    """100^3 x 100^3 with a history shorter than the longest delay (k_max = 343 > T-1 = 199):
    the m < 0 rule (Q4) is live.  fp32: the whole grid; fp64: a 100x100x12 slab of it."""
    w = wl.config5_large(dtype=dtype)
    ctx = make_ctx(w, jb)
    try:
        upload(ctx, w)
        n = w.steps[0]
        if dtype == "f32":
            begin, count = 0, w.N_o
        else:
            begin, count = 100 * 100 * 44, 100 * 100 * 12
        E, B = gpu_fields(ctx, w, n, begin, count)
        idx = w.obs_subset(400, seed_offset=1)
        idx = idx[(idx >= begin) & (idx < begin + count)]
        if dtype == "f64":
            extra = begin + np.arange(0, count, 997)
            idx = np.unique(np.concatenate([idx, extra]))[:320]
        Eo, Bo = oracle_fields(w, n, idx)
        check(w, E[:, idx - begin], B[:, idx - begin], Eo, Bo, None, f"c5 {dtype}")
    finally:
        ctx.close()


# ------------------------------------------------------------------ ragged shapes, c != 1, sub-ranges, point lists
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_ragged_anisotropic_offset_grids_with_c(jb, kernel, dtype):
    w = wl.random_history((13, 5, 7), 40, seed=77, dtype=dtype, spacing=(0.1, 0.15, 0.07),
                          n_obs=(9, 11, 3), spacing_obs=(0.12, 0.05, 0.2), origin_obs=(-0.31, -0.22, 0.13),
                          dt=0.02, c=1.7)
    for mode in (0, 1):
        run_case(jb, w, None, kernel, mode, steps=(39, 20, 3, 0))


@pytest.mark.parametrize("kernel", KERNELS)
def test_overlapping_grid_hits_the_screening_rule(jb, kernel):
    """obs == source centres (self cell at R = 0) plus points strictly inside / outside rcut."""
    w = wl.random_history((6, 6, 6), 24, seed=5, dtype="f64", spacing=(0.1, 0.1, 0.1), dt=0.05)
    run_case(jb, w, None, kernel)
    w2 = wl.random_history((6, 6, 6), 24, seed=5, dtype="f64", spacing=(0.1, 0.1, 0.1), dt=0.05,
                           origin_obs=(-0.25 + 0.03, -0.25, -0.25 + 0.02))     # R = 0.036 < 0.05
    run_case(jb, w2, None, kernel)
    w3 = wl.random_history((6, 6, 6), 24, seed=5, dtype="f64", spacing=(0.1, 0.1, 0.1), dt=0.05,
                           origin_obs=(-0.25 + 0.04, -0.25 + 0.04, -0.25))     # R = 0.0566 > 0.05
    run_case(jb, w3, None, kernel)


@pytest.mark.parametrize("kernel", KERNELS)
def test_single_stored_step_and_single_cell(jb, kernel):
    w = wl.random_history((1, 1, 1), 1, seed=9, dtype="f64", n_obs=(3, 2, 2), spacing_obs=(0.01, 0.01, 0.01),
                          origin_obs=(0.2, 0.0, 0.0), dt=10.0)
    run_case(jb, w, None, kernel, steps=(0,))


@pytest.mark.parametrize("kernel", KERNELS)
def test_obs_subranges_match_the_full_call(jb, kernel):
    w = wl.random_history((8, 8, 4), 30, seed=11, dtype="f32", n_obs=(10, 7, 5), dt=0.04)
    ctx = make_ctx(w, jb)
    try:
        ctx.set_kernel(kernel)
        upload(ctx, w)
        E, B = gpu_fields(ctx, w, 29)
        for begin, count in ((0, 1), (3, 64), (117, 233), (349, 1), (0, 350)):
            e, b = gpu_fields(ctx, w, 29, begin, count)
            np.testing.assert_allclose(e, E[:, begin:begin + count], rtol=2e-5, atol=1e-6)
            np.testing.assert_allclose(b, B[:, begin:begin + count], rtol=2e-5, atol=1e-6)
        e, b = gpu_fields(ctx, w, 29, 5, 0)          # empty range is a no-op
        assert e.shape == (3, 0)
    finally:
        ctx.close()


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_explicit_point_list_matches_oracle(jb, dtype):
    w = wl.random_history((7, 6, 5), 32, seed=13, dtype=dtype, dt=0.03)
    u = wl.uniform01(4242, 0, 3 * 257).reshape(257, 3)
    pts = (u - 0.5) * np.array([1.5, 1.2, 2.0])
    pts = pts.astype(w.np_dtype).astype(np.float64)     # both sides see the same rounded points
    ctx = make_ctx(w, jb, points=pts)
    try:
        upload(ctx, w)
        E, B = gpu_fields(ctx, w, 31)
        Eo, Bo = oracle_fields(w, 31, points=pts)
        check(w, E, B, Eo, Bo, None, "point list")
    finally:
        ctx.close()


def test_time_series_and_truncated_history(jb):
    """Every step from 0: early steps have most of the light cone before the stored history."""
    w = wl.random_history((6, 5, 4), 16, seed=21, dtype="f64", dt=0.05)
    run_case(jb, w, None, 0, steps=tuple(range(16)))


# ------------------------------------------------------------------ host-buffer entry points, errors
def test_host_buffer_entry_points_match_device_ones(jb):
    import torch
    w = wl.random_history((8, 6, 5), 20, seed=31, dtype="f32", n_obs=(7, 5, 3), dt=0.05)
    ctx = make_ctx(w, jb)
    try:
        rho_h = torch.from_numpy(w.rho).pin_memory()
        J_h = torch.from_numpy(w.J).pin_memory()
        ctx.upload_history_host(rho_h, J_h)
        E_h = torch.empty((3, w.N_o), dtype=torch.float32).pin_memory()
        B_h = torch.empty((3, w.N_o), dtype=torch.float32).pin_memory()
        ctx.fields_host(19, E_h, B_h)
        torch.cuda.synchronize()
        E, B = gpu_fields(ctx, w, 19)
        np.testing.assert_array_equal(E_h.numpy().astype(np.float64), E)
        np.testing.assert_array_equal(B_h.numpy().astype(np.float64), B)
        Eo, Bo = oracle_fields(w, 19)
        check(w, E, B, Eo, Bo)
    finally:
        ctx.close()


def test_error_codes_on_device(jb):
    import torch
    w = wl.random_history((4, 4, 4), 8, seed=1, dtype="f32")
    ctx = make_ctx(w, jb)
    try:
        E = torch.empty((3, w.N_o), dtype=torch.float32, device="cuda")
        B = torch.empty_like(E)
        with pytest.raises(jb.JefiError) as e:
            ctx.fields(7, E, B)
        assert e.value.status == jb.JEFI_ERR_NO_HISTORY
        upload(ctx, w)
        for step in (-1, 8):
            with pytest.raises(jb.JefiError) as e:
                ctx.fields(step, E, B)
            assert e.value.status == jb.JEFI_ERR_TIME_RANGE
        with pytest.raises(jb.JefiError) as e:
            ctx.fields(7, E, B, obs_begin=60, obs_count=5)
        assert e.value.status == jb.JEFI_ERR_INVALID_ARG
        with pytest.raises(jb.JefiError) as e:
            jb.jefi_fields(ctx.ctx, 7, 0, w.N_o, None, B)
        assert e.value.status == jb.JEFI_ERR_INVALID_ARG
        with pytest.raises(jb.JefiError) as e:
            jb.jefi_fields_at_time(ctx.ctx, 3.4 * w.dt, 0, w.N_o, E, B)
        assert e.value.status == jb.JEFI_ERR_TIME_RANGE
        jb.jefi_fields_at_time(ctx.ctx, 7 * w.dt, 0, w.N_o, E, B)
        torch.cuda.synchronize()
        E7, B7 = gpu_fields(ctx, w, 7)
        np.testing.assert_array_equal(E.cpu().numpy().astype(np.float64), E7)
        assert ctx.launches > 0
    finally:
        ctx.close()


# ------------------------------------------------------------------ sliding window (jefi_append_step)
def _window(w, lo, T):
    """The workload restricted to stored steps lo .. lo+T-1 (same arrays, sliced)."""
    import copy
    v = copy.copy(w)
    v.rho = np.ascontiguousarray(w.rho[lo:lo + T])
    v.J = np.ascontiguousarray(w.J[lo:lo + T])
    v.T = T
    return v


@pytest.mark.parametrize("dtype,c", [("f64", 1.0), ("f32", 1.0), ("f64", 1.7)])
@pytest.mark.parametrize("deriv_mode", [0, 1])
def test_append_step_slides_the_window(jb, dtype, c, deriv_mode):
    """T stored steps + A appended ones against (i) the oracle on the whole (T+A)-step raw history
    and (ii) a fresh upload of the last T steps, bit for bit.  The longest lag (k_max = 14 at
    c = 1) is below T-1 = 19, so neither the dropped steps nor the oldest record's derivative
    (centred after a slide, one-sided after a fresh upload) is ever read."""
    import torch
    T, A = 20, 5
    full = wl.random_history((6, 5, 4), T + A, seed=41, dtype=dtype, n_obs=(5, 4, 6), dt=0.05, c=c)
    first = _window(full, 0, T)
    ctx = make_ctx(first, jb, deriv_mode)
    try:
        upload(ctx, first)
        for a in range(A):
            rho_new = torch.from_numpy(full.rho[T + a]).cuda()
            J_new = torch.from_numpy(full.J[T + a]).cuda()
            if a % 2 == 0:
                ctx.append_step(rho_new, J_new)
            else:
                ctx.append_step_host(torch.from_numpy(full.rho[T + a]).pin_memory(),
                                     torch.from_numpy(full.J[T + a]).pin_memory())
            torch.cuda.synchronize()
            E, B = gpu_fields(ctx, first, T - 1)
            Eo, Bo = oracle_fields(full, T + a, None, deriv_mode)
            check(full, E, B, Eo, Bo, None, f"after {a + 1} appends")
        fresh_w = _window(full, A, T)
        fresh = make_ctx(fresh_w, jb, deriv_mode)
        try:
            upload(fresh, fresh_w)
            for kernel in KERNELS:
                ctx.set_kernel(kernel); fresh.set_kernel(kernel)
                E2, B2 = gpu_fields(fresh, fresh_w, T - 1)
                E1, B1 = gpu_fields(ctx, first, T - 1)
                np.testing.assert_array_equal(E1, E2)
                np.testing.assert_array_equal(B1, B2)
            # jefi_fields_at_time follows the advanced t0
            Ed = torch.empty((3, full.N_o), dtype=torch.float64 if dtype == "f64" else torch.float32, device="cuda")
            Bd = torch.empty_like(Ed)
            jb.jefi_fields_at_time(ctx.ctx, (T - 1 + A) * full.dt, 0, full.N_o, Ed, Bd)
            torch.cuda.synchronize()
            np.testing.assert_array_equal(Ed.cpu().numpy().astype(np.float64), E1)
        finally:
            fresh.close()
    finally:
        ctx.close()


def test_append_step_single_stored_step_and_errors(jb):
    import torch
    w = wl.random_history((3, 3, 2), 3, seed=43, dtype="f64", n_obs=(2, 2, 2), spacing_obs=(0.01, 0.01, 0.01),
                          origin_obs=(0.4, 0.0, 0.0), dt=10.0)
    one = _window(w, 0, 1)
    ctx = make_ctx(one, jb)
    try:
        with pytest.raises(jb.JefiError) as e:
            ctx.append_step(torch.from_numpy(w.rho[1]).cuda(), torch.from_numpy(w.J[1]).cuda())
        assert e.value.status == jb.JEFI_ERR_NO_HISTORY
        upload(ctx, one)
        with pytest.raises(jb.JefiError) as e:
            jb.jefi_append_step(ctx.ctx, None, torch.from_numpy(w.J[1]).cuda())
        assert e.value.status == jb.JEFI_ERR_INVALID_ARG
        # T = 1: every lag is 0 (dt = 10), the stored step is replaced and gets (f_new - f_prev)/dt
        for a in (1, 2):
            ctx.append_step(torch.from_numpy(w.rho[a]).cuda(), torch.from_numpy(w.J[a]).cuda())
            E, B = gpu_fields(ctx, one, 0)
            Eo, Bo = oracle_fields(_window(w, 0, a + 1), a, None, 1)     # backward difference == one-sided
            check(w, E, B, Eo, Bo, None, f"T=1 after {a} appends")
    finally:
        ctx.close()


# ------------------------------------------------------------------ long retarded-time windows
@pytest.mark.parametrize("dtype,kernel", [("f32", 2), ("f64", 2)])
def test_long_windows_use_the_widest_tile_variant(jb, dtype, kernel):
    """dx/(c dt) = 20: a tile's lag window is ~250 steps -> the kernel variant whose window
    capacity comes from the launch, one CTA per SM; kernel 2 = tiled or JEFI_ERR_UNSUPPORTED.  The history (T = 300) is shorter than
    the longest lag (~500).  Geometry: offsets are half-integer multiples of dx on two axes, so
    no pair sits on the screening radius and q = 10 sqrt(N) stays >= 5e-4 away from a tie."""
    w = wl.random_history((5, 4, 3), 300, seed=51, dtype=dtype, n_obs=(10, 8, 8), dt=0.005)
    ctx = make_ctx(w, jb)
    try:
        ctx.set_kernel(kernel)
        upload(ctx, w)
        for n in (299, 120, 7):
            E, B = gpu_fields(ctx, w, n)
            Eo, Bo = oracle_fields(w, n)
            check(w, E, B, Eo, Bo, None, f"long window step {n}")
    finally:
        ctx.close()


def test_windows_beyond_shared_memory_fall_back_to_the_point_kernel(jb):
    """dx/(c dt) = 500: ~6000-step windows (384 KB per cell in fp64) do not fit in shared memory;
    automatic selection uses the per-point kernel, forcing the tiled kernel is refused."""
    import torch
    w = wl.random_history((4, 4, 3), 64, seed=53, dtype="f64", n_obs=(9, 8, 8), dt=0.0002)
    ctx = make_ctx(w, jb)
    try:
        upload(ctx, w)
        E, B = gpu_fields(ctx, w, 63)
        Eo, Bo = oracle_fields(w, 63)
        check(w, E, B, Eo, Bo, None, "fallback")
        ctx.set_kernel(2)
        Ed = torch.empty((3, w.N_o), dtype=torch.float64, device="cuda")
        with pytest.raises(jb.JefiError) as e:
            ctx.fields(63, Ed, torch.empty_like(Ed))
        assert e.value.status == jb.JEFI_ERR_UNSUPPORTED
    finally:
        ctx.close()


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("n_obs", [(12, 9, 10), (4, 20, 3), (20, 12, 1), (33, 16, 2)])
def test_ragged_tiles_every_edge_shape(jb, dtype, n_obs):
    """Observation grids that end inside a tile in x (half-x variant), y (warps along y), z (idle
    warps), all three, and plane-shaped sets; full oracle comparison.  Same spacing as the
    source grid: offsets are integer on all axes or half-integer on two, so no pair sits on the
    screening radius (R = dx/2 needs exactly one half-integer axis) and q = 2 sqrt(M) or sqrt(N)
    stays >= 1.5e-3 away from a rounding tie (white-noise history: a flipped index would show)."""
    w = wl.random_history((6, 5, 4), 48, seed=57, dtype=dtype, n_obs=n_obs, dt=0.05)
    run_case(jb, w, None, 2, steps=(47, 11))


# ------------------------------------------------------------------ every output at full size
@pytest.mark.parametrize("make,step", [(lambda: wl.config3_collision(), 220), (lambda: wl.config4_detached(), 621)],
                         ids=["c3", "c4"])
def test_full_size_every_point_tiled_vs_point_kernel(jb, make, step):
    """The oracle can only afford a sample of the full-size configs; here EVERY output of the
    tiled kernel (the launch configuration bench.py times) is compared with the per-point
    kernel, which shares the packed history but none of the tiling, window staging, lag
    arithmetic (magic-constant rounding vs floor) or summation order.  Both are within 2e-4 of
    the oracle on the sample (rel-L2), so they must agree to 4e-4 in rel-L2 and, point by point,
    to a few 1e-3 of the field's rms (no single output may be off)."""
    w = make()
    ctx = make_ctx(w, jb)
    try:
        upload(ctx, w)
        ctx.set_kernel(2)
        E2, B2 = gpu_fields(ctx, w, step)
        ctx.set_kernel(1)
        E1, B1 = gpu_fields(ctx, w, step)
        for got, ref, name in ((E2, E1, "E"), (B2, B1, "B")):
            rms = np.sqrt(np.mean(ref * ref))
            worst = np.abs(got - ref).max()
            assert worst <= 4e-3 * rms, f"{name}: worst pointwise difference {worst:.3e} vs rms {rms:.3e}"
            assert max(rel_l2(got, ref, field_ref=ref)) <= 4e-4
    finally:
        ctx.close()


# ------------------------------------------------------------------ the paper's own test case (Sec. 3.1)
def test_paper_constant_sources_410_snapshots(jb):
    """PAPER.md:122-139, :213-219 (Table 2): rho = 1, J = (1,1,1) switched on at t = 0 on the 15^3
    grid over [-3,3]^3, 410 snapshots at dt = 0.05, fp32 storage.  All 411 steps through the C
    ABI; seven of them against the oracle on every point; the legend magnitude of Fig. 4/5 at
    t = 2.5 (~0.5); and the paper's saturation (after the longest
    light-travel time the fields no longer change) bit for bit on the CUDA output."""
    import time
    import torch
    T = 411
    w = wl.paper_x1_constant(T, n=15, dtype="f32")
    ctx = make_ctx(w, jb)
    try:
        upload(ctx, w)
        E = torch.empty((T, 3, w.N_o), dtype=torch.float32, device="cuda")
        B = torch.empty_like(E)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ctx.fields_series(0, T, E, B)                      # one C call, 411 evaluations
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        E1 = torch.empty((3, w.N_o), dtype=torch.float32, device="cuda")
        B1 = torch.empty_like(E1)
        for n in (0, 77, 410):                             # the series equals the single calls
            ctx.fields(n, E1, B1)
            torch.cuda.synchronize()
            assert torch.equal(E1, E[n]) and torch.equal(B1, B[n])
        with pytest.raises(jb.JefiError) as e:
            ctx.fields_series(400, 20, E, B)
        assert e.value.status == jb.JEFI_ERR_TIME_RANGE
        E, B = E.cpu().numpy().astype(np.float64), B.cpu().numpy().astype(np.float64)
        for n in (0, 1, 50, 100, 150, 250, 410):
            Eo, Bo = oracle_fields(w, n)
            check(w, E[n], B[n], Eo, Bo, None, f"paper X1 step {n}")
        plane = np.arange(15 * 15) + 7 * 15 * 15                     # the z = 0 layer
        e_max = np.sqrt(E[50][0][plane] ** 2 + E[50][1][plane] ** 2).max()
        b_max = np.sqrt(B[50][0][plane] ** 2 + B[50][1][plane] ** 2).max()
        assert abs(e_max - 0.529) < 2e-3 and abs(b_max - 0.529) < 2e-3
        k_max = int(np.floor(np.sqrt(3.0) * 14 * 0.4 / 0.05 + 0.5))  # longest lag on the grid: 194
        for n in range(k_max + 2, T):
            assert np.array_equal(E[n], E[T - 1]) and np.array_equal(B[n], B[T - 1]), n
        assert not np.array_equal(E[k_max - 20], E[T - 1])
        print(f"\npaper Table 2 workload: 411 snapshots of [15^3,15^3] in {wall * 1e3:.1f} ms wall "
              f"({wall / T * 1e6:.0f} us per snapshot; the paper: 8.696 s on a Tesla V100, PAPER.md:217)")
    finally:
        ctx.close()


# ------------------------------------------------------------------ seeded fuzz of the launch logic
def test_fuzz_random_geometries_fp64(jb):
    """150 seeded random set-ups (grid shapes, anisotropic spacings, offsets, c, dt from
    dx/(c dt) = 0.5 to 12, history lengths from 1 step to beyond the longest lag, evaluation step,
    observation sub-range, derivative mode) through the tiled kernel in fp64, each against the
    oracle on every requested point.  Exercises tile raggedness, window capacities (32 / 96 /
    sized by the launch), zero-filled pre-history slots, chunking and sub-range clipping in
    combinations the named cases do not.  fp64 and real-valued geometry: a rounding tie or a pair
    on the screening radius has measure zero."""
    import torch
    rng = np.random.default_rng(20210405)
    ran = 0
    for case in range(150):
        n_src = tuple(int(v) for v in rng.integers(1, 13, 3))
        n_obs = tuple(int(v) for v in rng.integers(1, 21, 3))
        sp_src = tuple(float(v) for v in rng.uniform(0.05, 0.3, 3))
        sp_obs = tuple(float(v) for v in rng.uniform(0.05, 0.3, 3))
        origin_obs = tuple(float(-(n - 1) / 2 * h + rng.uniform(-0.5, 0.5)) for n, h in zip(n_obs, sp_obs))
        c = float(rng.uniform(0.5, 2.0))
        dt = float(min(sp_src) / (c * rng.uniform(0.5, 12.0)))
        T = int(rng.integers(1, 81))
        w = wl.random_history(n_src, T, seed=1000 + case, dtype="f64", spacing=sp_src, n_obs=n_obs,
                              spacing_obs=sp_obs, origin_obs=origin_obs, dt=dt, c=c)
        step = int(rng.integers(0, T))
        begin = int(rng.integers(0, w.N_o))
        count = int(rng.integers(1, w.N_o - begin + 1))
        mode = int(rng.integers(0, 2))
        ctx = make_ctx(w, jb, mode)
        try:
            ctx.set_kernel(2)
            upload(ctx, w)
            try:
                E, B = gpu_fields(ctx, w, step, begin, count)
            except jb.JefiError as e:                      # window beyond shared memory
                assert e.status == jb.JEFI_ERR_UNSUPPORTED
                continue
            idx = np.arange(begin, begin + count)
            Eo, Bo = oracle_fields(w, step, idx, mode)
            check(w, E, B, Eo, Bo, None, f"fuzz case {case}: src {n_src} obs {n_obs} T {T} step {step} "
                                          f"range {begin}+{count} mode {mode} dx/cdt {min(sp_src) / (c * dt):.2f}")
            ran += 1
        finally:
            ctx.close()
    assert ran >= 120


def test_fuzz_random_lattices_fp32(jb):
    """The same for fp32 on white-noise histories, where one flipped retarded index is an O(1)
    error in its term: 80 seeded random shapes on commensurate lattices (equal spacing,
    dx/(c dt) in {1, 2, 4}, centred grids whose offsets are integer on all axes or half-integer
    on at least two, so that no lag is a rounding tie -- 4M = odd square is impossible mod 4 / mod
    8 -- and no pair sits on the screening radius)."""
    rng = np.random.default_rng(5426)
    ran = 0
    while ran < 80:
        n_src = tuple(int(v) for v in rng.integers(1, 13, 3))
        n_obs = tuple(int(v) for v in rng.integers(1, 21, 3))
        if sum((a - b) % 2 for a, b in zip(n_src, n_obs)) == 1:
            continue                                       # exactly one half-cell offset: R can equal rcut
        ratio = int(rng.choice([1, 2, 4]))
        T = int(rng.integers(1, 81))
        w = wl.random_history(n_src, T, seed=3000 + ran, dtype="f32", n_obs=n_obs, dt=0.1 / ratio)
        step = int(rng.integers(0, T))
        begin = int(rng.integers(0, w.N_o))
        count = int(rng.integers(1, w.N_o - begin + 1))
        mode = int(rng.integers(0, 2))
        ctx = make_ctx(w, jb, mode)
        try:
            ctx.set_kernel(2)
            upload(ctx, w)
            E, B = gpu_fields(ctx, w, step, begin, count)
            idx = np.arange(begin, begin + count)
            Eo, Bo = oracle_fields(w, step, idx, mode)
            check(w, E, B, Eo, Bo, None, f"fp32 fuzz {ran}: src {n_src} obs {n_obs} T {T} step {step} "
                                          f"range {begin}+{count} mode {mode} dx/cdt {ratio}")
            ran += 1
        finally:
            ctx.close()

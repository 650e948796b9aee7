"""jefi_fields_noalloc (include/jefi.h): the entry point for hosts that cannot allocate device
memory -- an application whose memory pool already owns every free byte of HBM, so cudaMalloc
fails, or a stepping loop that cannot afford the device-wide stall of cudaMalloc/cudaFree.  It
takes the caller's raw history and output planes, needs no jefi_ctx, and keeps its partial sums
in one fixed array inside libjefi.so, shared by every call on a device.

What is checked: its E and B agree with the existing path (jefi_create + jefi_upload_history +
jefi_fields) within the parity tolerance of the other GPU tests (rel-L2 per component 2e-4 in
fp32, 1e-5 in fp64, plus the pointwise bound), on TWO calls in a row of different shape, so
that the second call runs over whatever the first one left in the shared array; one case is
also held against the fp64 oracle.  Requests beyond the stated maximum are refused with a
message, before any CUDA call (that part needs no GPU).

This file is named to be collected last: under `pytest -x` a failure here hides nothing.
"""
import numpy as np
import pytest

import workloads as wl
from conftest import rel_l2
from gpu_util import gpu_fields, make_ctx, oracle_fields, tol_for, torch_dtype, upload

POINTWISE = 20.0        # as in test_parity_gpu.py: max |a - b| <= POINTWISE * tol * rms(reference field)


@pytest.fixture(scope="module")
def jb():
    import __graft_entry__
    __graft_entry__.build()
    import paper_2104_05426_b200 as jb
    return jb


def descriptors(jb, w, deriv_mode=0, points_dev=None):
    src = jb.make_grid(w.n_src, w.origin_src, w.spacing_src)
    if points_dev is None:
        obs = jb.make_obs_grid(w.n_obs, w.origin_obs, w.spacing_obs)
    else:
        obs = jb.jefi_obs_desc()
        obs.kind = 1
        obs.grid = jb.make_grid((1, 1, 1), (0, 0, 0), (1, 1, 1))
        obs.npoints = int(points_dev.shape[0])
        obs.points_dev = points_dev.data_ptr()
    tm = jb.jefi_time_desc(float(w.t0), float(w.dt), float(w.c), int(w.T), int(deriv_mode), 0)
    return src, obs, tm


def agree(w, got, ref, what):
    tol = tol_for(w)
    for (a, b, name) in ((got[0], ref[0], "E"), (got[1], ref[1], "B")):
        assert np.isfinite(a).all(), f"{what}: non-finite {name}"
        err = rel_l2(a, b, field_ref=b)
        assert max(err) <= tol, f"{what}: rel-L2 {name} {err} > {tol}"
        rms = float(np.sqrt(np.mean(np.sum(b * b, axis=0))))
        worst = float(np.abs(a - b).max())
        assert worst <= POINTWISE * tol * rms, f"{what}: worst pointwise {name} error {worst:.3e}, rms {rms:.3e}"


def noalloc_fields(jb, w, desc, rho, J, step, obs_begin, obs_count):
    import torch
    E = torch.full((3, obs_count), float("nan"), dtype=torch_dtype(w), device="cuda")
    B = torch.full((3, obs_count), float("nan"), dtype=torch_dtype(w), device="cuda")
    jb.jefi_fields_noalloc(*desc, jb.JEFI_F32 if w.dtype == "f32" else jb.JEFI_F64, step, rho, J, obs_begin,
                           obs_count, E, B)
    torch.cuda.synchronize()
    return E.cpu().numpy().astype(np.float64), B.cpu().numpy().astype(np.float64)


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("deriv_mode", [0, 1])
def test_two_calls_in_a_row_match_the_context_path(jb, dtype, deriv_mode):
    import torch
    w = wl.config2c_noise(dtype, n=16, T=40)          # white-noise history: every lag and derivative matters
    n_obs = w.N_o
    ctx = make_ctx(w, jb, deriv_mode)
    try:
        upload(ctx, w)
        rho, J = torch.from_numpy(w.rho).cuda(), torch.from_numpy(w.J).cuda()
        desc = descriptors(jb, w, deriv_mode)

        # call 1: the whole observation grid at the newest step (several source chunks in the scratch array)
        step1 = w.T - 1
        got1 = noalloc_fields(jb, w, desc, rho, J, step1, 0, n_obs)
        # call 2, straight after: a ragged sub-range at an early step (part of the sources not yet
        # "switched on": m < 0), running over what call 1 left in the shared array
        step2, begin2, count2 = 9, 517, 1203
        got2 = noalloc_fields(jb, w, desc, rho, J, step2, begin2, count2)

        ref1 = gpu_fields(ctx, w, step1)
        ref2 = gpu_fields(ctx, w, step2, begin2, count2)
        agree(w, got1, ref1, f"call 1 {dtype} deriv {deriv_mode}")
        agree(w, got2, ref2, f"call 2 {dtype} deriv {deriv_mode}")
        if deriv_mode == 0:
            agree(w, got1, oracle_fields(w, step1, None, deriv_mode), f"call 1 {dtype} against the oracle")
    finally:
        ctx.close()


@pytest.mark.gpu
def test_point_list_and_one_step_history(jb):
    import torch
    # explicit points (smooth history: fp32 near-ties on unstructured points, Q3), then
    # straight after it a one-step history (derivative 0 in centred mode) on a grid
    w = wl.smooth_in_time(wl.with_random_points(wl.config2c_noise("f32", n=12, T=24), 777), period=16.0)
    ctx = make_ctx(w, jb)
    try:
        upload(ctx, w)
        pts = torch.as_tensor(np.ascontiguousarray(w.points, dtype=w.np_dtype)).cuda()
        rho, J = torch.from_numpy(w.rho).cuda(), torch.from_numpy(w.J).cuda()
        got = noalloc_fields(jb, w, descriptors(jb, w, 0, pts), rho, J, w.T - 1, 0, 777)
        agree(w, got, gpu_fields(ctx, w, w.T - 1), "point list")
    finally:
        ctx.close()
    w1 = wl.config2c_noise("f64", n=8, T=1)
    ctx = make_ctx(w1, jb)
    try:
        upload(ctx, w1)
        rho, J = torch.from_numpy(w1.rho).cuda(), torch.from_numpy(w1.J).cuda()
        got = noalloc_fields(jb, w1, descriptors(jb, w1), rho, J, 0, 0, w1.N_o)
        agree(w1, got, gpu_fields(ctx, w1, 0), "T = 1")
    finally:
        ctx.close()


def test_the_object_file_references_no_allocator(jb):
    """The promise 'no cudaMalloc, cudaFree or allocating routine', checked on the compiled object:
    fields_noalloc.o may not even reference one (no GPU needed)."""
    import shutil
    import subprocess
    from pathlib import Path
    nm = shutil.which("nm")
    obj = Path(jb.LIB_PATH).parent / "build" / "fields_noalloc.o"
    if nm is None or not obj.exists():
        pytest.skip("needs binutils' nm and the in-tree object file")
    undefined = subprocess.run([nm, "-u", str(obj)], check=True, capture_output=True, text=True).stdout
    assert "cudaGetSymbolAddress" in undefined and "cudaLaunchKernel" in undefined
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMemPool", "cudaHostRegister", "cuMemAlloc",
                   "malloc", "_Znw", "_Zna"):
        assert banned not in undefined, f"fields_noalloc.o references {banned}"


def test_requests_beyond_the_fixed_scratch_are_refused_with_a_message(jb):
    """No GPU needed: the size and argument checks come before the first CUDA call."""
    assert 6 * jb.JEFI_NOALLOC_MAX_OBS * 8 <= jb.JEFI_NOALLOC_SCRATCH_BYTES
    src = jb.make_grid((4, 4, 4), (0, 0, 0), (0.1, 0.1, 0.1))
    obs = jb.make_obs_grid((64, 64, 64), (0, 0, 0), (0.1, 0.1, 0.1))
    tm = jb.jefi_time_desc(0.0, 0.05, 1.0, 8, 0, 0)
    fake = 256                                        # never dereferenced: the call fails before any launch
    with pytest.raises(jb.JefiError) as e:
        jb.jefi_fields_noalloc(src, obs, tm, jb.JEFI_F32, 7, fake, fake, 0, jb.JEFI_NOALLOC_MAX_OBS + 1, fake, fake)
    assert e.value.status == jb.JEFI_ERR_UNSUPPORTED
    assert "JEFI_NOALLOC_MAX_OBS" in str(e.value) and str(jb.JEFI_NOALLOC_MAX_OBS) in str(e.value)
    for args, status in (
        ((src, obs, tm, jb.JEFI_F32, 8, fake, fake, 0, 10, fake, fake), jb.JEFI_ERR_TIME_RANGE),
        ((src, obs, tm, jb.JEFI_F32, 0, fake, fake, 64 ** 3 - 5, 10, fake, fake), jb.JEFI_ERR_INVALID_ARG),
        ((src, obs, tm, jb.JEFI_F32, 0, None, fake, 0, 10, fake, fake), jb.JEFI_ERR_INVALID_ARG),
        ((src, obs, tm, 7, 0, fake, fake, 0, 10, fake, fake), jb.JEFI_ERR_INVALID_ARG),
        ((None, obs, tm, jb.JEFI_F32, 0, fake, fake, 0, 10, fake, fake), jb.JEFI_ERR_INVALID_ARG),
    ):
        with pytest.raises(jb.JefiError) as e:
            jb.jefi_fields_noalloc(*args)
        assert e.value.status == status and str(e.value)
    # an empty request is a no-op that needs no pointers and no device
    jb.jefi_fields_noalloc(src, obs, tm, jb.JEFI_F32, 0, None, None, 0, 0, None, None)

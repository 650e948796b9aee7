"""Helpers for the -m gpu parity tests: run a workloads.Workload through the C ABI (via the
thin binding) and through the oracle on the same seeded arrays."""
import numpy as np


def torch_dtype(w):
    import torch
    return torch.float32 if w.dtype == "f32" else torch.float64


def make_ctx(w, jb, deriv_mode=0, points=None):
    import torch
    if points is None and getattr(w, "points", None) is not None:
        points = w.points
    if points is None:
        return jb.Jefi(w.n_src, w.origin_src, w.spacing_src, dt=w.dt, c=w.c, nsteps=w.T, dtype=w.dtype,
                       n_obs=w.n_obs, origin_obs=w.origin_obs, spacing_obs=w.spacing_obs, t0=w.t0,
                       deriv_mode=deriv_mode)
    pts = torch.as_tensor(np.ascontiguousarray(points, dtype=w.np_dtype)).cuda()
    return jb.Jefi(w.n_src, w.origin_src, w.spacing_src, dt=w.dt, c=w.c, nsteps=w.T, dtype=w.dtype,
                   points_dev=pts, t0=w.t0, deriv_mode=deriv_mode)


def upload(ctx, w):
    import torch
    rho = torch.from_numpy(w.rho).cuda()
    J = torch.from_numpy(w.J).cuda()
    ctx.upload_history(rho, J)
    torch.cuda.synchronize()
    del rho, J


def gpu_fields(ctx, w, step, obs_begin=0, obs_count=None):
    """E, B as float64 numpy [3][count] computed by the CUDA path."""
    import torch
    n = ctx.n_points - obs_begin if obs_count is None else obs_count
    E = torch.full((3, n), float("nan"), dtype=torch_dtype(w), device="cuda")
    B = torch.full((3, n), float("nan"), dtype=torch_dtype(w), device="cuda")
    ctx.fields(step, E, B, obs_begin, n)
    torch.cuda.synchronize()
    return E.cpu().numpy().astype(np.float64), B.cpu().numpy().astype(np.float64)


_ORACLE_CACHE = {}


def oracle_fields(w, step, idx=None, deriv_mode=0, points=None):
    """Oracle E, B at the selected observation points (cached per workload within a session:
    several kernels are checked against the same oracle run)."""
    import hashlib
    import oracle
    pts = w.obs_points(idx) if points is None else np.asarray(points, dtype=np.float64)
    key = (w.name, w.dtype, w.n_src, w.spacing_src, w.T, w.seed, w.c, w.dt, step, deriv_mode,
           hashlib.sha1(np.ascontiguousarray(pts).tobytes()).hexdigest())
    if key not in _ORACLE_CACHE:
        if len(_ORACLE_CACHE) > 4000:
            _ORACLE_CACHE.clear()
        _ORACLE_CACHE[key] = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, dt=w.dt, c=w.c,
                                           step=step, obs_xyz=pts, deriv_mode=deriv_mode)
    return _ORACLE_CACHE[key]


def tol_for(w):
    """BASELINE.json north_star: rel-L2 per field component <= 1e-5 (fp64 mode), 2e-4 (fp32)."""
    return 2e-4 if w.dtype == "f32" else 1e-5


def gpu_fields_series(ctx, w, step_begin, step_count, obs_begin=0, obs_count=None):
    """E, B as float64 numpy [step_count][3][count] from one jefi_fields_series call."""
    import torch
    n = ctx.n_points - obs_begin if obs_count is None else obs_count
    E = torch.full((step_count, 3, n), float("nan"), dtype=torch_dtype(w), device="cuda")
    B = torch.full((step_count, 3, n), float("nan"), dtype=torch_dtype(w), device="cuda")
    ctx.fields_series(step_begin, step_count, E, B, obs_begin, n)
    torch.cuda.synchronize()
    return E.cpu().numpy().astype(np.float64), B.cpu().numpy().astype(np.float64)

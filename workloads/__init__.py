"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs).

This module serves BOTH the oracle tests and the CUDA path's tests/bench, and therefore holds
none of the method's arithmetic: no retarded time, no field formula, no derivative, no packing.
It only describes grids and fills rho / J histories.  The paper uses no public dataset; these
are stand-ins for its analytic test sources and its heavy-ion use
case, with the recipe stated in DESIGN.md.

Conventions: grids are centred on the origin, cell centres at (i - (n-1)/2)*dx (PAPER.md:137:
15 cells x 0.4 = [-3,3]); x is the fastest index; arrays are rho[T, nz, ny, nx] and
J[T, 3, nz, ny, nx]; c = 1.  Values are generated in fp64, magnitudes below 1e-30 are set to 0
(so fp32 denormals never enter either side) and then cast to the run dtype.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 210405426
_TINY = 1e-30


# ----------------------------------------------------------------------------- RNG
def splitmix64(x: np.ndarray) -> np.ndarray:
    """Counter-based generator: one splitmix64 output per 64-bit counter value."""
    with np.errstate(over="ignore"):
        z = (x + np.uint64(0x9E3779B97F4A7C15)).astype(np.uint64)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def uniform01(seed: int, start: int, count: int) -> np.ndarray:
    """u in [0,1): element i is a pure function of (seed, start+i)."""
    with np.errstate(over="ignore"):
        key = splitmix64(np.array([seed], dtype=np.uint64))[0]
        ctr = np.arange(start, start + count, dtype=np.uint64) + key * np.uint64(0x2545F4914F6CDD1D)
    return (splitmix64(ctr) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


# ----------------------------------------------------------------------------- description
@dataclass
class Workload:
    name: str
    n_src: tuple            # (nx, ny, nz)
    spacing_src: tuple      # (dx, dy, dz)
    n_obs: tuple            # (nxo, nyo, nzo) regular observation grid
    spacing_obs: tuple
    origin_obs: tuple       # centre of obs point (0,0,0)
    dt: float
    T: int                  # stored steps m = 0..T-1 at t0 + m*dt
    steps: tuple            # evaluation steps n
    dtype: str              # "f32" | "f64"
    rho: np.ndarray = field(repr=False, default=None)
    J: np.ndarray = field(repr=False, default=None)
    c: float = 1.0
    t0: float = 0.0
    seed: int = BASE_SEED
    points: np.ndarray = field(repr=False, default=None)   # explicit observation points [n,3] instead of a grid

    @property
    def origin_src(self):
        return tuple(-(n - 1) / 2.0 * h for n, h in zip(self.n_src, self.spacing_src))

    @property
    def N_s(self) -> int:
        return int(np.prod(self.n_src))

    @property
    def N_o(self) -> int:
        return int(self.points.shape[0]) if self.points is not None else int(np.prod(self.n_obs))

    @property
    def pairs_per_step(self) -> int:
        return self.N_s * self.N_o

    def obs_points(self, idx=None) -> np.ndarray:
        """float64 [n,3] positions of linear obs indices (x fastest); all points if idx is None."""
        nx, ny, nz = self.n_obs
        idx = np.arange(self.N_o, dtype=np.int64) if idx is None else np.asarray(idx, dtype=np.int64)
        if self.points is not None:
            return np.ascontiguousarray(self.points[idx], dtype=np.float64)
        ix, iy, iz = idx % nx, (idx // nx) % ny, idx // (nx * ny)
        p = np.empty((idx.size, 3), dtype=np.float64)
        for a, i in enumerate((ix, iy, iz)):
            p[:, a] = self.origin_obs[a] + i * self.spacing_obs[a]
        return p

    def obs_subset(self, count: int, seed_offset: int = 0) -> np.ndarray:
        """Seeded subset of linear obs indices: 8 corners, centre, 6 face centres, rest random."""
        if self.points is not None:
            if count >= self.N_o:
                return np.arange(self.N_o, dtype=np.int64)
            u = uniform01(self.seed + 7919 + seed_offset, 0, count)
            return np.unique(np.minimum((u * self.N_o).astype(np.int64), self.N_o - 1))
        nx, ny, nz = self.n_obs
        lin = lambda i, j, k: (k * ny + j) * nx + i
        fixed = [lin(i, j, k) for i in (0, nx - 1) for j in (0, ny - 1) for k in (0, nz - 1)]
        cx, cy, cz = nx // 2, ny // 2, nz // 2
        fixed += [lin(cx, cy, cz), lin(0, cy, cz), lin(nx - 1, cy, cz), lin(cx, 0, cz),
                  lin(cx, ny - 1, cz), lin(cx, cy, 0), lin(cx, cy, nz - 1)]
        fixed = list(dict.fromkeys(fixed))
        if count >= self.N_o:
            return np.arange(self.N_o, dtype=np.int64)
        n_rand = max(count - len(fixed), 0)
        u = uniform01(self.seed + 7919 + seed_offset, 0, n_rand)
        rnd = np.minimum((u * self.N_o).astype(np.int64), self.N_o - 1)
        out = np.unique(np.concatenate([np.array(fixed[:count], dtype=np.int64), rnd]))
        return out

    @property
    def np_dtype(self):
        return np.float32 if self.dtype == "f32" else np.float64


def _centres(n: int, h: float) -> np.ndarray:
    return (np.arange(n, dtype=np.float64) - (n - 1) / 2.0) * h


def _finish(w: Workload, rho64: np.ndarray, J64: np.ndarray) -> Workload:
    for a in (rho64, J64):
        a[np.abs(a) < _TINY] = 0.0
    w.rho = np.ascontiguousarray(rho64.astype(w.np_dtype))
    w.J = np.ascontiguousarray(J64.astype(w.np_dtype))
    return w


# ----------------------------------------------------------------------------- config 1
def config1_tiny() -> Workload:
    """8^3 drifting Gaussian blob, obs = the same 512 cell centres, fp64 (BASELINE.json configs[0])."""
    n, dx, dt, T = 8, 0.1, 0.05, 32
    w = Workload("c1_tiny", (n,) * 3, (dx,) * 3, (n,) * 3, (dx,) * 3, (-(n - 1) / 2 * dx,) * 3,
                 dt, T, (T - 1,), "f64", seed=BASE_SEED + 1)
    x = _centres(n, dx)
    sig, v, t_mid = 0.2, 0.3, 15.5 * dt
    rho = np.empty((T, n, n, n))
    gx = np.exp(-x * x / (2 * sig * sig))
    for m in range(T):
        zc = v * (m * dt - t_mid)
        gz = np.exp(-(x - zc) ** 2 / (2 * sig * sig))
        rho[m] = gz[:, None, None] * gx[None, :, None] * gx[None, None, :]
    J = np.zeros((T, 3, n, n, n))
    J[:, 2] = rho * v
    return _finish(w, rho, J)


# ----------------------------------------------------------------------------- config 2
def _config2_base(name: str, dtype: str, n: int = 32, T: int = 64) -> Workload:
    dx, dt = 0.05, 0.05
    o = -(n - 1) / 2 * dx + 0.5 * dx          # obs offset by half a cell on all three axes
    return Workload(name, (n,) * 3, (dx,) * 3, (n,) * 3, (dx,) * 3, (o,) * 3, dt, T, (T - 1,),
                    dtype, seed=BASE_SEED + 2)


def config2a_coulomb(dtype: str = "f64", n: int = 32, T: int = 64) -> Workload:
    """One cell with rho = 1, constant in time, J = 0 (BASELINE.json configs[1] (a))."""
    w = _config2_base("c2a_coulomb", dtype, n, T)
    rho = np.zeros((T, n, n, n))
    rho[:, n // 2, n // 2, n // 2] = 1.0
    return _finish(w, rho, np.zeros((T, 3, n, n, n)))


def config2b_wire(dtype: str = "f64", n: int = 32, T: int = 64) -> Workload:
    """A line of n cells along z with constant J_z = 1, rho = 0 (configs[1] (b))."""
    w = _config2_base("c2b_wire", dtype, n, T)
    J = np.zeros((T, 3, n, n, n))
    J[:, 2, :, n // 2, n // 2] = 1.0
    return _finish(w, np.zeros((T, n, n, n)), J)


def config2c_noise(dtype: str = "f64", n: int = 32, T: int = 64) -> Workload:
    """Every rho[m][j], J_c[m][j] i.i.d. uniform in [-1,1]: white in time, the harshest case for
    retarded-index parity (configs[1], seeded random part)."""
    w = _config2_base("c2c_noise", dtype, n, T)
    Ns = n ** 3
    rho = (2.0 * uniform01(w.seed, 0, T * Ns) - 1.0).reshape(T, n, n, n)
    J = (2.0 * uniform01(w.seed + 1, 0, T * 3 * Ns) - 1.0).reshape(T, 3, n, n, n)
    return _finish(w, rho, J)


# ----------------------------------------------------------------------------- config 3
def config3_collision(n: int = 64, dtype: str = "f32") -> Workload:
    """Two Lorentz-contracted Gaussian discs (gamma = 10) at +-0.995c along z (configs[2]).

    History length ceil(max R/c/dt)+2 (PAPER.md:231 rule + 2); the discs overlap at t_c = 20 and
    are evaluated at the last step.  ``n`` < 64 gives a reduced copy for CPU-sized tests.
    """
    dx, dt = 0.2, 0.1
    max_r = math.sqrt(3.0) * (n - 1) * dx
    T = int(math.ceil(max_r / dt)) + 2
    w = Workload(f"c3_collision_{n}", (n,) * 3, (dx,) * 3, (n,) * 3, (dx,) * 3,
                 (-(n - 1) / 2 * dx,) * 3, dt, T, (T - 1,), dtype, seed=BASE_SEED + 3)
    x = _centres(n, dx)
    sig_t, sig_l, v = 1.0, 1.0 / 10.0, 0.995
    t_c = (T - 1) * dt - 2.0                  # 20.0 at n = 64
    gxy = np.exp(-x * x / (2 * sig_t ** 2))
    plane = gxy[:, None] * gxy[None, :]
    rho = np.empty((T, n, n, n))
    J = np.zeros((T, 3, n, n, n))
    for m in range(T):
        zc = v * (m * dt - t_c)
        ga = np.exp(-(x - zc) ** 2 / (2 * sig_l ** 2))
        gb = np.exp(-(x + zc) ** 2 / (2 * sig_l ** 2))
        rho[m] = (ga + gb)[:, None, None] * plane[None]
        J[m, 2] = (v * (ga - gb))[:, None, None] * plane[None]
    return _finish(w, rho, J)


# ----------------------------------------------------------------------------- config 4
def config4_detached(n: int = 48, n_plane: int = 256, n_out: int = 128, dtype: str = "f32") -> Workload:
    """Oscillating Gaussian blob observed on a detached plane at z = +10 (configs[3];
    the paper's detached observation region)."""
    dx, dt, ho, z_obs = 0.1, 0.05, 0.1, 10.0
    half_s = (n - 1) / 2 * dx
    half_o = (n_plane - 1) / 2 * ho
    r_max = math.sqrt(2 * (half_s + half_o) ** 2 + (z_obs + half_s) ** 2)
    k_max = int(math.floor(r_max / dt + 0.5))
    T = k_max + 1 + n_out
    w = Workload(f"c4_detached_{n}_{n_plane}", (n,) * 3, (dx,) * 3, (n_plane, n_plane, 1), (ho, ho, ho),
                 (-half_o, -half_o, z_obs), dt, T, tuple(range(T - n_out, T)), dtype, seed=BASE_SEED + 4)
    x = _centres(n, dx)
    sig, v0, omega = 0.5, 0.5, 2 * math.pi / 2.0
    g = np.exp(-x * x / (2 * sig * sig))
    blob = g[:, None, None] * g[None, :, None] * g[None, None, :]
    s = np.sin(omega * np.arange(T) * dt)
    rho = s[:, None, None, None] * blob[None]
    J = np.empty((T, 3, n, n, n))
    J[:, 0] = rho * (v0 / sig) * x[None, None, None, :]
    J[:, 1] = rho * (v0 / sig) * x[None, None, :, None]
    J[:, 2] = rho * (v0 / sig) * x[None, :, None, None]
    return _finish(w, rho, J)


# ----------------------------------------------------------------------------- config 5
def config5_large(n: int = 100, T: int = 200, dtype: str = "f32") -> Workload:
    """Sum of 16 drifting Gaussians with random amplitude, width, centre and velocity (configs[4])."""
    dx, dt = 0.1, 0.05
    w = Workload(f"c5_large_{n}", (n,) * 3, (dx,) * 3, (n,) * 3, (dx,) * 3, (-(n - 1) / 2 * dx,) * 3,
                 dt, T, (T - 1,), dtype, seed=BASE_SEED + 5)
    x = _centres(n, dx)
    box = n * dx
    u = uniform01(w.seed, 0, 16 * 8).reshape(16, 8)
    t_mid = 0.5 * (T - 1) * dt
    npd = w.np_dtype
    rho = np.zeros((T, n, n, n), dtype=npd)
    J = np.zeros((T, 3, n, n, n), dtype=npd)
    for g in range(16):
        amp = 2 * u[g, 0] - 1
        sig = 0.5 + u[g, 1]
        cen = (u[g, 2:5] - 0.5) * 0.6 * box
        cos_t, phi = 2 * u[g, 5] - 1, 2 * math.pi * u[g, 6]
        sin_t = math.sqrt(max(0.0, 1 - cos_t * cos_t))
        vel = 0.9 * u[g, 7] * np.array([sin_t * math.cos(phi), sin_t * math.sin(phi), cos_t])
        for m in range(T):
            cm = cen + vel * (m * dt - t_mid)
            gx = np.exp(-(x - cm[0]) ** 2 / (2 * sig * sig))
            gy = np.exp(-(x - cm[1]) ** 2 / (2 * sig * sig))
            gz = amp * np.exp(-(x - cm[2]) ** 2 / (2 * sig * sig))
            blob = gz[:, None, None] * gy[None, :, None] * gx[None, None, :]
            blob[np.abs(blob) < _TINY] = 0.0
            # accumulate in the run dtype's container but from fp64 terms (16 terms: the
            # rounding of the running sum is part of the *input*, identical for both sides)
            rho[m] += blob.astype(npd)
            for a in range(3):
                J[m, a] += (blob * vel[a]).astype(npd)
    w.rho, w.J = rho, J
    return w


# ----------------------------------------------------------------------------- paper's analytic sources
def paper_x1_constant(T: int, n: int = 15, dtype: str = "f64") -> Workload:
    """PAPER.md:122-137 (Sec. 3.1, Eq. (7)): rho = 1, J = (1,1,1) for t >= 0 on [-3,3]^3, 15^3 cells."""
    dx, dt = 6.0 / n, 0.05
    w = Workload("paper_x1", (n,) * 3, (dx,) * 3, (n,) * 3, (dx,) * 3, (-(n - 1) / 2 * dx,) * 3,
                 dt, T, (T - 1,), dtype)
    return _finish(w, np.ones((T, n, n, n)), np.ones((T, 3, n, n, n)))


def random_history(n_src, T: int, seed: int, dtype: str = "f64", spacing=(0.1, 0.1, 0.1),
                   n_obs=None, spacing_obs=None, origin_obs=None, dt: float = 0.05, c: float = 1.0) -> Workload:
    """Uniform [-1,1] history on an arbitrary (possibly anisotropic) grid -- for property tests."""
    nx, ny, nz = n_src
    n_obs = n_obs or n_src
    spacing_obs = spacing_obs or spacing
    origin_obs = origin_obs or tuple(-(n - 1) / 2 * h for n, h in zip(n_obs, spacing_obs))
    w = Workload("random", tuple(n_src), tuple(spacing), tuple(n_obs), tuple(spacing_obs),
                 tuple(origin_obs), dt, T, (T - 1,), dtype, c=c, seed=seed)
    Ns = nx * ny * nz
    rho = (2 * uniform01(seed, 0, T * Ns) - 1).reshape(T, nz, ny, nx)
    J = (2 * uniform01(seed + 1, 0, T * 3 * Ns) - 1).reshape(T, 3, nz, ny, nx)
    return _finish(w, rho, J)


def paper_table4_largest(n: int = 160, T: int = 500, dtype: str = "f32") -> Workload:
    """The paper's largest timed configuration, ntg = [160^3, 160^3], lts = 500 (PAPER.md:254,
    Table 4 lower; dx = 0.1, c dt = 0.05 as in configs[4], so the longest lag exceeds the history).
    The raw history is 33 GB in fp32: only one seeded snapshot (uniform [-1,1]) is generated on the
    host; ``device_history(torch)`` fills the device arrays with that snapshot shifted by m cells
    along x at step m (a copy per step, no arithmetic).  ``lazy`` tells bench.py that there are
    no host arrays (no end-to-end leg, no oracle sample)."""
    dx, dt = 0.1, 0.05
    w = Workload(f"paper_table4_{n}", (n,) * 3, (dx,) * 3, (n,) * 3, (dx,) * 3, (-(n - 1) / 2 * dx,) * 3,
                 dt, T, (T - 1,), dtype, seed=BASE_SEED + 160)
    w.lazy = True

    def device_history(torch):
        base = (2 * uniform01(w.seed, 0, 4 * n ** 3) - 1).reshape(4, n, n, n).astype(w.np_dtype)
        b = torch.from_numpy(base).cuda()
        rho = torch.empty((T, n, n, n), dtype=b.dtype, device="cuda")
        J = torch.empty((T, 3, n, n, n), dtype=b.dtype, device="cuda")
        for m in range(T):
            rho[m] = torch.roll(b[0], m, dims=2)
            J[m] = torch.roll(b[1:], m, dims=3)
        return rho, J

    w.device_history = device_history
    return w


def with_random_points(w: Workload, n: int, seed_offset: int = 0, margin: float = 0.0) -> Workload:
    """Replaces the observation grid of ``w`` by ``n`` seeded points, uniform in the box of the
    source grid (grown by ``margin`` on every side), rounded to the run dtype so that both sides
    see the same positions.  Unstructured observation sets are what detector positions or
    particle positions of a coupled solver look like."""
    half = [(a - 1) / 2.0 * h + 0.5 * h + margin for a, h in zip(w.n_src, w.spacing_src)]
    u = uniform01(w.seed + 4242 + seed_offset, 0, 3 * n).reshape(n, 3)
    pts = (2.0 * u - 1.0) * np.array(half)
    w.points = pts.astype(w.np_dtype).astype(np.float64)
    w.name = f"{w.name}_points{n}"
    w.n_obs = (n, 1, 1)
    return w


def smooth_in_time(w: Workload, period: float, depth: float = 0.3, base_step: int = 0) -> Workload:
    """Replaces the history of ``w`` by its snapshot ``base_step`` times 1 + depth*sin(2 pi m/period + phase_j)
    with a seeded phase per cell: white in space, smooth in time.  For fp32 parity on UNSTRUCTURED
    geometry: there a pair can sit within the fp32 rounding error of a retarded-index tie, and
    with a history that is white in time one flipped index is an O(1) error in its term although
    either neighbouring step is an equally good nearest snapshot ('harmless for
    smooth histories')."""
    m = np.arange(w.T, dtype=np.float64)
    Ns = w.N_s
    ph = 2.0 * np.pi * uniform01(w.seed + 97, 0, Ns).reshape(w.rho.shape[1:])
    f = 1.0 + depth * np.sin(2.0 * np.pi * m[:, None, None, None] / period + ph[None])
    w.rho = np.ascontiguousarray((w.rho[base_step].astype(np.float64)[None] * f).astype(w.np_dtype))
    w.J = np.ascontiguousarray((w.J[base_step].astype(np.float64)[None] * f[:, None]).astype(w.np_dtype))
    w.name = f"{w.name}_smooth{period:g}"
    return w


def slab_workload(w: Workload, z0: int, z1: int) -> Workload:
    """The workload restricted to source layers [z0, z1) (a rank's share when the SOURCE region is
    partitioned): its own grid size, ``slab_origin`` = the centre of its cell
    (0,0,0), and its own slab of the history; observation set unchanged.  Slicing only."""
    import copy
    v = copy.copy(w)
    v.n_src = (w.n_src[0], w.n_src[1], z1 - z0)
    o = w.origin_src
    v.slab_origin = (o[0], o[1], o[2] + z0 * w.spacing_src[2])
    v.rho = np.ascontiguousarray(w.rho[:, z0:z1])
    v.J = np.ascontiguousarray(w.J[:, :, z0:z1])
    return v

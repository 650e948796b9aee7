"""Pins for the fp64 CPU oracle (oracle/jefi_oracle.c) against what the paper and the
mathematics fix -- never against the oracle itself and never against the CUDA path.

Each test names the part of the sum it pins (SURVEY.md 8c "What pins each part").
"""
import math
import os

import numpy as np
import pytest

import oracle
import workloads as wl

HERE = os.path.dirname(os.path.abspath(__file__))
FOURPI = 4.0 * math.pi


def _single_cell_grid(n=(5, 5, 5), h=(0.1, 0.1, 0.1)):
    origin = tuple(-(a - 1) / 2 * b for a, b in zip(n, h))
    return n, origin, h


# --------------------------------------------------------------------------- worked example
def _golden_rows():
    rows = []
    with open(os.path.join(HERE, "golden", "worked_example.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            p = line.split()
            rows.append((p[0], int(p[1]), [float(v) for v in p[2:8]]))
    return rows


@pytest.mark.parametrize("obs_name,mode,sums", _golden_rows())
def test_worked_example_hand_sum(obs_name, mode, sums):
    """Whole formula, prefactor dV/4pi, index rule, screening, both derivative modes
    (Eq. (4)-(6), hand-summed in tests/golden/worked_example.txt)."""
    T = 8
    m = np.arange(T, dtype=np.float64)
    rho = np.zeros((T, 1, 1, 2))
    J = np.zeros((T, 3, 1, 1, 2))
    rho[:, 0, 0, 0] = 1 + m
    J[:, 2, 0, 0, 0] = m * m
    rho[:, 0, 0, 1] = 2
    J[:, 0, 0, 0, 1] = m
    J[:, 2, 0, 0, 1] = 1
    obs = {"A": (0.0, 0.0, 0.0), "B": (0.0, 4.0, 0.0)}[obs_name]
    E, B = oracle.fields((2, 1, 1), (0, 0, 0), (3, 3, 3), rho, J, dt=1.0, c=1.0, step=7,
                         obs_xyz=[obs], deriv_mode=mode, nthreads=1)
    pref = 27.0 / FOURPI
    assert abs(pref - 2.148591732) < 1e-9
    np.testing.assert_allclose(E[:, 0], pref * np.array(sums[:3]), rtol=1e-14, atol=1e-15)
    np.testing.assert_allclose(B[:, 0], pref * np.array(sums[3:]), rtol=1e-14, atol=1e-15)


def test_worked_example_printed_decimals():
    """The decimals printed in SURVEY.md 8c for obs B, centred mode."""
    T = 8
    m = np.arange(T, dtype=np.float64)
    rho = np.zeros((T, 1, 1, 2)); J = np.zeros((T, 3, 1, 1, 2))
    rho[:, 0, 0, 0] = 1 + m; J[:, 2, 0, 0, 0] = m * m
    rho[:, 0, 0, 1] = 2; J[:, 0, 0, 0, 1] = m; J[:, 2, 0, 0, 1] = 1
    E, B = oracle.fields((2, 1, 1), (0, 0, 0), (3, 3, 3), rho, J, dt=1.0, c=1.0, step=7,
                         obs_xyz=[(0, 4, 0)], nthreads=1)
    np.testing.assert_allclose(E[:, 0], [-0.532850749, 1.211805737, -3.222887598], atol=5e-10)
    np.testing.assert_allclose(B[:, 0], [-4.500225382, -0.051566202, 0.481284548], atol=5e-10)


# --------------------------------------------------------------------------- Coulomb
def test_coulomb_static_point_charge():
    """rho/R^3 term and prefactor: one constant charged cell gives E = q d/(4 pi R^3), B = 0 exactly."""
    w = wl.config2a_coulomb("f64", n=16, T=64)
    idx = w.obs_subset(400)
    pts = w.obs_points(idx)
    E, B = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, dt=w.dt, c=w.c,
                         step=w.steps[0], obs_xyz=pts)
    n = 16
    src = np.array(w.origin_src) + np.array([n // 2] * 3) * np.array(w.spacing_src)
    d = pts - src
    R = np.linalg.norm(d, axis=1)
    assert R.max() / w.dt < 63            # every retarded step is inside the stored history
    q = w.spacing_src[0] ** 3             # rho * dV
    expect = (q / FOURPI) * d.T / R ** 3
    np.testing.assert_allclose(E, expect, rtol=1e-13, atol=0)
    assert np.all(B == 0.0)


def test_index_order_and_anisotropic_cells():
    """x-fastest layout, J component planes, dV = dx*dy*dz, cell centres = origin + i*spacing:
    a lone charge at a non-symmetric index of an anisotropic grid sits where it should."""
    n, h = (4, 5, 6), (0.3, 0.2, 0.1)
    origin = (1.0, -2.0, 0.5)
    T = 40
    rho = np.zeros((T, n[2], n[1], n[0]))
    rho[:, 3, 2, 1] = 2.5                  # (ix,jy,kz) = (1,2,3)
    J = np.zeros((T, 3, n[2], n[1], n[0]))
    src = np.array(origin) + np.array([1, 2, 3]) * np.array(h)
    pts = np.array([[2.0, -1.0, 1.4], [0.2, -2.2, 0.1], [1.3, -1.6, 0.8 + 0.3]])
    E, B = oracle.fields(n, origin, h, rho, J, dt=0.1, c=1.0, step=T - 1, obs_xyz=pts)
    d = pts - src
    R = np.linalg.norm(d, axis=1)
    expect = 2.5 * (h[0] * h[1] * h[2]) / FOURPI * d.T / R ** 3
    np.testing.assert_allclose(E, expect, rtol=1e-13)
    assert np.all(B == 0.0)
    # the same charge carried as J_y only: B = (J x d)/R^3, E = 0 (steady)
    rho[:] = 0
    J[:, 1, 3, 2, 1] = 2.5
    E, B = oracle.fields(n, origin, h, rho, J, dt=0.1, c=1.0, step=T - 1, obs_xyz=pts)
    Jv = np.array([0, 2.5, 0])
    expectB = (h[0] * h[1] * h[2]) / FOURPI * np.cross(Jv[None, :], d).T / R ** 3
    np.testing.assert_allclose(B, expectB, rtol=1e-13)
    assert np.all(E == 0.0)


def test_screening_rule_strict_half_min_spacing():
    """Q5 / PAPER.md:75: a cell contributes iff R >= 0.5*min(dx,dy,dz)."""
    n, origin, h = (3, 3, 3), (-0.3, -0.2, -0.1), (0.3, 0.2, 0.1)     # rcut = 0.05
    T = 8
    rho = np.zeros((T, 3, 3, 3)); rho[:, 1, 1, 1] = 1.0               # cell centre at (0,0,0)
    J = np.zeros((T, 3, 3, 3, 3))
    pts = [(0, 0, 0), (0.049, 0, 0), (0.0, 0.0499999, 0), (0.05, 0, 0), (0, 0.051, 0)]
    E, _ = oracle.fields(n, origin, h, rho, J, dt=0.05, c=1.0, step=T - 1, obs_xyz=pts)
    assert np.all(E[:, :3] == 0.0)
    q = 0.3 * 0.2 * 0.1
    assert E[0, 3] == pytest.approx(q / FOURPI / 0.05 ** 2, rel=1e-13)
    assert E[1, 4] == pytest.approx(q / FOURPI / 0.051 ** 2, rel=1e-13)


# --------------------------------------------------------------------------- Biot-Savart
def test_biot_savart_finite_wire():
    """J x d / R^3 term and the right-hand rule: a steady line current; E = 0 exactly, B against
    the closed form of a finite straight segment B_phi = I/(4 pi s) (sin th2 - sin th1)."""
    w = wl.config2b_wire("f64", n=32, T=64)
    dx = w.spacing_src[0]
    cx = w.origin_src[0] + 16 * dx
    z_lo, z_hi = w.origin_src[2] - 0.5 * dx, w.origin_src[2] + 31.5 * dx   # outer cell faces
    pts, svals = [], []
    for s_cells in (1.5, 2.5, 4.5, 8.5):
        for z in (0.0, w.origin_src[2] + 4 * dx + 0.5 * dx):            # mid-wire, 4 cells from the end
            pts.append((cx + s_cells * dx, cx, z)); svals.append(s_cells * dx)
    pts = np.array(pts)
    E, B = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, dt=w.dt, c=w.c,
                         step=63, obs_xyz=pts)
    assert np.all(E == 0.0)
    I = 1.0 * dx * dx
    for i, (p, s) in enumerate(zip(pts, svals)):
        sin2 = (z_hi - p[2]) / math.hypot(s, z_hi - p[2])
        sin1 = (z_lo - p[2]) / math.hypot(s, z_lo - p[2])
        closed = I / (FOURPI * s) * (sin2 - sin1)
        # J || +z, obs at +x  =>  B || +y
        assert B[1, i] > 0
        assert abs(B[1, i] - closed) / closed < 5e-3
        assert abs(B[0, i]) < 1e-16 and abs(B[2, i]) < 1e-16
    # 4.5 cells away at mid-wire the midpoint rule is very accurate (survey arithmetic: 0.003 %)
    assert abs(B[1, 4] - I / (FOURPI * svals[4]) * 2 * (z_hi / math.hypot(svals[4], z_hi))) / B[1, 4] < 1e-4


def test_biot_savart_exact_hand_sum():
    """The same wire against the 32-term sum written out term by term."""
    w = wl.config2b_wire("f64", n=32, T=64)
    dx = w.spacing_src[0]
    p = np.array([w.origin_src[0] + 18.5 * dx, w.origin_src[1] + 14.5 * dx, 0.31])
    _, B = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, dt=w.dt, c=w.c,
                         step=63, obs_xyz=[p])
    acc = np.zeros(3)
    for kz in range(32):
        s = np.array([w.origin_src[0] + 16 * dx, w.origin_src[1] + 16 * dx, w.origin_src[2] + kz * dx])
        d = p - s
        acc += np.cross([0, 0, 1.0], d) / np.linalg.norm(d) ** 3
    np.testing.assert_allclose(B[:, 0], acc * dx ** 3 / FOURPI, rtol=1e-13, atol=1e-18)


# --------------------------------------------------------------------------- linear structure
@pytest.mark.parametrize("mode", [0, 1])
def test_linearity_and_superposition(mode):
    a = wl.random_history((6, 5, 4), 48, seed=11, spacing=(0.1, 0.12, 0.09))
    b = wl.random_history((6, 5, 4), 48, seed=23, spacing=(0.1, 0.12, 0.09))
    pts = np.array([[0.05, 0.0, 0.0], [1.0, -0.5, 0.3], [-0.31, 0.22, -0.18], [0.25, 0.3, 0.135]])
    kw = dict(dt=a.dt, c=1.0, step=47, obs_xyz=pts, deriv_mode=mode)
    Ea, Ba = oracle.fields(a.n_src, a.origin_src, a.spacing_src, a.rho, a.J, **kw)
    Eb, Bb = oracle.fields(a.n_src, a.origin_src, a.spacing_src, b.rho, b.J, **kw)
    al, be = 1.75, -0.375
    Ec, Bc = oracle.fields(a.n_src, a.origin_src, a.spacing_src, al * a.rho + be * b.rho,
                           al * a.J + be * b.J, **kw)
    np.testing.assert_allclose(Ec, al * Ea + be * Eb, rtol=0, atol=1e-12 * np.abs(Ea).max())
    np.testing.assert_allclose(Bc, al * Ba + be * Bb, rtol=0, atol=1e-12 * np.abs(Ba).max())


def test_c_rescaling_invariance():
    """Powers of c (Q7): B(c,dt;J) = B(1,c dt;J) and E(c,dt;rho,J) = E(1,c dt;rho,J/c), exactly."""
    w = wl.random_history((5, 4, 6), 64, seed=5, spacing=(0.1, 0.1, 0.1))
    pts = np.array([[0.05, 0.0, 0.0], [0.7, -0.5, 0.3], [-0.3, 0.2, -0.15]])
    for mode in (0, 1):
        E2, B2 = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, dt=0.025, c=2.0,
                               step=63, obs_xyz=pts, deriv_mode=mode)
        _, B1 = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, dt=0.05, c=1.0,
                              step=63, obs_xyz=pts, deriv_mode=mode)
        E1, _ = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J / 2.0, dt=0.05, c=1.0,
                              step=63, obs_xyz=pts, deriv_mode=mode)
        np.testing.assert_allclose(B2, B1, rtol=1e-12, atol=1e-13 * np.abs(B1).max())
        np.testing.assert_allclose(E2, E1, rtol=1e-12, atol=1e-13 * np.abs(E1).max())


def test_time_translation():
    """Shifting the history and the evaluation step together changes nothing (interior steps)."""
    w = wl.random_history((4, 4, 4), 80, seed=3)
    pts = np.array([[0.0, 0.05, 0.0], [0.45, -0.2, 0.3]])
    shift = 9
    kmax = int(max(np.linalg.norm(pts[:, None, :] - _all_centres(w), axis=2).max() / w.dt + 0.5, 0)) + 1
    n = 60
    assert n - kmax >= 2 and n + shift + 1 <= 78
    E0, B0 = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, dt=w.dt, c=1.0,
                           step=n + shift, obs_xyz=pts)
    E1, B1 = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho[shift:], w.J[shift:], dt=w.dt,
                           c=1.0, step=n, obs_xyz=pts)
    assert np.array_equal(E0, E1) and np.array_equal(B0, B1)


def _all_centres(w):
    nx, ny, nz = w.n_src
    g = np.stack(np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij"), -1).reshape(-1, 3)
    return (np.array(w.origin_src) + g * np.array(w.spacing_src))[None, :, :]


# --------------------------------------------------------------------------- causality / index rule
@pytest.mark.parametrize("q_frac,k_expect", [(4.4, 4), (4.6, 5), (7.0, 7), (1.4, 1), (1.6, 2)])
def test_switch_on_causality_centred(q_frac, k_expect):
    """Retarded index k = floor(R/(c dt)+0.5), m<0 rule and centred derivative ends: a cell that
    switches on at step m0 is seen first at n = m0-1+k (the centred precursor), with the closed
    forms of SURVEY.md 8c, and is exactly Coulomb from n = m0+1+k on."""
    n, origin, h = _single_cell_grid()
    dt, c, T, m0, q0 = 0.05, 1.0, 40, 6, 1.5
    R = q_frac * dt * c
    if R < 0.05:
        pytest.skip("inside the screening radius")
    rho = np.zeros((T, 5, 5, 5)); rho[m0:, 2, 2, 2] = q0
    J = np.zeros((T, 3, 5, 5, 5))
    dvec = np.array([0.6, -0.48, 0.64]) * R                     # |dvec| = R
    assert oracle.lag(dvec, (0, 0, 0), dt=dt, c=c) == k_expect
    pref = h[0] * h[1] * h[2] / FOURPI
    for nstep in range(k_expect, T - 2):
        E, B = oracle.fields(n, origin, h, rho, J, dt=dt, c=c, step=nstep, obs_xyz=[dvec], nthreads=1)
        m = nstep - k_expect
        if m < m0 - 1:
            expect = 0.0
        elif m == m0 - 1:
            expect = q0 / (2 * dt * c * R ** 2)
        elif m == m0:
            expect = q0 / R ** 3 + q0 / (2 * dt * c * R ** 2)
        else:
            expect = q0 / R ** 3
        np.testing.assert_allclose(E[:, 0], pref * dvec * expect, rtol=1e-12, atol=0)
        assert np.all(B == 0)


def test_switch_on_backward_mode_has_no_precursor():
    """Paper's backward difference: zero for n-k < m0, q0/R^3 + q0/(dt c R^2) at
    n-k = m0 (the switch-on spike), Coulomb after; with m0 = 0 the spike uses f[-1] = 0."""
    n, origin, h = _single_cell_grid()
    dt, c, T, q0 = 0.05, 1.0, 30, 2.0
    dvec = np.array([0.0, 0.3, 0.4])                          # R = 0.5, k = 10
    R, k = 0.5, 10
    pref = h[0] ** 3 / FOURPI
    for m0 in (0, 5):
        rho = np.zeros((T, 5, 5, 5)); rho[m0:, 2, 2, 2] = q0
        J = np.zeros((T, 3, 5, 5, 5))
        for nstep in range(0, T):
            E, _ = oracle.fields(n, origin, h, rho, J, dt=dt, c=c, step=nstep, obs_xyz=[dvec],
                                 deriv_mode=1, nthreads=1)
            m = nstep - k
            expect = 0.0 if m < m0 else (q0 / R ** 3 + q0 / (dt * c * R ** 2) if m == m0 else q0 / R ** 3)
            np.testing.assert_allclose(E[:, 0], pref * dvec * expect, rtol=1e-12, atol=0)


def test_Jdot_term_sign_and_weight():
    """-J_dot/(c^2 R) term (Q1): a linearly ramping uniform current in one cell, rho = 0."""
    n, origin, h = _single_cell_grid()
    dt, c, T = 0.05, 2.0, 40
    rho = np.zeros((T, 5, 5, 5)); J = np.zeros((T, 3, 5, 5, 5))
    slope = np.array([0.7, -1.1, 0.4])
    for m in range(T):
        J[m, :, 2, 2, 2] = slope * (m * dt)
    dvec = np.array([0.3, 0.0, 0.4])
    R = 0.5
    k = oracle.lag(dvec, (0, 0, 0), dt=dt, c=c)
    assert k == 5
    E, B = oracle.fields(n, origin, h, rho, J, dt=dt, c=c, step=30, obs_xyz=[dvec], nthreads=1)
    pref = h[0] ** 3 / FOURPI
    Jm = slope * ((30 - k) * dt)
    np.testing.assert_allclose(E[:, 0], -pref * slope / (c * c * R), rtol=1e-11)
    np.testing.assert_allclose(B[:, 0], pref * np.cross(Jm / R ** 3 + slope / (c * R ** 2), dvec), rtol=1e-11)


def test_late_time_constancy():
    """Paper's 'saturation': with sources constant after switch-on the output is
    bit-identical from one step to the next once n - k_max >= m0 + 1."""
    T = 200
    w = wl.paper_x1_constant(T, n=7)
    m0 = 3
    w.rho[:m0] = 0; w.J[:m0] = 0
    pts = w.obs_points(w.obs_subset(40))
    kmax = int(np.floor(np.linalg.norm(pts[:, None, :] - _all_centres(w), axis=2).max() / w.dt + 0.5))
    n0 = kmax + m0 + 1
    assert n0 + 2 < T
    kw = dict(dt=w.dt, c=1.0, obs_xyz=pts)
    Ea, Ba = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, step=n0, **kw)
    Eb, Bb = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, step=n0 + 2, **kw)
    Ec, _ = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, step=n0 - 3, **kw)
    assert np.array_equal(Ea, Eb) and np.array_equal(Ba, Bb)
    assert not np.array_equal(Ea, Ec)


# --------------------------------------------------------------------------- symmetry
def test_mirror_symmetry_static_blob():
    """Spherically symmetric static blob on a symmetric grid: B = 0 and E(-x) = -E(x)."""
    n, dx, T = 8, 0.1, 40
    x = (np.arange(n) - (n - 1) / 2) * dx
    g = np.exp(-x * x / (2 * 0.2 ** 2))
    blob = g[:, None, None] * g[None, :, None] * g[None, None, :]
    rho = np.broadcast_to(blob, (T, n, n, n)).copy()
    J = np.zeros((T, 3, n, n, n))
    origin = (x[0],) * 3
    pts = np.array([[0.15, 0.05, -0.25], [0.62, -0.31, 0.2], [0.05, 0.05, 0.05]])
    pts = np.concatenate([pts, -pts])
    E, B = oracle.fields((n,) * 3, origin, (dx,) * 3, rho, J, dt=0.05, c=1.0, step=T - 1, obs_xyz=pts)
    np.testing.assert_allclose(E[:, :3], -E[:, 3:], rtol=1e-12, atol=1e-15)
    assert np.all(B == 0)
    # and E points outward for a positive blob
    assert np.all(np.sum(E[:, :3].T * pts[:3], axis=1) > 0)


# --------------------------------------------------------------------------- far-zone radiation
def _dipole_fields(R, nhat, n_times=40):
    """Oscillating Gaussian dipole P = z G sin(wt): rho = -div P, J = dP/dt (continuity holds
    everywhere, including the box edge where G ~ 1e-4 of its peak value is still small)."""
    ng, dx, sig, om, dt = 16, 0.25, 0.5, math.pi, 0.05
    x = (np.arange(ng) - (ng - 1) / 2) * dx
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    G = np.exp(-(X * X + Y * Y + Z * Z) / (2 * sig * sig))
    M0 = 0                                   # sources are zero for t < 0 (m < 0 rule)
    n_last = int(round((R + 12.0) / dt))
    T = n_last + 2
    t = np.arange(T) * dt
    rho = (Z / sig ** 2 * G)[None] * np.sin(om * t)[:, None, None, None]
    J = np.zeros((T, 3, ng, ng, ng))
    J[:, 2] = (G * om)[None] * np.cos(om * t)[:, None, None, None]
    p = R * np.asarray(nhat, dtype=np.float64)
    Es, Bs = [], []
    for n_abs in np.linspace(int(round((R + 10.0) / dt)), n_last, n_times).astype(int):
        E, B = oracle.fields((ng,) * 3, (x[0],) * 3, (dx,) * 3, rho, J, dt=dt, c=1.0,
                             step=int(n_abs) - M0, obs_xyz=[p], nthreads=1)
        Es.append(E[:, 0]); Bs.append(B[:, 0])
    return np.array(Es), np.array(Bs)


@pytest.mark.parametrize("R,nhat", [
    (20.0, (1.0, 0.0, 0.0)), (20.0, (0.6, 0.0, 0.8)), (40.0, (0.6, 0.0, 0.8)), (80.0, (0.6, 0.0, 0.8))])
def test_far_zone_radiation_is_transverse_and_outgoing(R, nhat):
    """Fixes the sign of the J_dot/R term (Q1) and the cross-product order (Q8) together: in the
    far zone of a source obeying continuity, |E_perp| = |B| (c = 1), E x B points outward, and the
    radial part of E is the textbook intermediate-zone term of an oscillating dipole,
    |E_r|/|E_theta| = 2 cot(theta)/(omega R) (0 on the equator, falling like 1/R).  With the '+'
    of Eq. (1) the radial part would be 2.66 |E_perp| at any R and the Poynting vector would point
    inward (that table's 1.3e-3 radial fraction is superseded by the closed form)."""
    Es, Bs = _dipole_fields(R, nhat)
    nh = np.asarray(nhat)
    Er = Es @ nh
    Eperp = Es - Er[:, None] * nh[None, :]
    nE, nB, nR = np.linalg.norm(Eperp), np.linalg.norm(Bs), np.linalg.norm(Er)
    assert 0.998 < nE / nB < 1.002
    if nhat[2] == 0.0:
        assert nR / nE < 1e-6                          # equator: no radial part at all
    else:
        closed = 2.0 * (nhat[2] / math.hypot(nhat[0], nhat[1])) / (math.pi * R)
        assert abs(nR / nE / closed - 1.0) < 0.05
    S = np.cross(Es, Bs).sum(axis=0)
    assert S @ nh / np.linalg.norm(S) > 0.999
    assert abs((Bs @ nh)).max() < 1e-3 * np.abs(Bs).max()


# --------------------------------------------------------------------------- the paper's own numbers (soft)
def test_paper_x1_legend_magnitude():
    """PAPER.md:165 (Fig. 4/5 legends): at t = 2.5 the in-plane |E_theo|, |B_theo| peak near 0.5 for
    rho = 1, J = (1,1,1) on the 15^3 grid.  This reading gives 0.529 for both (the
    switch-on shell does not contribute in centred mode): an order-one check of dV/4pi, cell
    centres, screening radius and the m<0 rule, not a tight pin (the figures are not available)."""
    n_eval = 50                                   # t = 2.5 at dt = 0.05
    w = wl.paper_x1_constant(n_eval + 1, n=15)
    plane = np.arange(15 * 15) + 7 * 15 * 15      # z = 0 layer
    pts = w.obs_points(plane)
    assert np.all(pts[:, 2] == 0.0)
    E, B = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, dt=w.dt, c=1.0,
                         step=n_eval, obs_xyz=pts)
    e_max = np.sqrt(E[0] ** 2 + E[1] ** 2).max()
    b_max = np.sqrt(B[0] ** 2 + B[1] ** 2).max()
    assert 0.4 < e_max < 0.65 and 0.4 < b_max < 0.65        # the paper's legend: ~0.5
    assert abs(e_max - 0.529) < 1e-3 and abs(b_max - 0.529) < 1e-3


def test_memory_model_eq10():
    """PAPER.md:233 Eq. (10) x 4 bytes reproduces Table 3 up to a constant
    context overhead -- the evidence that the paper stores fp32 (D2)."""
    table = {(160, 500): 31707, (100, 2000): 30899, (100, 500): 8011, (70, 6000): 31775,
             (70, 2000): 10839, (70, 500): 2991, (60, 9000): 30025, (60, 6000): 20137,
             (60, 2000): 6953, (60, 500): 2009, (20, 9000): 1461, (20, 6000): 1093,
             (20, 2000): 605, (20, 500): 421}
    resid = []
    for (n, lts), mib in table.items():
        floats = (lts + 1) * n ** 3 * 4 + n ** 3 * 6
        resid.append(mib - floats * 4 / 2 ** 20)
    resid = np.array(resid)
    assert resid.min() > 300 and resid.max() < 420 and resid.std() < 25


# --------------------------------------------------------------------------- input promotion
def test_f32_inputs_are_promoted_not_recomputed():
    w = wl.random_history((4, 3, 5), 40, seed=9, dtype="f32")
    pts = np.array([[0.3, 0.1, -0.2], [0.0, 0.0, 0.05]])
    kw = dict(dt=w.dt, c=1.0, step=39, obs_xyz=pts)
    E32, B32 = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, **kw)
    E64, B64 = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho.astype(np.float64),
                             w.J.astype(np.float64), **kw)
    assert np.array_equal(E32, E64) and np.array_equal(B32, B64)


def test_argument_validation():
    w = wl.random_history((2, 2, 2), 4, seed=1)
    with pytest.raises(ValueError):
        oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, dt=w.dt, c=1.0, step=4, obs_xyz=[(0, 0, 1)])
    with pytest.raises(ValueError):
        oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, dt=-1.0, c=1.0, step=0, obs_xyz=[(0, 0, 1)])


# --------------------------------------------------------------------------- derivative ends, T = 1, tie direction
def _one_cell_nonlinear(T):
    """One source cell at the origin (grid 1x1x1, spacing 0.1: dV = 1e-3, rcut = 0.05) with a
    history that is NOT linear in the step index, so that a centred, a one-sided and a
    half-weighted one-sided difference all give different numbers:
        rho[m] = m^2 + 1,    J[m] = (m^3, -2 m^2, 3 m + m^2)."""
    m = np.arange(T, dtype=np.float64)
    rho = (m * m + 1.0).reshape(T, 1, 1, 1)
    J = np.stack([m ** 3, -2.0 * m * m, 3.0 * m + m * m], axis=1).reshape(T, 3, 1, 1, 1)
    return rho, J


def _one_cell_expect(dvec, c, rho_m, rhod, J_m, Jd, dV=1e-3):
    """Eq. (4)-(5) for ONE cell, written out: the closed form the pins below
    compare with.  rho_m, J_m = stored values at the retarded step, rhod, Jd = the time
    derivative SURVEY.md 8c's definition of D prescribes there (worked out by hand per test)."""
    d = np.asarray(dvec, dtype=np.float64)
    R = float(np.linalg.norm(d))
    E = d * (rho_m / R ** 3 + rhod / (c * R ** 2)) - np.asarray(Jd) / (c * c * R)
    B = np.cross(np.asarray(J_m) / R ** 3 + np.asarray(Jd) / (c * R ** 2), d)
    return dV / FOURPI * E, dV / FOURPI * B


def test_centred_derivative_newest_step_is_one_sided():
    """Q2 / SURVEY.md 8c definition of D, end m = T-1: (f[T-1] - f[T-2])/dt -- NOT /(2 dt).
    c dt = 1 and R = 0.08 (outside rcut = 0.05) give q = 0.08, k = 0, so evaluating the newest
    step n = T-1 reads the record m = T-1 itself.  By hand, T = 6, dt = 0.5, c = 2:
      rho[5] = 26, rho[4] = 17  ->  rho_dot = 9/0.5 = 18           (half-weighted: 9)
      J[5] = (125, -50, 40), J[4] = (64, -32, 28)  ->  J_dot = (122, -36, 24)."""
    T, dt, c = 6, 0.5, 2.0
    rho, J = _one_cell_nonlinear(T)
    dvec = np.array([0.048, -0.064, 0.0])                   # |d| = 0.08
    assert oracle.lag(dvec, (0, 0, 0), dt=dt, c=c) == 0
    E, B = oracle.fields((1, 1, 1), (0, 0, 0), (0.1, 0.1, 0.1), rho, J, dt=dt, c=c, step=T - 1,
                         obs_xyz=[dvec], nthreads=1)
    Ee, Be = _one_cell_expect(dvec, c, 26.0, 18.0, (125.0, -50.0, 40.0), (122.0, -36.0, 24.0))
    np.testing.assert_allclose(E[:, 0], Ee, rtol=1e-13)
    np.testing.assert_allclose(B[:, 0], Be, rtol=1e-13)


def test_centred_derivative_oldest_step_is_one_sided():
    """Q2, end m = 0: (f[1] - f[0])/dt.  Same geometry (k = 0), evaluated at n = 0.  By hand:
      rho[0] = 1, rho[1] = 2 -> rho_dot = 1/0.5 = 2;  J[0] = 0, J[1] = (1, -2, 4) -> J_dot = (2, -4, 8)."""
    T, dt, c = 6, 0.5, 2.0
    rho, J = _one_cell_nonlinear(T)
    dvec = np.array([0.048, -0.064, 0.0])
    E, B = oracle.fields((1, 1, 1), (0, 0, 0), (0.1, 0.1, 0.1), rho, J, dt=dt, c=c, step=0,
                         obs_xyz=[dvec], nthreads=1)
    Ee, Be = _one_cell_expect(dvec, c, 1.0, 2.0, (0.0, 0.0, 0.0), (2.0, -4.0, 8.0))
    np.testing.assert_allclose(E[:, 0], Ee, rtol=1e-13)
    np.testing.assert_allclose(B[:, 0], Be, rtol=1e-13)


def test_centred_derivative_interior_step_same_geometry():
    """The interior formula in the same k = 0 set-up (n = 3): (f[4] - f[2])/(2 dt).  By hand:
      rho: (17 - 5)/1 = 12;  J[3] = (27, -18, 18), J_dot = ((64-8), (-32+8), (28-10))/1 = (56, -24, 18)."""
    T, dt, c = 6, 0.5, 2.0
    rho, J = _one_cell_nonlinear(T)
    dvec = np.array([0.048, -0.064, 0.0])
    E, B = oracle.fields((1, 1, 1), (0, 0, 0), (0.1, 0.1, 0.1), rho, J, dt=dt, c=c, step=3,
                         obs_xyz=[dvec], nthreads=1)
    Ee, Be = _one_cell_expect(dvec, c, 10.0, 12.0, (27.0, -18.0, 18.0), (56.0, -24.0, 18.0))
    np.testing.assert_allclose(E[:, 0], Ee, rtol=1e-13)
    np.testing.assert_allclose(B[:, 0], Be, rtol=1e-13)


def test_single_stored_step_has_zero_derivative():
    """Q2, T = 1: no second snapshot exists, D = 0 in centred mode: pure Coulomb + Biot-Savart of
    the one stored record (rho = 1, J = 0 from the recipe above is too dull: use rho = 3, J = (1,2,-1)).
    In the paper's backward mode f[-1] = 0 gives D = f[0]/dt instead."""
    rho = np.full((1, 1, 1, 1), 3.0)
    J = np.array([1.0, 2.0, -1.0]).reshape(1, 3, 1, 1, 1)
    dvec = np.array([0.0, 0.06, 0.08])                      # |d| = 0.1, q = 0.1 -> k = 0
    kw = dict(dt=0.5, c=2.0, step=0, obs_xyz=[dvec], nthreads=1)
    E, B = oracle.fields((1, 1, 1), (0, 0, 0), (0.1, 0.1, 0.1), rho, J, **kw)
    Ee, Be = _one_cell_expect(dvec, 2.0, 3.0, 0.0, (1.0, 2.0, -1.0), (0.0, 0.0, 0.0))
    np.testing.assert_allclose(E[:, 0], Ee, rtol=1e-13)
    np.testing.assert_allclose(B[:, 0], Be, rtol=1e-13)
    E1, B1 = oracle.fields((1, 1, 1), (0, 0, 0), (0.1, 0.1, 0.1), rho, J, deriv_mode=1, **kw)
    Ee1, Be1 = _one_cell_expect(dvec, 2.0, 3.0, 6.0, (1.0, 2.0, -1.0), (2.0, 4.0, -2.0))
    np.testing.assert_allclose(E1[:, 0], Ee1, rtol=1e-13)
    np.testing.assert_allclose(B1[:, 0], Be1, rtol=1e-13)


@pytest.mark.parametrize("R,k_expect", [(0.3125, 3), (0.0625, 1), (0.4375, 4), (0.5625, 5)])
def test_rounding_tie_goes_up(R, k_expect):
    """Q3: k = floor(q + 1/2) -- an exact tie rounds UP (round-half-even would give 2 at q = 2.5,
    0 at q = 0.5 and 4 at q = 4.5).  Binary-exact numbers: c = 1, dt = 0.125, axis-aligned
    R = 0.3125 = 2.5 dt (0.0625 = 0.5 dt, 0.4375 = 3.5 dt, 0.5625 = 4.5 dt), all representable, so
    q is the exact half-integer in the oracle's arithmetic.  A charge switched on at step m0 in
    backward mode is first seen at exactly n = m0 + k (no precursor), which fixes k."""
    dt, c, T, m0, q0 = 0.125, 1.0, 16, 4, 2.0
    dvec = np.array([R, 0.0, 0.0])
    assert R / (c * dt) == k_expect - 0.5                   # an exact tie
    assert oracle.lag(dvec, (0, 0, 0), dt=dt, c=c) == k_expect
    rho = np.zeros((T, 1, 1, 1)); rho[m0:] = q0
    J = np.zeros((T, 3, 1, 1, 1))
    first = None
    for n in range(T):
        E, _ = oracle.fields((1, 1, 1), (0, 0, 0), (0.1, 0.1, 0.1), rho, J, dt=dt, c=c, step=n,
                             obs_xyz=[dvec], deriv_mode=1, nthreads=1)
        if first is None and E[0, 0] != 0.0:
            first = n
            # the switch-on spike of the backward difference, closed form
            expect = 1e-3 / FOURPI * R * (q0 / R ** 3 + q0 / (dt * c * R ** 2))
            assert E[0, 0] == pytest.approx(expect, rel=1e-13)
    assert first == m0 + k_expect

"""Property of the input recipe (Q3), checked without a GPU.

The retarded step is k = floor(R/(c dt) + 1/2).  The oracle decides it in fp64, the fp32 kernel
in fp32: the two can only disagree when q = R/(c dt) sits within the fp32 error of a
half-integer.  On every BASELINE.json config the source and observation lattices are
commensurate, so q takes a finite set of values; this test enumerates that set (every distinct
|offset| triple of the lattice pair) and asserts that none comes closer to a tie than several
times the fp32 error of q, and that an fp32 evaluation of q with a +-2 ulp perturbation of R
picks the same step as fp64 for every one of them.  It also fixes the history lengths the
configs promise (T covers the longest delay, or is deliberately shorter in c5)."""
import numpy as np
import pytest

import workloads as wl


def _axis_offsets(w, a):
    no, ns = w.n_obs[a], w.n_src[a]
    xo = w.origin_obs[a] + np.arange(no) * w.spacing_obs[a]
    xs = w.origin_src[a] + np.arange(ns) * w.spacing_src[a]
    d = np.abs(xo[:, None] - xs[None, :]).ravel()
    return np.unique(np.round(d, 10))


def _lattice_q(w):
    dx, dy, dz = (_axis_offsets(w, a) for a in range(3))
    r2 = (dx * dx)[:, None, None] + (dy * dy)[None, :, None] + (dz * dz)[None, None, :]
    r2 = np.unique(np.round(r2.ravel(), 9))
    return np.sqrt(r2) / (w.c * w.dt)


CONFIGS = [("c1", 5e-3), ("c2", 3e-3), ("c3", 5e-4), ("c4", 5e-4), ("c5", 3e-4)]


@pytest.mark.parametrize("name,margin", CONFIGS, ids=[c[0] for c in CONFIGS])
def test_no_lag_sits_near_a_tie(name, margin):
    w = _geometry_only(name)          # descriptors only: no multi-GB histories are generated
    q = _lattice_q(w)
    tie_dist = np.abs(q - np.floor(q) - 0.5)
    assert tie_dist.min() > margin, (name, tie_dist.min())
    # fp32 decision with a perturbed R equals the fp64 decision for every lattice distance
    k64 = np.floor(q + 0.5).astype(np.int64)
    R32 = (q * (w.c * w.dt)).astype(np.float32)
    inv = np.float32(1.0 / (w.c * w.dt))
    for ulps in (-2, 0, 2):
        Rp = R32 if ulps == 0 else np.nextafter(np.nextafter(R32, np.float32(np.inf * ulps)),
                                                np.float32(np.inf * ulps))
        k32 = np.floor((Rp * inv).astype(np.float32) + np.float32(0.5)).astype(np.int64)
        assert np.array_equal(k32, k64), (name, ulps, int((k32 != k64).sum()))
        # the tiled kernels' form: one FMA R * (1 + 2^-21)/(c dt) + 1.5*2^23, rounded to nearest even
        # (the relative bias sends exact ties up, Q3) -- no lattice distance may sit so
        # close BELOW a tie that the bias lifts it over
        inv_b = np.float32((1.0 / (w.c * w.dt)) * (1.0 + 2.0 ** -21))
        kb = np.rint(Rp.astype(np.float64) * np.float64(inv_b)).astype(np.int64)
        assert np.array_equal(kb, k64), (name, ulps, "biased", int((kb != k64).sum()))


def _geometry_only(name):
    """The Workload descriptors of a config without its (large) rho/J arrays."""
    W = wl.Workload
    if name == "c1":
        return wl.config1_tiny()
    if name == "c2":
        return wl.config2a_coulomb("f32")
    if name == "c3":
        w = wl.config3_collision(n=16)
        return W("c3geom", (64, 64, 64), w.spacing_src, (64, 64, 64), w.spacing_obs,
                 tuple(-(64 - 1) / 2 * h for h in w.spacing_obs), w.dt, 221, (220,), "f32", c=w.c)
    if name == "c4":
        w = wl.config4_detached(n=8, n_plane=8, n_out=2)
        return W("c4geom", (48, 48, 48), w.spacing_src, (256, 256, 1), w.spacing_obs,
                 (-(256 - 1) / 2 * w.spacing_obs[0], -(256 - 1) / 2 * w.spacing_obs[1], w.origin_obs[2]),
                 w.dt, 622, (621,), "f32", c=w.c)
    w = wl.config5_large(n=8, T=4)
    return W("c5geom", (100, 100, 100), w.spacing_src, (100, 100, 100), w.spacing_obs,
             tuple(-(100 - 1) / 2 * h for h in w.spacing_obs), w.dt, 200, (199,), "f32", c=w.c)


def test_geometry_only_descriptors_match_the_generators():
    """_geometry_only must describe the same lattices as the real generators (checked on the
    configs that are cheap to generate in full, and on the spacings/offsets of the others)."""
    w3 = wl.config3_collision(n=16)
    assert w3.spacing_src == (0.2, 0.2, 0.2) and w3.dt == 0.1 and w3.c == 1.0
    g4 = _geometry_only("c4")
    w4 = wl.config4_detached(n=8, n_plane=8, n_out=2)
    assert g4.spacing_src == w4.spacing_src == (0.1, 0.1, 0.1) and g4.origin_obs[2] == w4.origin_obs[2] == 10.0
    assert g4.dt == w4.dt == 0.05
    g5 = _geometry_only("c5")
    assert g5.spacing_src == (0.1, 0.1, 0.1) and g5.dt == 0.05


def test_history_lengths_cover_the_longest_delay():
    for name, T_expected, covered in (("c1", 32, True), ("c2", 64, True), ("c3", 221, True),
                                      ("c4", 622, True), ("c5", 200, False)):
        w = _geometry_only(name)
        assert w.T == T_expected
        k_max = int(np.floor(_lattice_q(w).max() + 0.5))
        # covered: the newest evaluation step reaches no lag before the stored history
        assert (k_max <= w.T - 1) == covered, (name, k_max, w.T)

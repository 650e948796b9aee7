"""Host-side pieces that hold none of the method's arithmetic: the seeded input generators added in
round 2 (unstructured observation points, time-smooth histories, the lazily generated 160^3
workload) and the bench's descriptors.  No GPU, no oracle arithmetic."""
import numpy as np
import pytest

import workloads as wl


def test_random_points_are_seeded_rounded_and_inside_the_source_box():
    w = wl.with_random_points(wl.config3_collision(n=16), 5000)
    v = wl.with_random_points(wl.config3_collision(n=16), 5000)
    assert w.N_o == 5000 and w.points.shape == (5000, 3) and w.points.dtype == np.float64
    np.testing.assert_array_equal(w.points, v.points)                        # pure function of the seed
    np.testing.assert_array_equal(w.points, w.points.astype(np.float32).astype(np.float64))   # fp32-exact
    half = 16 * 0.2 / 2
    assert np.abs(w.points).max() <= half and np.abs(w.points).max() > 0.9 * half
    assert w.obs_points([3, 7]).shape == (2, 3)
    np.testing.assert_array_equal(w.obs_points([3, 7]), w.points[[3, 7]])
    idx = w.obs_subset(300)
    assert idx.min() >= 0 and idx.max() < 5000 and len(np.unique(idx)) == len(idx)
    assert len(w.obs_subset(10 ** 6)) == 5000
    u = wl.with_random_points(wl.config3_collision(n=16), 5000, seed_offset=1)
    assert not np.array_equal(u.points, w.points)


def test_smooth_in_time_is_white_in_space_and_smooth_in_time():
    w = wl.smooth_in_time(wl.random_history((5, 4, 3), 32, seed=3, dtype="f64"), 32.0)
    assert w.rho.shape == (32, 3, 4, 5) and w.J.shape == (32, 3, 3, 4, 5)
    # every cell's history is its first-snapshot value times 1 + 0.3 sin(...): bounded, no jumps
    base = wl.random_history((5, 4, 3), 32, seed=3, dtype="f64").rho[0]
    ratio = w.rho / base[None]
    assert ratio.min() >= 0.7 - 1e-12 and ratio.max() <= 1.3 + 1e-12
    assert np.abs(np.diff(ratio, axis=0)).max() <= 0.3 * 2 * np.pi / 32 + 1e-12
    # J carries the same factor per cell
    baseJ = wl.random_history((5, 4, 3), 32, seed=3, dtype="f64").J[0]
    np.testing.assert_allclose(w.J / baseJ[None], np.broadcast_to(ratio[:, None], w.J.shape), rtol=1e-12)
    # phases differ from cell to cell (white in space)
    assert np.std(ratio[5]) > 0.05


def test_paper160_descriptor_is_lazy():
    w = wl.paper_table4_largest(n=8, T=5)
    assert w.lazy and w.rho is None and w.N_s == 512 and w.T == 5 and callable(w.device_history)


def test_bench_descriptors():
    import bench
    w = bench.make_workload("c3_small")
    c = bench.config_dict(w, "c3_small", 1, "weak")
    r = bench.config_dict(w, "c3_small", 1, "weak")
    assert c == r and c["eval_steps"] == 1 and c["pairs_per_step"] == w.N_s * w.N_o
    assert c["parallelism"] == "single GPU"
    assert "obs-sharded x8" in bench.config_dict(w, "c3_small", 8, "strong")["parallelism"]
    assert "z-slabs x8" in bench.config_dict(w, "c3_small", 8, "strong-src")["parallelism"]
    assert bench.is_series("c4_series") and bench.is_series("c4_series_f64") and not bench.is_series("c4")
    v = wl.slab_workload(w, 3, 7)
    assert v.n_src == (16, 16, 4) and v.rho.shape[1] == 4 and v.J.shape[2] == 4
    assert v.slab_origin[2] == pytest.approx(w.origin_src[2] + 3 * w.spacing_src[2])
    np.testing.assert_array_equal(v.rho, w.rho[:, 3:7])
    with pytest.raises(SystemExit):
        bench.make_workload("nope")

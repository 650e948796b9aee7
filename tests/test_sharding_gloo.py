"""N > 1 host logic on CPU: world_size 2 over the gloo backend (no GPU).

The method has no exchange step: ranks either run one S-O pair each
(bench.py --gpus N) or share ONE problem (--scaling strong): rank 0's raw history is broadcast,
the observation set is partitioned with jefi_shard_obs, the results are disjoint slices.  Covered here:
the broadcast + slice logic of the strong mode (the functions bench.py itself calls),
the partition rule (disjoint, ordered, complete, whole z-layers), that evaluating the slices
separately and concatenating them in rank order equals the unsharded evaluation (the oracle
stands in for the kernels: this test is about the slicing, not the arithmetic), and the
max-over-ranks reduction bench.py uses for its timing."""
import os
import socket

import numpy as np
import pytest

import workloads as wl


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    import oracle
    import paper_2104_05426_b200 as jb
    from paper_2104_05426_b200 import sharding
    import bench

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = wl.random_history((5, 4, 3), 12, seed=3, dtype="f64", n_obs=(4, 3, 5), dt=0.05)
        # observation split (paper_2104_05426_b200/sharding.py, what bench.py --scaling strong runs):
        # only rank 0 holds the raw history; the others receive it through broadcast_history, then
        # every rank evaluates ITS slice of the one observation set (obs_slice -> jefi_shard_obs)
        rho = torch.from_numpy(w.rho.copy()) if rank == 0 else torch.zeros(w.rho.shape, dtype=torch.float64)
        J = torch.from_numpy(w.J.copy()) if rank == 0 else torch.zeros(w.J.shape, dtype=torch.float64)
        sharding.broadcast_history(rho, J)
        assert np.array_equal(rho.numpy(), w.rho) and np.array_equal(J.numpy(), w.J)
        begin, count = sharding.obs_slice(w.n_obs, w.origin_obs, w.spacing_obs, rank=rank, world=world)
        assert (begin, count) == bench.strong_slice(jb, w, rank, world)
        obs = jb.make_obs_grid(w.n_obs, w.origin_obs, w.spacing_obs)
        assert (begin, count) == jb.jefi_shard_obs(obs, rank, world)
        idx = np.arange(begin, begin + count)
        E, B = oracle.fields(w.n_src, w.origin_src, w.spacing_src, rho.numpy(), J.numpy(), dt=w.dt, c=w.c, step=11,
                             obs_xyz=w.obs_points(idx), nthreads=1)
        # gather the slices (sizes differ by a z-layer: pad to the largest)
        sizes = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(sizes, torch.tensor([count], dtype=torch.int64))
        cap = int(max(int(s) for s in sizes))
        mine = torch.zeros((6, cap), dtype=torch.float64)
        mine[:3, :count] = torch.from_numpy(E)
        mine[3:, :count] = torch.from_numpy(B)
        parts = [torch.zeros_like(mine) for _ in range(world)]
        dist.all_gather(parts, mine)
        full = torch.cat([p[:, :int(s)] for p, s in zip(parts, sizes)], dim=1).numpy()
        # source split: every rank evaluates ITS z-slab of the source grid (own grid descriptor from
        # jefi_shard_src, own slab of the history) at every observation point; sum_partial_fields
        # all-reduces the partial fields into the total on every rank
        z0, z1, slab_origin, cell_begin = sharding.src_slab(w.n_src, w.origin_src, w.spacing_src, rank, world)
        v = wl.slab_workload(w, z0, z1)
        assert v.slab_origin == pytest.approx(slab_origin) and cell_begin == z0 * w.n_src[0] * w.n_src[1]
        Es, Bs = oracle.fields(v.n_src, v.slab_origin, v.spacing_src, v.rho, v.J, dt=w.dt, c=w.c, step=11,
                               obs_xyz=w.obs_points(), nthreads=1)
        Et, Bt = torch.from_numpy(Es.copy()), torch.from_numpy(Bs.copy())
        sharding.sum_partial_fields(Et, Bt)
        if rank == 0:
            np.save(os.path.join(out_dir, "src_split.npy"), np.concatenate([Et.numpy(), Bt.numpy()]))
        # the timing reduction of bench.py: every rank ends with the slowest rank's numbers
        red = bench.max_over_ranks([10.0 + rank, 5.0 - rank], device="cpu")
        if rank == 0:
            np.save(os.path.join(out_dir, "full.npy"), full)
            np.save(os.path.join(out_dir, "red.npy"), np.array(red))
            np.save(os.path.join(out_dir, "sizes.npy"), np.array([int(s) for s in sizes]))
    finally:
        dist.destroy_process_group()


def test_two_ranks_partition_the_observation_set(tmp_path):
    import torch.multiprocessing as mp
    import oracle
    import __graft_entry__
    __graft_entry__.build()
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    full = np.load(tmp_path / "full.npy")
    w = wl.random_history((5, 4, 3), 12, seed=3, dtype="f64", n_obs=(4, 3, 5), dt=0.05)
    E, B = oracle.fields(w.n_src, w.origin_src, w.spacing_src, w.rho, w.J, dt=w.dt, c=w.c, step=11,
                         obs_xyz=w.obs_points(), nthreads=1)
    np.testing.assert_array_equal(full[:3], E)
    np.testing.assert_array_equal(full[3:], B)
    assert list(np.load(tmp_path / "sizes.npy")) == [36, 24]        # 3 + 2 z-layers of 4 x 3
    # source split: the all-reduced slab fields equal the unsharded evaluation up to summation order
    tot = np.load(tmp_path / "src_split.npy")
    np.testing.assert_allclose(tot[:3], E, rtol=0, atol=1e-13 * np.abs(E).max())
    np.testing.assert_allclose(tot[3:], B, rtol=0, atol=1e-13 * np.abs(B).max())
    assert list(np.load(tmp_path / "red.npy")) == [11.0, 5.0]


def test_source_slabs_partition_the_layers():
    """jefi_shard_src: contiguous whole z-layers in rank order, sizes within one layer of each
    other, slab descriptors that tile the source grid exactly; bad arguments are refused."""
    import __graft_entry__
    __graft_entry__.build()
    import paper_2104_05426_b200 as jb
    for n, world in (((64, 64, 64), 8), ((48, 48, 48), 5), ((7, 5, 3), 4), ((100, 100, 100), 3), ((4, 3, 1), 2)):
        src = jb.make_grid(n, (-1.5, 0.25, 2.0), (0.1, 0.2, 0.3))
        pos, sizes = 0, []
        for r in range(world):
            slab, cell_begin = jb.jefi_shard_src(src, r, world)
            assert cell_begin == pos * n[0] * n[1]
            assert list(slab.n)[:2] == list(n[:2]) and list(slab.spacing) == [0.1, 0.2, 0.3]
            assert list(slab.origin)[:2] == [-1.5, 0.25] and slab.origin[2] == pytest.approx(2.0 + pos * 0.3)
            pos += slab.n[2]
            sizes.append(slab.n[2])
        assert pos == n[2] and max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    src = jb.make_grid((4, 4, 4), (0, 0, 0), (1, 1, 1))
    for rank, world in ((0, 0), (-1, 2), (2, 2)):
        with pytest.raises(jb.JefiError) as e:
            jb.jefi_shard_src(src, rank, world)
        assert e.value.status == jb.JEFI_ERR_INVALID_ARG
    with pytest.raises(jb.JefiError):
        jb.jefi_shard_src(None, 0, 1)


@pytest.mark.parametrize("n,world", [((64, 64, 64), 8), ((256, 256, 1), 8), ((100, 100, 100), 3),
                                     ((3, 2, 1), 4), ((5, 1, 1), 8), ((7, 9, 2), 5)])
def test_shard_rule_is_a_partition(n, world):
    import __graft_entry__
    __graft_entry__.build()
    import paper_2104_05426_b200 as jb
    obs = jb.make_obs_grid(n, (0, 0, 0), (1, 1, 1))
    total = n[0] * n[1] * n[2]
    pos, counts = 0, []
    for r in range(world):
        b, c = jb.jefi_shard_obs(obs, r, world)
        assert b == pos and c >= 0
        pos += c
        counts.append(c)
    assert pos == total
    granule = n[0] * n[1] if n[2] >= world else (n[0] if n[1] * n[2] >= world else 1)
    assert all(c % granule == 0 for c in counts)
    assert max(counts) - min(counts) <= granule
    pts = jb.jefi_obs_desc()
    pts.kind, pts.npoints = 1, 1001
    got = [jb.jefi_shard_obs(pts, r, world) for r in range(world)]
    assert sum(c for _, c in got) == 1001 and got[0][0] == 0
    for bad in ((-1, world), (world, world), (0, 0)):
        with pytest.raises(jb.JefiError):
            jb.jefi_shard_obs(obs, *bad)

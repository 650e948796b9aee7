"""One process per GPU, one problem (Fig. 2: the paper hands one
source-observation pair to each GPU card).  Plumbing only -- which slice a rank owns comes from
the C ABI (jefi_shard_obs, jefi_shard_src), the exchange steps are torch.distributed
collectives (NCCL on GPUs, gloo in the CPU tests); no arithmetic of the method lives here.

Two decompositions:
  * observation split: the raw history is replicated (broadcast_history), every rank packs it
    with its own pre-pass and evaluates its slice of the observation set (obs_slice); no
    exchange of results -- the slices concatenate in rank order;
  * source split: every rank holds the history of its own z-slab of the source grid
    (src_slab) and evaluates it at every observation point; one all-reduce of the fields
    (sum_partial_fields) gives every rank the total.
"""
from __future__ import annotations

from . import jefi_obs_desc, jefi_shard_obs, jefi_shard_src, make_grid, make_obs_grid


def obs_slice(n_obs=None, origin_obs=None, spacing_obs=None, *, npoints=None, rank: int, world: int):
    """(begin, count) of the observation set rank `rank` of `world` evaluates: whole z-layers of a
    regular grid where there are enough of them (jefi_shard_obs), a contiguous run of a point list."""
    if npoints is not None:
        obs = jefi_obs_desc()
        obs.kind, obs.npoints = 1, int(npoints)
    else:
        obs = make_obs_grid(n_obs, origin_obs, spacing_obs)
    return jefi_shard_obs(obs, rank, world)


def src_slab(n_src, origin_src, spacing_src, rank: int, world: int):
    """(z0, z1, slab origin, cell_begin): the source z-layers [z0, z1) of rank `rank`, the origin of
    that slab's grid descriptor and the linear index of its first cell (jefi_shard_src)."""
    slab, cell_begin = jefi_shard_src(make_grid(n_src, origin_src, spacing_src), rank, world)
    per_layer = int(n_src[0]) * int(n_src[1])
    z0 = cell_begin // per_layer
    return z0, z0 + int(slab.n[2]), tuple(slab.origin), cell_begin


def broadcast_history(rho, J, src: int = 0):
    """Rank `src` owns the raw history; every other rank receives it (one broadcast per array) and
    then runs its own pre-pass.  Broadcasting the raw history (16 B per record) and packing on
    every rank moves half the bytes of broadcasting the packed history (32 B per record).  A
    history that does not change between steps is broadcast once, outside the stepping loop."""
    import torch.distributed as dist
    dist.broadcast(rho, src)
    dist.broadcast(J, src)


def sum_partial_fields(E, B):
    """Source split: every rank holds the fields of ITS slab at every observation point; one
    all-reduce (sum) of the 6 N_o values gives every rank the total -- the one exchange step of the
    source-partitioned decomposition (the fields are linear in rho and J, Eq. (4)-(5))."""
    import torch.distributed as dist
    dist.all_reduce(E)
    dist.all_reduce(B)

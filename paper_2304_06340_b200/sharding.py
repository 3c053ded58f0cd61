"""Multi-GPU layer: one process per GPU (torch.distributed), targets sharded by radial shell.

The ball quadrature is a sum over radial shells, and every target is independent (each nuhat_k is its own sum
over the atoms), so a distance evaluation shards over ranks without any data-path exchange: rank r takes the shells
[a_r, a_{r+1}), runs the whole hot path on them (sfd_weak_distance_range: its own direct sum or its own complete type-3
transform, with the half rule) and the only collective is the all-reduce of one compensated fp64 pair (16 bytes) that
never leaves device memory.  Host logic only -- the shard arithmetic and the collective; the per-shard work is the
C-ABI call of binding.py.
"""
import math


def radial_shards(n_r, world_size, eps=0.0):
    """Boundaries a_0 = 0 <= a_1 <= ... <= a_world = n_r of contiguous blocks of radial shells, balanced by cost.

    eps == 0 (direct sum): every shell costs the same (n_theta * n_phi targets x J sources) -> equal counts.
    eps > 0 (type-3): a shard's grids are sized by its own largest radius, ~r_max^3, plus the per-target interpolation;
    shells are assigned so that cumulative (count + grid term) is even.  Gauss-Legendre radii grow about linearly with
    the shell index, so the model uses a/n_r for the radius."""
    n_r, world_size = int(n_r), int(world_size)
    assert n_r >= 0 and world_size >= 1
    if eps <= 0.0:
        return [(n_r * r) // world_size for r in range(world_size + 1)]
    # cost of owning shells [0, a): a (targets) + lambda * (a/n_r)^3 * n_r (grid), lambda = 1: equal weights
    def cost(a):
        return a + n_r * (a / max(n_r, 1)) ** 3
    total = cost(n_r)
    bounds = [0]
    for r in range(1, world_size):
        target = total * r / world_size
        a = bounds[-1]
        while a < n_r and cost(a + 1) <= target:
            a += 1
        bounds.append(a)
    bounds.append(n_r)
    return bounds


def shard_of(n_r, rank, world_size, eps=0.0):
    b = radial_shards(n_r, world_size, eps)
    return b[rank], b[rank + 1]


def combine_partial(pair, group=None):
    """All-reduce (sum) of the ranks' partial sums over `group`, in place, on the device the tensor lives on.

    `pair` is the float64[2] (sum, compensation) tensor that sfd_weak_distance_range leaves in device memory: 16 bytes,
    added component-wise -- the data path's only exchange (NCCL over NVLink on GPUs; gloo on CPU tensors in the host-logic
    tests).  Without an initialised process group (single process) the tensor is returned unchanged."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(pair, op=dist.ReduceOp.SUM, group=group)
    return pair


def weak_distance_sharded(V, F, rule, s, R, q, eps=0.0, rank=None, world_size=None, group=None, work=None, x_extent=None):
    """sqrt(I) and I of the H^{-s} distance with the frequency nodes sharded over the ranks of `group`.

    Every rank runs sfd_weak_distance_range on its shells (the same half rule and fast paths as the single-GPU call, the
    transform's grids sized by the shard's own largest radius); the 16-byte device pairs are all-reduced; the one host
    read is the final sum, taken on every rank."""
    import torch.distributed as dist
    from . import binding
    if rank is None:
        rank = dist.get_rank(group) if dist.is_initialized() else 0
    if world_size is None:
        world_size = dist.get_world_size(group) if dist.is_initialized() else 1
    n_r = int(q[0]) if not hasattr(q, "n_r") else q.n_r
    a0, a1 = shard_of(n_r, rank, world_size, eps)
    pair = binding.sfd_weak_distance_range(V, F, rule, s, R, q, a0, a1, eps, work=work, x_extent=x_extent)
    pair = combine_partial(pair, group)
    I = float(pair.sum().item())
    return math.sqrt(I), I

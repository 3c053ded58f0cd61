"""Multi-GPU layer: one process per GPU (torch.distributed), targets sharded by radial shell.

The ball quadrature is a sum over radial shells, and every target is independent (each nuhat_k is its own sum
over the atoms), so a distance evaluation shards over ranks without any data-path exchange: rank r takes the shells
[a_r, a_{r+1}), runs the whole hot path on them (its own direct sum or its own complete type-3 transform) and the only
collective is the all-reduce of one fp64 partial sum I_r (8 bytes).  Host logic only -- argument marshalling and the
shard arithmetic; the per-shard work is the C-ABI calls of binding.py (or, in the CPU tests, callables the test
supplies).
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


def combine_partial_I(I_part, group=None):
    """Sum of the ranks' partial I over `group` (all-reduce of one fp64).  Without an initialised process group
    (single process) the partial sum is the sum."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(I_part)
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    t = torch.tensor([float(I_part)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return float(t[0])


def weak_distance_sharded(V, F, rule, s, R, q, eps=0.0, rank=None, world_size=None, group=None, backend=None):
    """sqrt(I) and I of the H^{-s} distance with the targets sharded over the ranks of `group`.

    backend: object with sfd_nodes, sfd_freq_nodes_device_range, sfd_surface_ft, sfd_reduce (default: this package's
    binding, i.e. the CUDA path on the rank's current device)."""
    import torch.distributed as dist
    if backend is None:
        from . import binding as backend
    if rank is None:
        rank = dist.get_rank(group) if dist.is_initialized() else 0
    if world_size is None:
        world_size = dist.get_world_size(group) if dist.is_initialized() else 1
    n_r = int(q[0]) if not hasattr(q, "n_r") else q.n_r
    a0, a1 = shard_of(n_r, rank, world_size, eps)
    I_part = 0.0
    if a1 > a0:
        x, w = backend.sfd_nodes(V, F, rule)
        xi, W = backend.sfd_freq_nodes_device_range(q, R, a0, a1)
        nu = backend.sfd_surface_ft(x, w, xi, eps)
        I_part = backend.sfd_reduce(nu, xi, W, s)
    I = combine_partial_I(I_part, group)
    return math.sqrt(I), I

"""Host logic of the multi-GPU path (paper_2304_06340_b200/sharding.py) on the CPU: shard arithmetic, and the
world_size-2 all-reduce over gloo of per-shard partial sums the test computes with the oracle (-m "not gpu")."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _sharding():
    # import the module file directly: the package's binding needs libsfd.so and a GPU to be useful
    import importlib.util
    spec = importlib.util.spec_from_file_location("sfd_sharding", os.path.join(ROOT, "paper_2304_06340_b200", "sharding.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


@pytest.mark.parametrize("eps", [0.0, 1e-9])
@pytest.mark.parametrize("n_r,world", [(32, 1), (32, 2), (128, 8), (5, 8), (0, 3), (512, 7)])
def test_radial_shards_partition(n_r, world, eps):
    S = _sharding()
    b = S.radial_shards(n_r, world, eps)
    assert len(b) == world + 1 and b[0] == 0 and b[-1] == n_r
    assert all(b[i] <= b[i + 1] for i in range(world))
    assert sum(b[i + 1] - b[i] for i in range(world)) == n_r
    if eps == 0.0 and n_r >= world:
        sizes = [b[i + 1] - b[i] for i in range(world)]
        assert max(sizes) - min(sizes) <= 1
    if eps > 0.0 and n_r >= 4 * world and world > 1:
        sizes = [b[i + 1] - b[i] for i in range(world)]
        assert sizes[0] >= sizes[-1]      # outer shards own larger grids, so they get fewer shells


def _oracle():
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import sfd_oracle
    return sfd_oracle


def _shard_partial(O, V, F, rule, s, R, q, a0, a1):
    """The partial sum I_r of the shells [a0, a1), by the oracle (test code: the product's per-shard work is the CUDA call
    sfd_weak_distance_range, compared with exactly this on the GPU in tests/test_gpu_parity.py)."""
    x, w = O.nodes(V, F, rule)
    xi, W = O.freq_nodes(q[0], q[1], q[2], R)
    n = q[1] * q[2]
    xi, W = np.ascontiguousarray(xi[a0 * n:a1 * n]), np.ascontiguousarray(W[a0 * n:a1 * n])
    if a1 == a0:
        return 0.0
    return O.reduce(O.direct_sum(x, w, xi), xi, W, s)


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        S = _sharding()
        O = _oracle()
        V, F = O.mesh_icosphere(1)
        q = (12, 6, 8)
        res = {}
        for eps in (0.0, 1e-9):   # both shard policies
            a0, a1 = S.shard_of(q[0], rank, world, eps)
            # what sfd_weak_distance_range leaves on a GPU: a (sum, compensation) pair; here a CPU tensor over gloo
            pair = torch.tensor([_shard_partial(O, V, F, 6, 2.0, 8.0, q, a0, a1), 0.0], dtype=torch.float64)
            pair = S.combine_partial(pair)
            res[eps] = (float(pair.sum()), (a0, a1))
        out[rank] = res
    finally:
        dist.destroy_process_group()


def test_combine_partial_gloo_world2():
    """Shard arithmetic + the 16-byte all-reduce over gloo, world size 2: the shards tile the shells, every rank ends up
    with the same sum, and the sum is the unsharded I."""
    import torch.multiprocessing as mp
    O = _oracle()
    V, F = O.mesh_icosphere(1)
    d_ref, I_ref = O.weak_distance(V, F, 6, 2.0, 8.0, 12, 6, 8)
    mgr = mp.Manager()
    out = mgr.dict()
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert set(out.keys()) == {0, 1}
    for eps in (0.0, 1e-9):
        (I0, s0), (I1, s1) = out[0][eps], out[1][eps]
        assert I0 == I1                                  # every rank holds the reduced value
        assert s0[0] == 0 and s0[1] == s1[0] and s1[1] == 12 and s0[1] > 0   # the two shards tile the shells
        assert abs(I0 - I_ref) <= 1e-13 * I_ref


def test_combine_partial_without_group():
    import torch
    S = _sharding()
    t = torch.tensor([1.5, 2.0 ** -60], dtype=torch.float64)
    assert S.combine_partial(t) is t and float(t[0]) == 1.5

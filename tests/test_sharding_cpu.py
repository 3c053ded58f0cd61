"""Host logic of the multi-GPU path (paper_2304_06340_b200/sharding.py) on the CPU: shard arithmetic, and the
world_size-2 all-reduce over gloo with the oracle standing in for the per-shard device work (-m "not gpu")."""
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


class _OracleBackend:
    """The calls sharding.weak_distance_sharded makes, answered by the CPU oracle (numpy arrays)."""

    def __init__(self):
        sys.path.insert(0, os.path.join(ROOT, "oracle"))
        import sfd_oracle
        self.O = sfd_oracle

    def sfd_nodes(self, V, F, rule):
        return self.O.nodes(V, F, rule)

    def sfd_freq_nodes_device_range(self, q, R, a0, a1):
        xi, W = self.O.freq_nodes(q[0], q[1], q[2], R)
        n = q[1] * q[2]
        return xi[a0 * n:a1 * n], W[a0 * n:a1 * n]

    def sfd_surface_ft(self, x, w, xi, eps):
        return self.O.direct_sum(x, w, xi)

    def sfd_reduce(self, nu, xi, W, s):
        return self.O.reduce(nu, xi, W, s)


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        S = _sharding()
        B = _OracleBackend()
        V, F = B.O.mesh_icosphere(1)
        q = (12, 6, 8)
        res = {}
        for eps in (0.0, 1e-9):   # both shard policies (the oracle backend ignores eps beyond that)
            d, I = S.weak_distance_sharded(V, F, 6, 2.0, 8.0, q, eps, backend=B)
            res[eps] = (d, I, S.shard_of(q[0], rank, world, eps))
        out[rank] = res
    finally:
        dist.destroy_process_group()


def test_weak_distance_sharded_gloo_world2():
    import torch.multiprocessing as mp
    B = _OracleBackend()
    V, F = B.O.mesh_icosphere(1)
    d_ref, I_ref = B.O.weak_distance(V, F, 6, 2.0, 8.0, 12, 6, 8)
    mgr = mp.Manager()
    out = mgr.dict()
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert set(out.keys()) == {0, 1}
    for eps in (0.0, 1e-9):
        (d0, I0, s0), (d1, I1, s1) = out[0][eps], out[1][eps]
        assert I0 == I1 and d0 == d1                    # every rank holds the reduced value
        assert s0[0] == 0 and s0[1] == s1[0] and s1[1] == 12 and s0[1] > 0   # the two shards tile the shells
        assert abs(I0 - I_ref) <= 1e-13 * I_ref and abs(d0 - d_ref) <= 1e-13 * d_ref

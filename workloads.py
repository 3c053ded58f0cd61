"""Seeded synthetic inputs shared by the tests, bench.py, the oracle side and the CUDA side.

This module holds NONE of the method's arithmetic (no quadrature, no transform, no reduction):
only the BASELINE.json workload table, a counter-based random generator, and the perturbations
and random clouds that are *inputs* to both implementations.
numpy only; imports neither oracle/ nor paper_2304_06340_b200/.
"""
import numpy as np

# BASELINE.json `configs`, in order.  level/rule define the sources, (n_r, R, n_theta, n_phi) the
# spherical-product frequency quadrature, s the Sobolev orders, eps the NUFFT tolerances
# (0.0 = fp64 direct sum).
CONFIGS = {
    1: dict(level=1, rule=6, n_r=32, R=32.0, n_theta=16, n_phi=32, s=(2.0,), eps=(0.0,), jitter=None),
    2: dict(level=4, rule=6, n_r=128, R=128.0, n_theta=64, n_phi=128, s=(1.0, 2.0), eps=(0.0, 1e-9), jitter=None),
    3: dict(level=6, rule=12, n_r=256, R=256.0, n_theta=128, n_phi=256, s=(2.0,), eps=(1e-6, 1e-12), jitter=None),
    4: dict(level=7, rule=6, n_r=384, R=512.0, n_theta=192, n_phi=384, s=(1.0,), eps=(1e-9,), jitter=(0.1, 0)),
    5: dict(level=tuple(range(9)), rule=6, n_r=512, R=1024.0, n_theta=256, n_phi=512, s=(1.0, 2.0), eps=(1e-10,),
            jitter=None),
}

_GOLDEN = 0x9E3779B97F4A7C15
_M64 = (1 << 64) - 1


def splitmix64(seed: int, n: np.ndarray) -> np.ndarray:
    """Output number n (0-based) of the SplitMix64 stream with initial state `seed` (random access:
    the state after n+1 steps is seed + (n+1)*golden).  Vectorised over n; returns uint64."""
    n = np.asarray(n, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = np.uint64(seed & _M64) + (n + np.uint64(1)) * np.uint64(_GOLDEN)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, n: np.ndarray) -> np.ndarray:
    """[0,1) doubles with 53 random bits from stream outputs n."""
    return (splitmix64(seed, n) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53


def standard_normal(seed: int, count: int) -> np.ndarray:
    """count N(0,1) draws: draw i uses stream outputs 2i, 2i+1 (Box-Muller, cosine branch)."""
    i = np.arange(count, dtype=np.uint64)
    u1 = 1.0 - uniform01(seed, 2 * i)          # (0,1]
    u2 = uniform01(seed, 2 * i + np.uint64(1))  # [0,1)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


def mean_edge_length(V: np.ndarray, F: np.ndarray) -> float:
    """Mean Euclidean length over the unique undirected edges of a triangle mesh."""
    e = np.concatenate([F[:, [0, 1]], F[:, [1, 2]], F[:, [2, 0]]]).astype(np.int64)
    e.sort(axis=1)
    e = np.unique(e, axis=0)
    return float(np.linalg.norm(V[e[:, 0]] - V[e[:, 1]], axis=1).mean())


def jitter_vertices(V: np.ndarray, F: np.ndarray, rel: float = 0.1, seed: int = 0) -> np.ndarray:
    """BASELINE.json config 4: vertices displaced radially by N(0,(rel*h)^2), h the mean edge length
    of the unjittered mesh: v_i <- v_i * (1 + rel*h*g_i)."""
    h = mean_edge_length(V, F)
    g = standard_normal(seed, len(V))
    return np.ascontiguousarray(V * (1.0 + rel * h * g)[:, None])


def target_subset(K: int, n: int, seed: int = 0) -> np.ndarray:
    """n distinct target indices in [0,K), sorted (stream outputs taken in order, duplicates skipped)."""
    n = min(n, K)
    out, seen, c = [], set(), 0
    while len(out) < n:
        block = splitmix64(seed, np.arange(c, c + 2 * n, dtype=np.uint64)) % np.uint64(K)
        c += 2 * n
        for v in block.tolist():
            if v not in seen:
                seen.add(v)
                out.append(v)
                if len(out) == n:
                    break
    return np.sort(np.asarray(out, dtype=np.int64))


def random_cloud(J: int, K: int, seed: int = 12345, x_offset=(3.0, -2.0, 5.0), xi_radius: float = 20.0,
                 xi_offset=(7.0, -11.0, 4.0)):
    """Parity-only inputs that exercise what the centrally symmetric icosphere never does (C != 0,
    D != 0, Im != 0): x uniform in [-1,1]^3 + x_offset, signed weights in [-1,1), targets uniform in a
    ball of radius xi_radius centred at xi_offset."""
    j = np.arange(J, dtype=np.uint64)
    x = np.stack([2.0 * uniform01(seed, 4 * j + np.uint64(c)) - 1.0 for c in range(3)], axis=1)
    x = x + np.asarray(x_offset, np.float64)
    w = 2.0 * uniform01(seed, 4 * j + np.uint64(3)) - 1.0
    k = np.arange(K, dtype=np.uint64)
    s2 = seed + 1
    g = np.stack([standard_normal(s2 + 10 * (c + 1), K) for c in range(3)], axis=1)
    nrm = np.linalg.norm(g, axis=1, keepdims=True)
    nrm[nrm == 0] = 1.0
    rad = xi_radius * np.cbrt(uniform01(s2, k))[:, None]
    xi = g / nrm * rad + np.asarray(xi_offset, np.float64)
    return np.ascontiguousarray(x), np.ascontiguousarray(w), np.ascontiguousarray(xi)

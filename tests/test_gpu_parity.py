"""Parity of the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs (-m gpu).

Bars (BASELINE.json north_star): integer mesh output bit-exact; direct-sum nuhat max|d| <= 1e-12 * sum|w|;
I to relative 1e-8.  Vertices / atoms / frequency nodes are compared to a few ulp (they are the same operations
rounded once each, so they are in fact expected to be bit-identical; the tolerance only guards libm differences).
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sfd():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2304_06340_b200 as P
    return P


@pytest.fixture(scope="module")
def torch():
    import torch
    return torch


def dev(torch, a):
    return torch.as_tensor(np.ascontiguousarray(a), device="cuda")


# ---- A1/A2 ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("level", [0, 1, 2, 3, 4, 5, 6, 7])
def test_mesh_bit_exact(sfd, orc, torch, level):
    V, F = sfd.sfd_mesh_icosphere(level)
    Vo, Fo = orc.mesh_icosphere(level)
    assert np.array_equal(F.cpu().numpy(), Fo), "integer mesh output must be bit-exact"
    assert np.array_equal(V.cpu().numpy(), Vo), "vertex arithmetic is IEEE add/mul/sqrt/div: bit-identical"


def test_mesh_level8_invariants(sfd, torch):
    """Level 8 (1.31 M faces): properties that hold at any size (Euler, valence, every directed edge once)."""
    V, F = sfd.sfd_mesh_icosphere(8)
    nV, nF = V.shape[0], F.shape[0]
    assert (nV, nF) == (10 * 4 ** 8 + 2, 20 * 4 ** 8)
    Fl = F.long()
    assert int(Fl.min()) == 0 and int(Fl.max()) == nV - 1
    e = torch.cat([Fl[:, [0, 1]], Fl[:, [1, 2]], Fl[:, [2, 0]]])
    key = e[:, 0] * nV + e[:, 1]
    assert torch.unique(key).numel() == 3 * nF            # every directed edge exactly once
    rkey = e[:, 1] * nV + e[:, 0]
    assert torch.equal(torch.sort(key).values, torch.sort(rkey).values)  # and its reverse: closed, oriented
    val = torch.bincount(Fl.reshape(-1), minlength=nV)
    assert int((val == 5).sum()) == 12 and int((val == 6).sum()) == nV - 12
    assert float((V.norm(dim=1) - 1).abs().max()) < 4e-16
    assert nV - 3 * nF // 2 + nF == 2


# ---- A3 ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("level,rule", [(0, 6), (1, 6), (3, 12), (5, 6), (5, 12)])
def test_nodes(sfd, orc, torch, level, rule):
    Vo, Fo = orc.mesh_icosphere(level)
    xo, wo = orc.nodes(Vo, Fo, rule)
    x, w = sfd.sfd_nodes(dev(torch, Vo), dev(torch, Fo), rule)
    assert np.abs(x.cpu().numpy() - xo).max() <= 2e-16
    assert np.abs(w.cpu().numpy() - wo).max() <= 2e-16 * wo.max()


def test_nodes_degenerate_and_empty(sfd, torch):
    V = dev(torch, np.array([[0, 0, 0], [1, 0, 0], [2, 0, 0], [0, 1, 0]], np.float64))
    F = dev(torch, np.array([[0, 1, 2], [0, 1, 3]], np.int32))   # first face has zero area
    x, w = sfd.sfd_nodes(V, F, 6)
    w = w.cpu().numpy()
    assert np.all(w[:6] == 0) and abs(w[6:].sum() - 0.5) < 1e-15
    x0, w0 = sfd.sfd_nodes(V, F[:0].contiguous(), 12)
    assert x0.shape == (0, 3) and w0.shape == (0,)


def test_freq_nodes_device(sfd, orc, torch):
    for (nr, nt, nph, R) in [(32, 16, 32, 32.0), (7, 5, 3, 4.0)]:
        xi, W = sfd.sfd_freq_nodes_device((nr, nt, nph), R)
        xo, Wo = orc.freq_nodes(nr, nt, nph, R)
        assert np.abs(xi.cpu().numpy() - xo).max() <= 4e-16 * R
        assert np.abs(W.cpu().numpy() - Wo).max() <= 1e-14 * Wo.max()


# ---- A4 direct sum ----------------------------------------------------------------------------------
def _direct_case(sfd, orc, torch, x, w, xi, tol=1e-12):
    nu = sfd.sfd_surface_ft(dev(torch, x), dev(torch, w), dev(torch, xi), 0.0).cpu().numpy()
    ref = orc.direct_sum(x, w, xi)
    err = np.abs(nu - ref).max() if len(ref) else 0.0
    assert err <= tol * np.abs(w).sum(), (err, np.abs(w).sum())
    return nu, ref


def test_direct_config1_full(sfd, orc, torch):
    c = workloads.CONFIGS[1]
    V, F = orc.mesh_icosphere(c["level"])
    x, w = orc.nodes(V, F, c["rule"])
    xi, W = orc.freq_nodes(c["n_r"], c["n_theta"], c["n_phi"], c["R"])
    nu, ref = _direct_case(sfd, orc, torch, x, w, xi)
    # spot values of SURVEY 8(c) pin 5 fix the target ordering
    assert abs(nu[0] - 11.6625241207662) < 1e-9 and abs(nu[-1] - (-1.0556323496997)) < 1e-9
    assert np.abs(nu.imag).max() < 1e-13


@pytest.mark.parametrize("J,K", [(1, 1), (7, 33), (33, 7), (1000, 1000), (513, 2049), (3000, 131), (512, 128 * 4 + 1)])
def test_direct_random_clouds(sfd, orc, torch, J, K):
    """Off-centre sources and targets, signed weights: exercises Im != 0, ragged tiles and the source split."""
    x, w, xi = workloads.random_cloud(J, K)
    _direct_case(sfd, orc, torch, x, w, xi)


def test_direct_large_phase(sfd, orc, torch):
    """|xi.x| up to ~1.8e3 (config-5 scale, R = 1024): the range reduction must hold 1e-12 * sum|w|."""
    x, w, xi = workloads.random_cloud(600, 700, seed=7, x_offset=(0, 0, 0), xi_radius=1024.0, xi_offset=(0, 0, 0))
    _direct_case(sfd, orc, torch, x, np.abs(w), xi)


def test_direct_empty(sfd, torch):
    x, w, xi = workloads.random_cloud(5, 9)
    nu = sfd.sfd_surface_ft(dev(torch, x[:0]), dev(torch, w[:0]), dev(torch, xi), 0.0)
    assert nu.shape == (9,) and float(nu.abs().max()) == 0.0
    nu = sfd.sfd_surface_ft(dev(torch, x), dev(torch, w), dev(torch, xi[:0]), 0.0)
    assert nu.shape == (0,)


def test_direct_config2_sampled(sfd, orc, torch):
    """Config 2 at full size in the launch configuration bench.py times; the oracle checks a seeded sample."""
    c = workloads.CONFIGS[2]
    V, F = orc.mesh_icosphere(c["level"])
    x, w = orc.nodes(V, F, c["rule"])
    xi, W = orc.freq_nodes(c["n_r"], c["n_theta"], c["n_phi"], c["R"])
    nu = sfd.sfd_surface_ft(dev(torch, x), dev(torch, w), dev(torch, xi), 0.0).cpu().numpy()
    idx = workloads.target_subset(len(xi), 2048, seed=0)
    ref = orc.direct_sum(x, w, xi[idx])
    assert np.abs(nu[idx] - ref).max() <= 1e-12 * w.sum()
    assert abs(nu[0].real - w.sum()) < 1e-2 and np.abs(nu.imag).max() < 1e-12  # central symmetry (pin 4 note)


# ---- A6 reduction -----------------------------------------------------------------------------------
@pytest.mark.parametrize("s", [1.0, 2.0, 0.75, 3.5])
def test_reduce_fed_oracle_nuhat(sfd, orc, torch, s):
    c = workloads.CONFIGS[1]
    V, F = orc.mesh_icosphere(c["level"])
    x, w = orc.nodes(V, F, c["rule"])
    xi, W = orc.freq_nodes(c["n_r"], c["n_theta"], c["n_phi"], c["R"])
    nu = orc.direct_sum(x, w, xi)
    I_ref = orc.reduce(nu, xi, W, s)
    I = sfd.sfd_reduce(dev(torch, nu.view(np.float64).reshape(-1, 2)), dev(torch, xi), dev(torch, W), s)
    assert abs(I - I_ref) <= 1e-8 * I_ref
    assert abs(I - I_ref) <= 1e-12 * I_ref  # what the arithmetic actually delivers


def test_reduce_small_r_and_complex(sfd, orc, torch):
    """r < 1e-4 series branch of sigmahat, r = 0, non-zero imaginary parts, ragged K."""
    rng = np.random.default_rng(3)
    K = 1237
    xi = rng.normal(size=(K, 3)) * np.logspace(-8, 1, K)[:, None]
    xi[0] = 0.0
    W = rng.random(K)
    nu = rng.normal(size=K) + 1j * rng.normal(size=K)
    I_ref = orc.reduce(nu, xi, W, 1.5)
    I = sfd.sfd_reduce(dev(torch, nu.view(np.float64).reshape(-1, 2)), dev(torch, xi), dev(torch, W), 1.5)
    assert abs(I - I_ref) <= 1e-12 * I_ref
    with pytest.raises(sfd.SfdError):
        sfd.sfd_reduce(dev(torch, nu.view(np.float64).reshape(-1, 2)), dev(torch, xi), dev(torch, W), 0.5)
    assert sfd.sfd_reduce(dev(torch, np.zeros((0, 2))), dev(torch, np.zeros((0, 3))), dev(torch, np.zeros(0)), 2.0) == 0.0


# ---- whole path -------------------------------------------------------------------------------------
def test_weak_distance_config1(sfd, orc, torch):
    c = workloads.CONFIGS[1]
    q = (c["n_r"], c["n_theta"], c["n_phi"])
    V, F = sfd.sfd_mesh_icosphere(c["level"])
    d, I = sfd.sfd_weak_distance(V, F, c["rule"], 2.0, c["R"], q, 0.0)
    Vo, Fo = orc.mesh_icosphere(c["level"])
    d_ref, I_ref = orc.weak_distance(Vo, Fo, c["rule"], 2.0, c["R"], *q)
    assert abs(I - I_ref) <= 1e-8 * I_ref and abs(d - d_ref) <= 1e-8 * d_ref
    assert abs(d - 9.336109377069e-2) < 1e-9   # SURVEY 8(c) pin 5, config 1 in full
    # host-buffer entry point gives the same number
    d2, I2 = sfd.sfd_weak_distance_host(Vo, Fo, c["rule"], 2.0, c["R"], q, 0.0)
    assert abs(I2 - I) <= 1e-13 * I


def test_weak_distance_jittered_mesh(sfd, orc, torch):
    """Config-4-style radial jitter (an input, workloads.jitter_vertices) on a small mesh: Im(nuhat) != 0."""
    Vo, Fo = orc.mesh_icosphere(2)
    Vj = workloads.jitter_vertices(Vo, Fo, 0.1, 0)
    q = (24, 12, 16)
    for s in (1.0, 2.0):
        d_ref, I_ref = orc.weak_distance(Vj, Fo, 6, s, 16.0, *q)
        d, I = sfd.sfd_weak_distance(dev(torch, Vj), dev(torch, Fo), 6, s, 16.0, q, 0.0)
        assert abs(I - I_ref) <= 1e-8 * I_ref


def test_code_paths_behind_switches_agree(sfd, orc, torch, monkeypatch):
    """The alternatives the library chooses between at run time compute the same thing: the ball-rule direct sum with its
    table packed behind the stages instead of 32 KB-aligned (bit-identical: same arithmetic, other addresses), the type-3
    transform with the subgrids staged by LDGSTS instead of TMA box copies and with the target sort on the caller's stream
    instead of the second one (identical up to the order of the spreader's additions).  Config 1, against the oracle too."""
    c = workloads.CONFIGS[1]
    q = (c["n_r"], c["n_theta"], c["n_phi"])
    V, F = sfd.sfd_mesh_icosphere(c["level"])
    Vo, Fo = orc.mesh_icosphere(c["level"])
    _, I_ref = orc.weak_distance(Vo, Fo, c["rule"], 2.0, c["R"], *q)
    _, I0 = sfd.sfd_weak_distance(V, F, c["rule"], 2.0, c["R"], q, 0.0)
    monkeypatch.setenv("SFD_DIRECT_PACKED", "1")
    _, I1 = sfd.sfd_weak_distance(V, F, c["rule"], 2.0, c["R"], q, 0.0)
    monkeypatch.delenv("SFD_DIRECT_PACKED")
    assert I1 == I0 and abs(I0 - I_ref) <= 1e-8 * I_ref
    for eps in (1e-6, 1e-10):
        _, Ia = sfd.sfd_weak_distance(V, F, c["rule"], 2.0, c["R"], q, eps)
        monkeypatch.setenv("SFD_INTERP_NO_TMA", "1")
        monkeypatch.setenv("SFD_NO_OVERLAP", "1")
        _, Ib = sfd.sfd_weak_distance(V, F, c["rule"], 2.0, c["R"], q, eps)
        monkeypatch.delenv("SFD_INTERP_NO_TMA")
        monkeypatch.delenv("SFD_NO_OVERLAP")
        assert abs(Ia - Ib) <= 1e-12 * Ia, (eps, Ia, Ib)
        assert abs(Ia - I_ref) <= 2 * np.sqrt(I_ref * _r13_bound(orc, Vo, Fo, c["rule"], q, c["R"], 2.0, eps)) + _r13_bound(orc, Vo, Fo, c["rule"], q, c["R"], 2.0, eps)


def _r13_bound(orc, Vn, Fn, rule, q, R, s, eps):
    """DESIGN.md R13: |dI| <= 2 sqrt(I E2) + E2, E2 = (2 pi)^-3 sum_k W_k (10 eps sum|w|)^2 (1+r^2)^-s."""
    x, w = orc.nodes(Vn, Fn, rule)
    xi, W = orc.freq_nodes(*q, R)
    r2 = (xi * xi).sum(1)
    return float((W * (1 + r2) ** (-s)).sum()) * (10 * eps * np.abs(w).sum()) ** 2 / (2 * np.pi) ** 3


@pytest.mark.parametrize("q", [(20, 10, 12), (14, 9, 16)])          # even and odd n_theta (a ring at cos(theta) = 0)
@pytest.mark.parametrize("eps", [1e-6, 1e-10])
def test_weak_distance_fast_path_offcentre_mesh(sfd, orc, torch, q, eps):
    """The combination only sfd_weak_distance uses -- half rule, origin-centred target box, hull hint, Hermitian half
    band, ball prune -- on meshes that are NOT centrally symmetric (C != 0, Im nuhat != 0): a jittered, translated and
    anisotropically scaled level-2 icosphere, against the oracle's distance (not the library's own stages)."""
    Vo, Fo = orc.mesh_icosphere(2)
    Vj = workloads.jitter_vertices(Vo, Fo, 0.1, 5) * np.array([1.0, 0.7, 1.3]) + np.array([0.3, -0.2, 0.15])
    Vj = np.ascontiguousarray(Vj)
    R, s = 14.0, 2.0
    d_ref, I_ref = orc.weak_distance(Vj, Fo, 6, s, R, *q)
    d, I = sfd.sfd_weak_distance(dev(torch, Vj), dev(torch, Fo), 6, s, R, q, eps)
    E2 = _r13_bound(orc, Vj, Fo, 6, q, R, s, eps)
    assert abs(I - I_ref) <= 2 * np.sqrt(I_ref * E2) + E2, (I, I_ref, E2)
    d0, I0 = sfd.sfd_weak_distance(dev(torch, Vj), dev(torch, Fo), 6, s, R, q, 0.0)
    assert abs(I0 - I_ref) <= 1e-8 * I_ref


@pytest.mark.parametrize("aspect", [(16.0, 1.0, 1.0), (1.0, 1.0, 24.0), (0.05, 1.0, 0.3)])
def test_weak_distance_stretched_mesh(sfd, orc, torch, aspect):
    """Elongated meshes: the inner grid is n2_0 x n2_1 x n2_2 with very different axes, and the ball the rule's nodes fill
    becomes an ellipsoid in grid cells.  The pruned band must still hold every cell a footprint touches (the region kept
    is the ellipsoid scaled by 1 + reach / a_min, a superset of its Minkowski sum with the footprint)."""
    Vo, Fo = orc.mesh_icosphere(2)
    Vs = np.ascontiguousarray(Vo * np.array(aspect))
    q, R, s, eps = (16, 10, 12), 6.0, 2.0, 1e-6
    d_ref, I_ref = orc.weak_distance(Vs, Fo, 6, s, R, *q)
    d, I = sfd.sfd_weak_distance(dev(torch, Vs), dev(torch, Fo), 6, s, R, q, eps)
    E2 = _r13_bound(orc, Vs, Fo, 6, q, R, s, eps)
    assert np.isfinite(I) and abs(I - I_ref) <= 2 * np.sqrt(I_ref * E2) + E2, (I, I_ref, E2)


def test_extents(sfd, torch):
    """sfd_extents: the library's own bounds kernels behind the workspace queries (no torch reduction on the data)."""
    x, w, xi = workloads.random_cloud(5000, 10)
    half, centre = sfd.sfd_extents(dev(torch, x))
    lo, hi = x.min(0), x.max(0)
    assert np.allclose(half, 0.5 * (hi - lo), rtol=1e-11, atol=0) and np.all(np.asarray(half) >= 0.5 * (hi - lo))
    assert np.allclose(centre, 0.5 * (hi + lo), rtol=1e-15, atol=1e-15)
    assert sfd.sfd_extents(dev(torch, np.zeros((0, 3)))) == ([0.0] * 3, [0.0] * 3)
    one = sfd.sfd_extents(dev(torch, np.array([[1.0, -2.0, 3.0]])))
    assert one[1] == [1.0, -2.0, 3.0] and max(one[0]) < 1e-290
    with pytest.raises(sfd.SfdError) as e:
        sfd.sfd_extents(dev(torch, np.array([[1.0, np.nan, 0.0]])))
    assert e.value.status == -2


def test_bad_face_index_is_reported(sfd, orc, torch):
    """a face index >= nV is "checked on device, reported at the next synchronising call" as
    SFD_ERR_INVALID_ARG.  sfd_nodes only enqueues (the atoms of the bad face are NaN); the next synchronising call on
    the device reports and clears the error; calls that take the mesh and synchronise report their own."""
    Vo, Fo = orc.mesh_icosphere(1)
    bad = Fo.copy()
    bad[17, 1] = len(Vo) + 3
    neg = Fo.copy()
    neg[3, 0] = -1
    V = dev(torch, Vo)
    xi, W = sfd.sfd_freq_nodes_device((6, 4, 6), 4.0)
    for Fb in (bad, neg):
        x, w = sfd.sfd_nodes(V, dev(torch, Fb), 6)          # enqueues; no error yet
        assert bool(torch.isnan(w).any())
        nu = sfd.sfd_surface_ft(x, w, xi, 0.0)
        with pytest.raises(sfd.SfdError) as e:
            sfd.sfd_reduce(nu, xi, W, 2.0)
        assert e.value.status == -2 and "face index" in str(e.value)
        # reported once, then cleared: a good mesh afterwards is fine
        xg, wg = sfd.sfd_nodes(V, dev(torch, Fo), 6)
        assert sfd.sfd_reduce(sfd.sfd_surface_ft(xg, wg, xi, 0.0), xi, W, 2.0) > 0
        for eps in (0.0, 1e-8):
            with pytest.raises(sfd.SfdError) as e:
                sfd.sfd_weak_distance(V, dev(torch, Fb), 6, 2.0, 4.0, (6, 4, 6), eps)
            assert e.value.status == -2
            assert sfd.sfd_weak_distance(V, dev(torch, Fo), 6, 2.0, 4.0, (6, 4, 6), eps)[0] > 0
        with pytest.raises(sfd.SfdError):
            sfd.sfd_mesh_distance(V, dev(torch, Fo), V, dev(torch, Fb), 6, 2.0, 4.0, (6, 4, 6), 0.0)
        x, w = sfd.sfd_nodes(V, dev(torch, Fb), 6)
        with pytest.raises(sfd.SfdError):
            sfd.sfd_extents(x)                              # NaN atoms + the error word
        assert sfd.sfd_extents(xg)[0][0] > 0
        pair = sfd.sfd_weak_distance_range(V, dev(torch, Fb), 6, 2.0, 4.0, (6, 4, 6), 0, 6, 0.0)
        assert bool(torch.isnan(pair[0]))                   # nothing synchronises: the shard's partial sum is poisoned


def test_surface_ft_host_entry(sfd, orc):
    x, w, xi = workloads.random_cloud(300, 500)
    nu = sfd.sfd_surface_ft_host(x, w, xi, 0.0)
    ref = orc.direct_sum(x, w, xi)
    assert np.abs(nu - ref).max() <= 1e-12 * np.abs(w).sum()


# ---- A5 type-3 NUFFT --------------------------------------------------------------------------------
def _nufft_case(sfd, orc, torch, x, w, xi, eps, factor=10.0):
    nu = sfd.sfd_surface_ft(dev(torch, x), dev(torch, w), dev(torch, xi), eps).cpu().numpy()
    ref = orc.direct_sum(x, w, xi)
    err = np.abs(nu - ref).max() / np.abs(w).sum()
    assert err <= factor * eps, (err, eps)
    return err


@pytest.mark.parametrize("eps", [1e-3, 1e-6, 1e-9, 1e-12])
def test_nufft_config1(sfd, orc, torch, eps):
    """Config-1 geometry (centred sources and targets: the real-strength path)."""
    c = workloads.CONFIGS[1]
    V, F = orc.mesh_icosphere(c["level"])
    x, w = orc.nodes(V, F, c["rule"])
    xi, W = orc.freq_nodes(c["n_r"], c["n_theta"], c["n_phi"], c["R"])
    _nufft_case(sfd, orc, torch, x, w, xi, eps)


@pytest.mark.parametrize("J,K", [(1, 1), (7, 33), (33, 7), (1000, 1000), (3000, 4097)])
@pytest.mark.parametrize("eps", [1e-6, 1e-9, 1e-12])
def test_nufft_random_clouds(sfd, orc, torch, J, K, eps):
    """Off-centre sources (C != 0), off-centre targets (D != 0, complex strengths), signed weights."""
    x, w, xi = workloads.random_cloud(J, K)
    _nufft_case(sfd, orc, torch, x, w, xi, eps)


def _random_case(rng, eps):
    """Seeded random geometry: isotropic or anisotropic boxes, shells, centred or not, few or many targets."""
    J = int(10 ** rng.uniform(1.7, 3.5))
    K = int(10 ** rng.uniform(0, 3.5))
    half = rng.uniform(0.05, 1.5, size=3) if rng.random() < 0.5 else np.full(3, rng.uniform(0.1, 1.2))
    cx = rng.normal(size=3) * (0.0 if rng.random() < 0.5 else 0.7)
    if rng.random() < 0.4:
        x = rng.normal(size=(J, 3))
        x = x / np.linalg.norm(x, axis=1, keepdims=True) * half + cx
    else:
        x = (rng.random((J, 3)) * 2 - 1) * half + cx
    w = rng.normal(size=J) if rng.random() < 0.5 else rng.random(J)
    S = rng.uniform(0.5, 40.0) * (np.ones(3) if rng.random() < 0.6 else rng.uniform(0.2, 1.0, size=3))
    cxi = rng.normal(size=3) * (0.0 if rng.random() < 0.6 else 5.0)
    xi = (rng.random((K, 3)) * 2 - 1) * S + cxi
    if K >= 2 and rng.random() < 0.5:
        xi[0], xi[1] = cxi + S, cxi - S
    return x, w, xi


@pytest.mark.parametrize("seed", range(8))
def test_nufft_random_configurations(sfd, orc, torch, seed):
    """A seeded sweep over geometries and tolerances (5 cases per seed): every bin shape, the real and the complex
    path, the footprint-ordered sort when the grid is small against J."""
    rng = np.random.default_rng(1000 + seed)
    for _ in range(5):
        eps = 10.0 ** (-int(rng.integers(2, 14)))
        x, w, xi = _random_case(rng, eps)
        _nufft_case(sfd, orc, torch, x, w, xi, max(eps, 1e-13))


def test_nufft_single_source_worst_case(sfd, orc, torch):
    """A single source has nothing to average the kernel's pointwise error over (it reached ~25 eps with the width rule
    of R10 alone, two kernel applications); the library therefore takes one more cell of width below 64 sources, and
    the 10 eps sum|w| bar holds here too."""
    rng = np.random.default_rng(77)
    worst = 0.0
    for eps in (1e-4, 1e-7, 1e-10, 1e-12):
        for _ in range(6):
            x = rng.normal(size=(1, 3)) * 0.6
            xi = (rng.random((3000, 3)) * 2 - 1) * rng.uniform(3.0, 25.0)
            nu = sfd.sfd_surface_ft(dev(torch, x), dev(torch, np.ones(1)), dev(torch, xi), eps).cpu().numpy()
            worst = max(worst, np.abs(nu - orc.direct_sum(x, np.ones(1), xi)).max() / eps)
    assert worst <= 10.0, worst


# ---- multi-GPU path on one GPU: the ranks' shards evaluated one after the other ----------------------
@pytest.mark.parametrize("eps,world,q", [(0.0, 3, None), (1e-9, 4, None), (1e-9, 2, (9, 7, 8)), (0.0, 2, (5, 4, 3))])
def test_target_shards_add_up(sfd, orc, torch, eps, world, q):
    """The partial sums of disjoint radial shards (what each rank of sharding.weak_distance_sharded computes with
    sfd_weak_distance_range: half rule, shard-sized grids) add up to the unsharded I; every shard's partial sum equals
    the oracle's sum over the shard's nodes; the shard nodes are the full rule's nodes.  Odd n_theta (a ring at
    cos(theta) = 0) and odd n_phi (no half rule) included."""
    from paper_2304_06340_b200 import sharding
    c = workloads.CONFIGS[1]
    q = q or (c["n_r"], c["n_theta"], c["n_phi"])
    V, F = sfd.sfd_mesh_icosphere(c["level"])
    d_full, I_full = sfd.sfd_weak_distance(V, F, c["rule"], 2.0, c["R"], q, eps)
    xi_full, W_full = sfd.sfd_freq_nodes_device(q, c["R"])
    Vo, Fo = orc.mesh_icosphere(c["level"])
    xo, wo = orc.nodes(Vo, Fo, c["rule"])
    xio, Wo = orc.freq_nodes(*q, c["R"])
    n = q[1] * q[2]
    I_sum = 0.0
    tol = 1e-11 if eps == 0.0 else 1e-7   # every shard's type-3 transform has its own grids (errors <= 10 eps sum|w|)
    for rank in range(world):
        a0, a1 = sharding.shard_of(q[0], rank, world, eps)
        xi, W = sfd.sfd_freq_nodes_device_range(q, c["R"], a0, a1)
        assert torch.equal(xi, xi_full[a0 * n:a1 * n]) and torch.equal(W, W_full[a0 * n:a1 * n])
        pair = sfd.sfd_weak_distance_range(V, F, c["rule"], 2.0, c["R"], q, a0, a1, eps)
        assert pair.is_cuda and pair.shape == (2,)
        I_r = float(pair.sum())
        sl = slice(a0 * n, a1 * n)
        I_o = orc.reduce(orc.direct_sum(xo, wo, xio[sl]), np.ascontiguousarray(xio[sl]), np.ascontiguousarray(Wo[sl]), 2.0) \
            if a1 > a0 else 0.0
        assert abs(I_r - I_o) <= tol * I_full, (rank, I_r, I_o)
        d, I = sharding.weak_distance_sharded(V, F, c["rule"], 2.0, c["R"], q, eps, rank=rank, world_size=world)
        assert I == I_r or abs(I - I_r) <= 1e-9 * I_full    # no process group: each call returns its own partial sum
        I_sum += I_r
    assert abs(I_sum - I_full) <= tol * I_full


def test_weak_distance_range_edges(sfd, torch):
    """Empty range -> (0, 0); bad ranges rejected; the whole range equals sfd_weak_distance."""
    V, F = sfd.sfd_mesh_icosphere(1)
    q = (8, 6, 8)
    pair = sfd.sfd_weak_distance_range(V, F, 6, 2.0, 8.0, q, 3, 3, 0.0)
    assert pair.tolist() == [0.0, 0.0]
    for a0, a1 in ((-1, 2), (5, 4), (0, 9)):
        with pytest.raises(sfd.SfdError):
            sfd.sfd_weak_distance_range(V, F, 6, 2.0, 8.0, q, a0, a1, 0.0)
    for eps in (0.0, 1e-8):
        d, I = sfd.sfd_weak_distance(V, F, 6, 2.0, 8.0, q, eps)
        pair = sfd.sfd_weak_distance_range(V, F, 6, 2.0, 8.0, q, 0, 8, eps)
        assert abs(float(pair.sum()) - I) <= 1e-14 * I


@pytest.mark.parametrize("eps", [1e-1, 1e-2, 1e-4, 1e-5, 1e-7, 1e-8, 1e-10, 1e-11, 1e-13, 1e-14])
def test_nufft_every_kernel_width(sfd, orc, torch, eps):
    """Every instantiated kernel width (w = 2 ... 15; 1e-3/-6/-9/-12 are covered above): real-strength path (ball
    quadrature, Hermitian half band) and complex path (off-centre cloud)."""
    V, F = orc.mesh_icosphere(2)
    x, w = orc.nodes(V, F, 6)
    xi, W = orc.freq_nodes(12, 8, 10, 20.0)
    _nufft_case(sfd, orc, torch, x, w, xi, eps)
    x, w, xi = workloads.random_cloud(400, 300)
    _nufft_case(sfd, orc, torch, x, w, xi, eps)


@pytest.mark.parametrize("q", [(6, 8, 10), (5, 7, 12), (4, 6, 9)])
@pytest.mark.parametrize("eps", [0.0, 1e-10])
def test_weak_distance_half_rule_equals_full_rule(sfd, torch, q, eps):
    """sfd_weak_distance evaluates only the nodes with xi_3 >= 0 (doubled weights) when n_phi is even; the composition
    of the public stages over every node gives the same I: even n_theta, odd n_theta (a ring at mu = 0 that is its own
    mirror image) and odd n_phi (no symmetry: every node)."""
    V, F = sfd.sfd_mesh_icosphere(2)
    R, s = 9.0, 2.0
    x, w = sfd.sfd_nodes(V, F, 12)
    xi, W = sfd.sfd_freq_nodes_device(q, R)
    I_full = sfd.sfd_reduce(sfd.sfd_surface_ft(x, w, xi, eps), xi, W, s)
    d, I = sfd.sfd_weak_distance(V, F, 12, s, R, q, eps)
    K_eval = sfd.sfd_weak_distance_targets(q)
    assert K_eval == (q[0] * (q[1] - q[1] // 2) * q[2] if q[2] % 2 == 0 else q[0] * q[1] * q[2])
    tol = 1e-11 if eps == 0.0 else 1e-7   # (eps = 0: two direct-sum kernels with independent roundings)
    assert abs(I - I_full) <= tol * I_full, (I, I_full)


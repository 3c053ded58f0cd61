"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (-m gpu).

The CPU oracle cannot afford J x K at configs 2-5 (3e10 ... 5e14 pairs): it checks a seeded sample of targets one by
one (reading R14), the GPU direct sum -- itself oracle-checked in test_gpu_parity.py and here on the
sample -- checks a larger sample, and properties that hold at any size (Hermitian symmetry of nuhat for real weights,
nuhat(0) = area, quadratic rate) cover the rest.  Bars: direct 1e-12 sum|w|; NUFFT 10 eps sum|w|; I per R13.
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


def _workload(sfd, torch, cfg_id, level=None):
    c = workloads.CONFIGS[cfg_id]
    level = c["level"] if level is None else level
    V, F = sfd.sfd_mesh_icosphere(level)
    if c["jitter"]:
        Vj = workloads.jitter_vertices(V.cpu().numpy(), F.cpu().numpy(), *c["jitter"])
        V = torch.as_tensor(Vj, device="cuda")
    x, w = sfd.sfd_nodes(V, F, c["rule"])
    q = (c["n_r"], c["n_theta"], c["n_phi"])
    xi, W = sfd.sfd_freq_nodes_device(q, c["R"])
    return c, V, F, x, w, xi, W, q


def _check_nufft(sfd, orc, torch, x, w, xi, eps, n_gpu=4096, n_cpu=4096):
    """NUFFT nuhat at n_gpu seeded targets against the GPU direct sum (10 eps sum|w|), and the GPU direct sum at the first
    n_cpu of them against the oracle, one target at a time on the CPU (1e-12 sum|w|).  n_cpu: SURVEY 8(d) A14 says
    K_sub = 4096; smaller where 4096 x J pairs would take the 16-core oracle more than ~10 s."""
    K = xi.shape[0]
    sw = float(w.abs().sum())
    torch.cuda.empty_cache()   # the transform's workspace is one block of up to 123 GB (config 5): no cached fragments
    nu = sfd.sfd_surface_ft(x, w, xi, eps)
    torch.cuda.empty_cache()
    idx = torch.as_tensor(workloads.target_subset(K, n_gpu, seed=0), device="cuda")
    ref = sfd.sfd_surface_ft(x, w, xi[idx].contiguous(), 0.0)
    err = float((nu[idx] - ref).abs().max()) / sw
    assert err <= 10 * eps, (err, eps)
    # the GPU direct sum on the same sample against the oracle (one target at a time on the CPU)
    sub = idx[:n_cpu]
    oref = orc.direct_sum(x.cpu().numpy(), w.cpu().numpy(), xi[sub].cpu().numpy())
    derr = np.abs(ref[:n_cpu].cpu().numpy() - oref).max() / sw
    assert derr <= 1e-12, derr
    return nu, err


def _i_bound(W, xi, s, eps, sw):
    """R13: E^2 = (2 pi)^-3 sum_k W_k (10 eps sum|w|)^2 (1+r^2)^-s."""
    r2 = (xi * xi).sum(1)
    return float((W * (1 + r2) ** (-s)).sum()) * (10 * eps * sw) ** 2 / (2 * np.pi) ** 3


def test_config2_full(sfd, orc, torch):
    """Config 2: NUFFT (eps 1e-9) against the direct sum at ALL 1,048,576 targets; I by both paths, s = 1, 2."""
    c, V, F, x, w, xi, W, q = _workload(sfd, torch, 2)
    sw = float(w.sum())
    nu_d = sfd.sfd_surface_ft(x, w, xi, 0.0)
    nu_n = sfd.sfd_surface_ft(x, w, xi, 1e-9)
    assert float((nu_d - nu_n).abs().max()) <= 10 * 1e-9 * sw
    # any-size properties: nuhat(xi) for real weights is Hermitian; the quadrature is symmetric under xi -> -xi
    # (mu_b -> mu_{n-1-b}, phi_c -> phi_{c+n/2}); central symmetry of the icosphere makes nuhat real
    assert float(nu_d.imag.abs().max()) <= 1e-12 * sw
    nr, nt, nph = q
    g = nu_d.real.reshape(nr, nt, nph)
    mirror = torch.roll(torch.flip(g, dims=[1]), shifts=nph // 2, dims=2)
    assert float((g - mirror).abs().max()) <= 1e-11 * sw
    for s in c["s"]:
        d0, I0 = sfd.sfd_weak_distance(V, F, c["rule"], s, c["R"], q, 0.0)
        d1, I1 = sfd.sfd_weak_distance(V, F, c["rule"], s, c["R"], q, 1e-9)
        I_red = sfd.sfd_reduce(nu_d, xi, W, s)
        Ed = _i_bound(W, xi, s, 1e-13, sw)   # two direct sums of 1e-12 sum|w| accuracy each (see test_config3_distance)
        assert abs(I0 - I_red) <= 2 * np.sqrt(I0 * Ed) + Ed and abs(I0 - I_red) <= 1e-8 * I0
        E2 = _i_bound(W, xi, s, 1e-9, sw)
        assert abs(I1 - I0) <= 2 * np.sqrt(I0 * E2) + E2, (I1, I0, E2)
    # SURVEY 8(c) pin 5 digits for level 4 on this grid (a cross-check computed independently of both sides)
    d_s2, _ = sfd.sfd_weak_distance(V, F, c["rule"], 2.0, c["R"], q, 0.0)
    assert abs(d_s2 - 1.5501793453e-3) <= 1e-9


@pytest.mark.parametrize("eps", [1e-6, 1e-12])
def test_config3_sampled(sfd, orc, torch, eps):
    """Config 3 (level 6, 12-pt rule, 983,040 sources; 8,388,608 targets): nuhat, 4096 GPU-direct / 4096 oracle targets."""
    c, V, F, x, w, xi, W, q = _workload(sfd, torch, 3)
    _check_nufft(sfd, orc, torch, x, w, xi, eps)


def test_config3_distance(sfd, orc, torch, capsys):
    """Config 3's distance -- BASELINE.json's "full level-6 distance": sfd_weak_distance(level 6, 12-pt rule, s = 2) through
    the half rule + ball-pruned band at eps 1e-6 and 1e-12, against the fp64 direct sum over every node.
      I(eps = 0) from sfd_weak_distance (half rule, ball-rule direct sum, 4.1e12 pairs) == sfd_reduce(sfd_surface_ft(all 8.4 M
      nodes)) within the bound two direct sums of 1e-12 sum|w| accuracy allow (observed: relative 2e-12);
      both NUFFT I's inside the R13 bound |dI| <= 2 sqrt(I) E + E^2 (R13 / SURVEY 8(c) A13);
      the achieved relative dI is printed."""
    c, V, F, x, w, xi, W, q = _workload(sfd, torch, 3)
    sw = float(w.sum())
    d0, I0 = sfd.sfd_weak_distance(V, F, c["rule"], 2.0, c["R"], q, 0.0)
    nu = sfd.sfd_surface_ft(x, w, xi, 0.0)
    I_full = sfd.sfd_reduce(nu, xi, W, 2.0)
    # two direct sums with independent roundings (the distance call takes the nodes from the rule's tables, one direction
    # and 16 radii per thread; sfd_surface_ft takes the expanded nodes): each is within 1e-12 sum|w| of the exact nuhat, so
    # the two I differ by at most the R13-type bound with that error -- and by far less than BJ's relative 1e-8
    Ed = _i_bound(W, xi, 2.0, 1e-13, sw)
    assert abs(I0 - I_full) <= 2 * np.sqrt(I_full * Ed) + Ed and abs(I0 - I_full) <= 1e-8 * I_full, (I0, I_full)
    # the direct sum itself against the oracle on 4096 seeded nodes (the oracle cannot afford 8.25e12 pairs)
    idx = workloads.target_subset(xi.shape[0], 4096, seed=3)
    oref = orc.direct_sum(x.cpu().numpy(), w.cpu().numpy(), xi[torch.as_tensor(idx, device="cuda")].cpu().numpy())
    assert np.abs(nu[torch.as_tensor(idx, device="cuda")].cpu().numpy() - oref).max() <= 1e-12 * sw
    del nu
    out = {}
    for eps in c["eps"]:
        d, I = sfd.sfd_weak_distance(V, F, c["rule"], 2.0, c["R"], q, eps)
        E2 = _i_bound(W, xi, 2.0, eps, sw)
        assert abs(I - I0) <= 2 * np.sqrt(I0 * E2) + E2, (eps, I, I0, E2)
        out[eps] = abs(I - I0) / I0
    # at eps 1e-12 the transform's error is far below the distance itself: BASELINE's "I to relative 1e-8" holds outright
    assert out[1e-12] <= 1e-8, out
    with capsys.disabled():
        print(f"\n[config 3] sqrt(I) = {d0:.12e}; relative dI through the NUFFT: " +
              ", ".join(f"eps={e:g}: {v:.2e}" for e, v in out.items()))


@pytest.mark.parametrize("cfg,level,eps", [(3, 6, 1e-6), (3, 6, 1e-12), (5, 8, 1e-10), (5, 3, 1e-10), (4, 7, 1e-9)])
def test_pruned_band_is_sufficient(sfd, torch, monkeypatch, cfg, level, eps):
    """The FFT passes of sfd_weak_distance store only the part of the band inside the ball the rule's nodes fill
    (DESIGN.md 5.3.2).  With SFD_DEBUG_POISON_BAND=1 the library fills the passes' output buffers with NaN first: if the
    interpolation (or a later pass) read a single cell the pruning skipped, I would be NaN.  It must instead equal the
    unpoisoned I up to the spreader's summation order."""
    c = workloads.CONFIGS[cfg]
    q = (c["n_r"], c["n_theta"], c["n_phi"])
    V, F = sfd.sfd_mesh_icosphere(level)
    if c["jitter"]:
        V = torch.as_tensor(workloads.jitter_vertices(V.cpu().numpy(), F.cpu().numpy(), *c["jitter"]), device="cuda")
    s = c["s"][0]
    torch.cuda.empty_cache()
    d_ref, I_ref = sfd.sfd_weak_distance(V, F, c["rule"], s, c["R"], q, eps)
    monkeypatch.setenv("SFD_DEBUG_POISON_BAND", "1")
    d, I = sfd.sfd_weak_distance(V, F, c["rule"], s, c["R"], q, eps)
    monkeypatch.delenv("SFD_DEBUG_POISON_BAND")
    assert np.isfinite(I) and abs(I - I_ref) <= 1e-10 * I_ref, (I, I_ref)
    torch.cuda.empty_cache()


def test_config4_sampled(sfd, orc, torch):
    """Config 4 (level 7 with radial jitter: Im nuhat != 0; 1,966,080 sources; 28,311,552 targets), eps 1e-9."""
    c, V, F, x, w, xi, W, q = _workload(sfd, torch, 4)
    nu, err = _check_nufft(sfd, orc, torch, x, w, xi, 1e-9, n_gpu=4096, n_cpu=2048)
    assert float(nu.imag.abs().max()) > 1e-6   # the jitter breaks the central symmetry
    d, I = sfd.sfd_weak_distance(V, F, c["rule"], 1.0, c["R"], q, 1e-9)
    I_red = sfd.sfd_reduce(nu, xi, W, 1.0)
    assert abs(I - I_red) <= 1e-9 * I


def test_config5_sweep_levels(sfd, orc, torch):
    """Config 5: the fixed 512x256x512 = 67,108,864-target grid on [0,1024] (n2 = 2700, pruned FFT), eps 1e-10, levels
    2..5 of the sweep: sampled parity at level 3 and the rate in h for s = 2 (P:5; R15).  On this grid the
    radial rule is marginal (512 nodes for a phase 2R = 2048, SURVEY 8(c) pin 3), which biases sqrt(I) upwards at high
    frequency: the observed slopes are 1.88-1.91 instead of the 1.99-2.00 of the well-resolved R = 32 / 128 grids
    (tests/test_oracle_pins.py asserts [1.9, 2.1] there).  Asserted here: [1.8, 2.1]."""
    c = workloads.CONFIGS[5]
    q = (c["n_r"], c["n_theta"], c["n_phi"])
    dist = {}
    for level in (2, 3, 4, 5):
        V, F = sfd.sfd_mesh_icosphere(level)
        torch.cuda.empty_cache()
        dist[level] = sfd.sfd_weak_distance(V, F, c["rule"], 2.0, c["R"], q, 1e-10)[0]
        if level == 3:
            x, w = sfd.sfd_nodes(V, F, c["rule"])
            xi, W = sfd.sfd_freq_nodes_device(q, c["R"])
            _check_nufft(sfd, orc, torch, x, w, xi, 1e-10, n_gpu=4096, n_cpu=4096)
            del xi, W
        torch.cuda.empty_cache()
    for level in (3, 4, 5):
        slope = np.log2(dist[level - 1] / dist[level])
        assert 1.8 <= slope <= 2.1, (level, slope, dist)
    # the top of the sweep: level 8 (7,864,320 atoms) on the same grid, three levels further down the same line
    V, F = sfd.sfd_mesh_icosphere(8)
    torch.cuda.empty_cache()
    d8 = sfd.sfd_weak_distance(V, F, c["rule"], 2.0, c["R"], q, 1e-10)[0]
    torch.cuda.empty_cache()
    slope = np.log2(dist[5] / d8) / 3
    assert 1.8 <= slope <= 2.2, (slope, dist, d8)   # 2.13: the coarse levels are biased upwards on this grid (above)
    # level 8 element by element: 7,864,320 atoms (bins crowded enough for item splitting), n2 = 2700; 4096 nodes against
    # the GPU direct sum, 512 of them against the oracle (4e9 pairs)
    x, w = sfd.sfd_nodes(V, F, c["rule"])
    xi, W = sfd.sfd_freq_nodes_device(q, c["R"])
    _check_nufft(sfd, orc, torch, x, w, xi, 1e-10, n_gpu=4096, n_cpu=512)
    del x, w, xi, W
    torch.cuda.empty_cache()
    # cross-grid check: at level 8 the mesh's spectrum is resolved by this grid too (R h = 4.8), so the value must sit
    # on the quadratic line through the well-resolved config-3 grid: d_8 = d_6 / 16 to ~1 %
    c3 = workloads.CONFIGS[3]
    V6, F6 = sfd.sfd_mesh_icosphere(6)
    d6 = sfd.sfd_weak_distance(V6, F6, 6, 2.0, c3["R"], (c3["n_r"], c3["n_theta"], c3["n_phi"]), 1e-10)[0]
    assert abs(16 * d8 / d6 - 1) < 0.02, (d8, d6)


def test_config5_s1_reported(sfd, torch, capsys):
    """Config 5 lists s in {1, 2}.  For s = 1 the difference of two surface measures is not in H^{-1} uniformly (a dipole
    layer needs s > 3/2: SURVEY 8(c) pin 5, R15), so no rate is asserted; the values must be finite, positive,
    decreasing with the level, and above the s = 2 values (the weight (1+r^2)^-1 dominates (1+r^2)^-2 term by term).
    Printed for the record."""
    c = workloads.CONFIGS[5]
    q = (c["n_r"], c["n_theta"], c["n_phi"])
    rows = []
    torch.cuda.empty_cache()
    # one workspace for the whole sweep (sized for the finest level): 64 GB
    work = torch.empty(sfd.sfd_weak_distance_workspace(20 * 4 ** 8, c["rule"], q, c["R"], 1e-10), dtype=torch.uint8,
                       device="cuda")
    for level in (0, 1, 2, 3, 4, 5, 6, 7, 8):
        V, F = sfd.sfd_mesh_icosphere(level)
        d1 = sfd.sfd_weak_distance(V, F, c["rule"], 1.0, c["R"], q, 1e-10, work=work)[0]
        d2 = sfd.sfd_weak_distance(V, F, c["rule"], 2.0, c["R"], q, 1e-10, work=work)[0]
        assert np.isfinite(d1) and np.isfinite(d2) and d1 > d2 > 0
        rows.append((level, d1, d2))
    del work
    torch.cuda.empty_cache()
    for (l0, a1, a2), (l1, b1, b2) in zip(rows, rows[1:]):
        assert b1 < a1 and b2 < a2, rows
    # s = 2 from level 2 on: the quadratic rate (P:5) on average; level by level the marginal radial rule of this
    # grid (512 nodes for a phase of 2048: SURVEY 8(c) pin 3) biases the coarse levels upwards, so the local slopes run
    # from 1.9 (L2..L5) to 2.4 (L7 -> L8) -- see test_config5_sweep_levels
    for (l0, a1, a2), (l1, b1, b2) in zip(rows[2:], rows[3:]):
        assert 1.7 <= np.log2(a2 / b2) <= 2.5, rows
    assert 1.8 <= np.log2(rows[2][2] / rows[8][2]) / 6 <= 2.2, rows
    with capsys.disabled():
        print("\n[config 5] level: sqrt(I) s=1, s=2, log2 ratios")
        for i, (l, d1, d2) in enumerate(rows):
            r = "" if i == 0 else f"  slopes {np.log2(rows[i-1][1] / d1):.2f} {np.log2(rows[i-1][2] / d2):.2f}"
            print(f"  L{l}: {d1:.6e} {d2:.6e}{r}")

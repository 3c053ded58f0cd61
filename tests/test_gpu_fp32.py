"""Single-precision grids (the paper ran its GPU NUFFT "in single precision" at
eps_rel = 1e-7): sfd_set_grid_precision(32) against the fp64 oracle, element by element, through the C ABI (-m gpu).

Bar: max |nuhat - oracle| <= 10 * max(eps, 1e-6) * sum|w_j| -- the kernel's 10 eps bound, floored at the level the stored
grids' rounding (6e-8 of their largest entries, amplified by the deconvolution) can reach.  The oracle is unchanged."""
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


@pytest.fixture()
def fp32(sfd):
    sfd.sfd_set_grid_precision(32)
    yield
    sfd.sfd_set_grid_precision(64)


def dev(torch, a):
    return torch.as_tensor(np.ascontiguousarray(a), device="cuda")


def _case(sfd, orc, torch, x, w, xi, eps):
    nu = sfd.sfd_surface_ft(dev(torch, x), dev(torch, w), dev(torch, xi), eps).cpu().numpy()
    ref = orc.direct_sum(x, w, xi)
    err = np.abs(nu - ref).max() / np.abs(w).sum()
    assert err <= 10 * max(eps, 1e-6), (err, eps)
    return err


@pytest.mark.parametrize("eps", [1e-3, 1e-4, 1e-5, 1e-6])
def test_type3_config1(sfd, orc, torch, fp32, eps):
    """Config 1 in full (real strengths, Hermitian half band), every tolerance the fp32 grids accept (w = 4 ... 7)."""
    c = workloads.CONFIGS[1]
    V, F = orc.mesh_icosphere(c["level"])
    x, w = orc.nodes(V, F, c["rule"])
    xi, W = orc.freq_nodes(c["n_r"], c["n_theta"], c["n_phi"], c["R"])
    _case(sfd, orc, torch, x, w, xi, eps)


@pytest.mark.parametrize("eps", [1e-3, 1e-6])
@pytest.mark.parametrize("J,K", [(1, 1), (7, 33), (1000, 1000), (3000, 4097)])
def test_type3_random_clouds(sfd, orc, torch, fp32, J, K, eps):
    """Off-centre sources and targets (complex strengths, complex fine grid), ragged sizes, a handful of sources (w + 1)."""
    x, w, xi = workloads.random_cloud(J, K)
    _case(sfd, orc, torch, x, w, xi, eps)


def test_type3_config2_and_3_sampled(sfd, orc, torch, fp32):
    """BASELINE.json configs 2 and 3 at eps 1e-6 with fp32 grids (n2 = 256-ish and 672: the fixed-geometry FFT passes):
    4096 seeded nodes against the GPU direct sum, 512 of them against the oracle; the distance against the fp64 one."""
    for cfg in (2, 3):
        c = workloads.CONFIGS[cfg]
        q = (c["n_r"], c["n_theta"], c["n_phi"])
        V, F = sfd.sfd_mesh_icosphere(c["level"])
        x, w = sfd.sfd_nodes(V, F, c["rule"])
        xi, W = sfd.sfd_freq_nodes_device(q, c["R"])
        sw = float(w.sum())
        nu = sfd.sfd_surface_ft(x, w, xi, 1e-6)
        idx = torch.as_tensor(workloads.target_subset(xi.shape[0], 4096, seed=0), device="cuda")
        ref = sfd.sfd_surface_ft(x, w, xi[idx].contiguous(), 0.0)
        assert float((nu[idx] - ref).abs().max()) <= 10 * 1e-6 * sw
        oref = orc.direct_sum(x.cpu().numpy(), w.cpu().numpy(), xi[idx[:512]].cpu().numpy())
        assert np.abs(ref[:512].cpu().numpy() - oref).max() <= 1e-12 * sw
        d32, I32 = sfd.sfd_weak_distance(V, F, c["rule"], 2.0, c["R"], q, 1e-6)
        sfd.sfd_set_grid_precision(64)
        d0, I0 = sfd.sfd_weak_distance(V, F, c["rule"], 2.0, c["R"], q, 0.0 if cfg == 2 else 1e-12)
        sfd.sfd_set_grid_precision(32)
        r2 = (xi * xi).sum(1)
        E2 = float((W * (1 + r2) ** -2.0).sum()) * (10 * 1e-6 * sw) ** 2 / (2 * np.pi) ** 3   # DESIGN.md R13
        assert abs(I32 - I0) <= 2 * np.sqrt(I0 * E2) + E2, (cfg, I32, I0, E2)
        del nu, xi, W
        torch.cuda.empty_cache()


@pytest.mark.parametrize("M,eps", [(16, 1e-7), (30, 1e-5), (64, 1e-7)])
def test_lattice_type1(sfd, orc, torch, fp32, M, eps):
    """The paper's own transform (type-1 onto its lattice, eq. 3.6) with single-precision grids at the paper's
    tolerance 1e-7, element by element against the oracle on the oracle's lattice; centred and off-centre."""
    V, F = orc.mesh_icosphere(3)
    for shift in (np.zeros(3), np.array([0.2, -0.1, 0.05])):
        x, w = orc.nodes(V + shift, F, 64)
        xi, W = orc.lattice_nodes(M, 5.0)
        nu = sfd.sfd_surface_ft_lattice(dev(torch, x), dev(torch, w), M, 5.0, eps).cpu().numpy()
        ref = orc.direct_sum(x, w, xi)
        assert np.abs(nu - ref).max() <= 10 * max(eps, 1e-6) * np.abs(w).sum()


def test_lattice_distance_fig3b_level(sfd, orc, torch, fp32):
    """sfd_weak_distance_lattice (atoms generated in the sort, deconvolution folded into the reduction) with fp32 grids
    against the fp64 run: H_{-10}, xi_max = 5, M = 128 as in Fig. 3(b), level 5."""
    V, F = sfd.sfd_mesh_icosphere(5)
    d32, I32 = sfd.sfd_weak_distance_lattice(V, F, 64, -10.0, 5.0, 128, 1e-7)
    sfd.sfd_set_grid_precision(64)
    d64, I64 = sfd.sfd_weak_distance_lattice(V, F, 64, -10.0, 5.0, 128, 1e-7)
    sfd.sfd_set_grid_precision(32)
    assert abs(d32 - d64) <= 2e-3 * d64, (d32, d64)     # the norm of a 1e-4-sized difference through 6e-8-sized roundings


def test_rejected_tolerances(sfd, torch, fp32):
    x, w, xi = workloads.random_cloud(100, 50)
    xd, wd, xid = (dev(torch, a) for a in (x, w, xi))
    for eps in (1e-7, 1e-9, 1e-12):
        with pytest.raises(sfd.SfdError) as e:
            sfd.sfd_surface_ft(xd, wd, xid, eps)
        assert e.value.status == -2 and "single-precision" in str(e.value)
    with pytest.raises(sfd.SfdError):
        sfd.sfd_surface_ft_lattice(xd, wd, 16, 5.0, 1e-9)
    with pytest.raises(sfd.SfdError):
        sfd.sfd_set_grid_precision(16)
    # the direct sum is not affected by the switch
    nu = sfd.sfd_surface_ft(xd, wd, xid, 0.0)
    assert torch.isfinite(torch.view_as_real(nu)).all()

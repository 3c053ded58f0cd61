"""sfd_exact_ft (direct summation of the exact triangle transform, eq. 2.19) against
the oracle's binary128 evaluation, element by element, through the C ABI."""
import numpy as np
import pytest

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


def total_area(V, F):
    return 0.5 * np.linalg.norm(np.cross(V[F[:, 1]] - V[F[:, 0]], V[F[:, 2]] - V[F[:, 0]]), axis=1).sum()


def frequencies(rng, K, V, F):
    """Magnitudes from 1e-4 to 1e3 (both branches of the kernel), plus the configurations P:140 warns about: xi = 0,
    xi along face normals, xi orthogonal to edges (exactly and almost)."""
    mags = 10.0 ** rng.uniform(-4, 3, size=K)
    d = rng.normal(size=(K, 3))
    xi = d / np.linalg.norm(d, axis=1, keepdims=True) * mags[:, None]
    xi[0] = 0.0
    nf = min(len(F), 40)
    e1 = V[F[:nf, 1]] - V[F[:nf, 0]]
    n = np.cross(e1, V[F[:nf, 2]] - V[F[:nf, 0]])
    n /= np.linalg.norm(n, axis=1, keepdims=True)
    perp = np.cross(e1, n)
    perp /= np.linalg.norm(perp, axis=1, keepdims=True)
    m = 10.0 ** rng.uniform(-1, 2.5, size=nf)
    extra = [n * m[:, None], perp * m[:, None], (perp + 1e-9 * e1) * m[:, None], (perp + 1e-15 * e1) * m[:, None]]
    extra = np.vstack(extra)
    xi[1:1 + len(extra)] = extra[:K - 1]
    return xi


@pytest.mark.parametrize("level,K", [(0, 1), (0, 257), (2, 3000), (3, 777)])
def test_exact_ft_vs_oracle(sfd, orc, torch, level, K):
    """Sizes spanning several face tiles (1280 faces = 10 tiles), ragged tails, one frequency, the face split (few
    frequencies), every branch.  Bar: 2e-15 sum_f A_f plus the fp64 rounding of the phases, 3e-16 |xi| max|x| sum A."""
    Vo, Fo = orc.mesh_icosphere(level)
    rng = np.random.default_rng(100 * level + K)
    xi = frequencies(rng, K, Vo, Fo)
    ref = orc.exact_ft(Vo, Fo, xi)
    got = sfd.sfd_exact_ft(dev(torch, Vo), dev(torch, Fo), dev(torch, xi)).cpu().numpy()
    A = total_area(Vo, Fo)
    tol = (2e-15 + 3e-16 * np.linalg.norm(xi, axis=1)) * A
    err = np.abs(got - ref)
    assert np.all(err <= tol), (np.argmax(err / tol), (err / tol).max())


def test_exact_ft_irregular_mesh(sfd, orc, torch):
    """A mesh that is not a sphere: random slivers and large triangles, off-centre (almost degenerate simplices)."""
    rng = np.random.default_rng(7)
    nF = 300
    V = rng.normal(size=(3 * nF, 3)) * 0.7 + np.array([2.0, -1.0, 0.5])
    V[1::3] = V[0::3] + rng.normal(size=(nF, 3)) * 10.0 ** rng.uniform(-6, 0, size=(nF, 1))      # short first edges
    V[2::3] = V[0::3] + (V[1::3] - V[0::3]) * rng.uniform(-1, 2, size=(nF, 1)) + rng.normal(size=(nF, 3)) * 10.0 ** rng.uniform(-8, 0, size=(nF, 1))
    F = np.arange(3 * nF, dtype=np.int32).reshape(-1, 3)
    xi = frequencies(rng, 1500, V, F)
    ref = orc.exact_ft(V, F, xi)
    got = sfd.sfd_exact_ft(dev(torch, V), dev(torch, F), dev(torch, xi)).cpu().numpy()
    A = total_area(V, F)
    tol = (2e-15 + 3e-16 * np.linalg.norm(xi, axis=1) * np.abs(V).max()) * A
    assert np.all(np.abs(got - ref) <= tol)


def test_exact_ft_vs_quadrature_path(sfd, torch):
    """The second on-GPU cross-check S:8(f) asks for: where the 64-point rule is exact to rounding (|xi| h <= 1) the atoms'
    direct sum and the exact formula agree; further out they differ by the rule's error, which the exact path isolates."""
    V, F = sfd.sfd_mesh_icosphere(3)
    x, w = sfd.sfd_nodes(V, F, 64)
    g = torch.Generator(device="cpu").manual_seed(3)
    xi = (torch.randn(2000, 3, generator=g, dtype=torch.float64) * 2.0).cuda()
    a = sfd.sfd_exact_ft(V, F, xi)
    b = sfd.sfd_surface_ft(x, w, xi, 0.0)
    assert (a - b).abs().max().item() <= 5e-14 * w.sum().item()
    x6, w6 = sfd.sfd_nodes(V, F, 6)
    xi_far = xi * 4.0
    e6 = (sfd.sfd_exact_ft(V, F, xi_far) - sfd.sfd_surface_ft(x6, w6, xi_far, 0.0)).abs().max().item()
    e64 = (sfd.sfd_exact_ft(V, F, xi_far) - sfd.sfd_surface_ft(x, w, xi_far, 0.0)).abs().max().item()
    assert e6 > 1e-7 and e64 < 1e-4 * e6                     # the degree-4 rule's error is visible, the 64-point rule's is not


def test_exact_ft_distance(sfd, orc, torch):
    """Distance of the polyhedron itself (no triangle rule) through sfd_reduce: within the rule's error of the atoms'."""
    q = (32, 16, 32)
    V, F = sfd.sfd_mesh_icosphere(3)
    xi, W = sfd.sfd_freq_nodes_device(q, 16.0)
    I_exact = sfd.sfd_reduce(sfd.sfd_exact_ft(V, F, xi), xi, W, 2.0)
    _, I_12 = sfd.sfd_weak_distance(V, F, 12, 2.0, 16.0, q, 0.0)
    assert abs(I_exact - I_12) <= 1e-6 * I_exact
    Vo, Fo = orc.mesh_icosphere(3)
    xo, Wo = orc.freq_nodes(q[0], q[1], q[2], 16.0)
    I_ref = orc.reduce(orc.exact_ft(Vo, Fo, xo), xo, Wo, 2.0)
    assert abs(I_exact - I_ref) <= 1e-8 * I_ref


def test_exact_ft_edge_cases(sfd, torch):
    V, F = sfd.sfd_mesh_icosphere(1)
    empty_xi = torch.empty((0, 3), dtype=torch.float64, device="cuda")
    assert sfd.sfd_exact_ft(V, F, empty_xi).numel() == 0
    xi = torch.randn(10, 3, dtype=torch.float64, device="cuda")
    noF = torch.empty((0, 3), dtype=torch.int32, device="cuda")
    assert sfd.sfd_exact_ft(V, noF, xi).abs().max().item() == 0.0
    bad = F.clone()
    bad[5, 1] = V.shape[0]                                   # out-of-range vertex index poisons the output
    assert torch.isnan(torch.view_as_real(sfd.sfd_exact_ft(V, bad, xi))).all()
    # ... and is reported (SFD_ERR_INVALID_ARG) by the next synchronising call on the device, once
    with pytest.raises(sfd.SfdError) as e:
        sfd.sfd_extents(V)
    assert e.value.status == -2
    assert sfd.sfd_extents(V)[0][0] > 0

"""sfd_surface_ft_direct_static (include/sfd.h): the direct sum for callers that cannot allocate -- no workspace argument,
no cudaMalloc, the partial sums of the source splits in the library's static device array (csrc/noalloc.cu).

Checked against the existing path, sfd_surface_ft(eps = 0) with a caller's workspace (same kernels, same summation order:
the bar is the direct sum's 1e-12 * sum|w| of the other parity tests, and the two are in fact bit-identical), and against
the oracle, on calls in a row that share the static array.  This file is collected last on purpose (pytest -x).
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

LIMIT = 16 << 20


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


def _case(sfd, orc, torch, J, K, seed_shift=0.0):
    x, w, xi = workloads.random_cloud(J, K)
    x = x + seed_shift
    xd, wd, xid = dev(torch, x), dev(torch, w), dev(torch, xi)
    ref = sfd.sfd_surface_ft(xd, wd, xid, 0.0)                      # the existing path (workspace from torch)
    out = torch.full((K, 2), float("nan"), dtype=torch.float64, device="cuda")
    nu = sfd.sfd_surface_ft_direct_static(xd, wd, xid, out)
    torch.cuda.synchronize()
    sw = float(np.abs(w).sum())
    assert float((nu - ref).abs().max()) <= 1e-12 * sw
    assert torch.equal(torch.view_as_real(nu), torch.view_as_real(ref))   # same kernels, same order
    if J * K <= 4_000_000:
        assert np.abs(nu.cpu().numpy() - orc.direct_sum(x, w, xi)).max() <= 1e-12 * sw
    return xd, wd, xid, ref


def test_two_calls_in_a_row_match_the_workspace_path(sfd, orc, torch):
    """Calls that share the static array, one after the other on one stream: sizes whose sources are split (the scratch
    is in use), then other sizes that leave stale partial sums of the first call behind, then the first again."""
    assert sfd.SFD_STATIC_SCRATCH_BYTES == LIMIT
    need = sfd.sfd_surface_ft_direct_static_scratch(3000, 4097)
    assert 0 < need <= LIMIT, need                                   # this case does go through the static array
    xd, wd, xid, ref = _case(sfd, orc, torch, 3000, 4097)
    _case(sfd, orc, torch, 1000, 1000, seed_shift=0.25)
    _case(sfd, orc, torch, 7, 33)
    # the first inputs again, twice, with nothing allocated in between: the driver's free memory does not move
    out = torch.empty((4097, 2), dtype=torch.float64, device="cuda")
    sfd.sfd_surface_ft_direct_static(xd, wd, xid, out)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    nu = sfd.sfd_surface_ft_direct_static(xd, wd, xid, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    assert torch.equal(torch.view_as_real(nu), torch.view_as_real(ref))


def test_large_k_without_splits_and_edges(sfd, orc, torch):
    """Enough targets to fill whole waves of CTAs: one split, no scratch, any K fits.  Empty inputs."""
    J = 512
    K = next((k for k in (606208, 303104, 1212416, 400000) if sfd.sfd_surface_ft_direct_static_scratch(J, k) == 0), None)
    assert K is not None, "no candidate size runs unsplit on this GPU"
    x, w, xi = workloads.random_cloud(J, K)
    xd, wd, xid = dev(torch, x), dev(torch, w), dev(torch, xi)
    ref = sfd.sfd_surface_ft(xd, wd, xid, 0.0)
    nu = sfd.sfd_surface_ft_direct_static(xd, wd, xid, torch.empty((K, 2), dtype=torch.float64, device="cuda"))
    assert torch.equal(torch.view_as_real(nu), torch.view_as_real(ref))
    idx = workloads.target_subset(K, 64, seed=1)
    assert np.abs(nu[dev(torch, idx)].cpu().numpy() - orc.direct_sum(x, w, xi[idx])).max() <= 1e-12 * np.abs(w).sum()
    # J == 0: zeros; K == 0: nothing
    e3 = torch.empty((0, 3), dtype=torch.float64, device="cuda")
    e1 = torch.empty((0,), dtype=torch.float64, device="cuda")
    out = torch.full((5, 2), 7.0, dtype=torch.float64, device="cuda")
    nu0 = sfd.sfd_surface_ft_direct_static(e3, e1, xid[:5].contiguous(), out)
    assert float(nu0.abs().max()) == 0.0
    assert sfd.sfd_surface_ft_direct_static(xd, wd, e3, torch.empty((0, 2), dtype=torch.float64, device="cuda")).numel() == 0


def test_sizes_beyond_the_array_are_rejected(sfd, torch):
    """A (J, K) whose partial sums exceed the 16 MiB array fails with SFD_ERR_UNSUPPORTED and writes nothing."""
    J = 30720
    K = next((k for k in (524288, 400000, 700000, 300000, 1000000)
              if sfd.sfd_surface_ft_direct_static_scratch(J, k) > LIMIT), None)
    assert K is not None, "no candidate size splits its sources on this GPU"
    x, w, xi = workloads.random_cloud(J, K)
    out = torch.full((K, 2), 3.0, dtype=torch.float64, device="cuda")
    with pytest.raises(sfd.SfdError) as e:
        sfd.sfd_surface_ft_direct_static(dev(torch, x), dev(torch, w), dev(torch, xi), out)
    assert e.value.status == -7 and "SFD_STATIC_SCRATCH_BYTES" in str(e.value)
    torch.cuda.synchronize()
    assert float(out.min()) == 3.0 and float(out.max()) == 3.0
    # the same sizes go through the workspace path
    nu = sfd.sfd_surface_ft(dev(torch, x), dev(torch, w), dev(torch, xi), 0.0)
    assert torch.isfinite(torch.view_as_real(nu)).all()

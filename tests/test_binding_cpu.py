"""CPU-side checks of the CUDA path's host logic (-m "not gpu"): the C-ABI library loads and exports every
symbol include/sfd.h declares, argument checking, size queries, the rule table and the host frequency
quadrature.  No compute call needs a GPU here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def sfd():
    from paper_2304_06340_b200 import build
    build.build()
    import paper_2304_06340_b200 as P
    return P


def test_exports_match_header(sfd):
    hdr = open(os.path.join(ROOT, "include", "sfd.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(sfd_[a-z0-9_]+)\s*\(", hdr))
    assert len(declared) >= 20
    lib = C.CDLL(sfd.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in sfd.h but not exported"
    assert declared == set(sfd.EXPORTS), declared ^ set(sfd.EXPORTS)


def test_mesh_sizes_P228(sfd):
    for line in open(os.path.join(ROOT, "tests", "golden", "mesh_counts.txt")):
        if line.startswith("#") or not line.strip():
            continue
        lvl, nv, nf = [int(t) for t in line.split()[:3]]
        got = sfd.sfd_mesh_icosphere_sizes(lvl)
        assert got[:2] == (nv, nf)
    with pytest.raises(sfd.SfdError) as e:
        sfd.sfd_mesh_icosphere_sizes(11)
    assert e.value.status == -2
    with pytest.raises(sfd.SfdError):
        sfd.sfd_mesh_icosphere_sizes(-1)


@pytest.mark.parametrize("q,deg", [(6, 4), (12, 6)])
def test_rule_exactness(sfd, q, deg):
    """Integral of u^a v^b over the standard simplex is a! b!/(a+b+2)!; weights sum to 1 (times area 1/2)."""
    from math import factorial
    lam, om = sfd.sfd_rule_table(q)
    assert abs(om.sum() - 1) < 1e-15 and (om > 0).all() and (lam > 0).all()
    assert np.abs(lam.sum(1) - 1).max() < 1e-15
    for a in range(deg + 1):
        for b in range(deg + 1 - a):
            got = 0.5 * np.sum(om * lam[:, 1] ** a * lam[:, 2] ** b)
            assert abs(got - factorial(a) * factorial(b) / factorial(a + b + 2)) < 2e-16 * 8
    # first inexact degree
    a, b = deg + 1, 0
    got = 0.5 * np.sum(om * lam[:, 1] ** a)
    assert abs(got - factorial(a) / factorial(a + 2)) > 1e-8
    with pytest.raises(sfd.SfdError):
        sfd.sfd_rule_table(7)


def test_freq_nodes_match_oracle(sfd, orc):
    for (nr, nt, nph, R) in [(32, 16, 32, 32.0), (5, 3, 4, 2.5), (1, 1, 1, 1.0), (128, 64, 8, 128.0)]:
        xi, W = sfd.sfd_freq_nodes((nr, nt, nph), R)
        xo, Wo = orc.freq_nodes(nr, nt, nph, R)
        assert np.abs(xi - xo).max() <= 4e-16 * R
        assert np.abs(W - Wo).max() <= 1e-14 * np.abs(Wo).max()
        # volume of the ball: sum W = 4/3 pi R^3 (n-point GL is exact for r^2 once n >= 2)
        if nr >= 2:
            assert abs(W.sum() - 4 / 3 * np.pi * R ** 3) < 1e-12 * R ** 3


def test_argument_errors(sfd):
    with pytest.raises(sfd.SfdError) as e:
        sfd.sfd_freq_nodes((0, 4, 4), 1.0)
    assert e.value.status == -2
    with pytest.raises(sfd.SfdError):
        sfd.sfd_freq_nodes((4, 4, 4), -1.0)
    with pytest.raises(sfd.SfdError):
        sfd.sfd_surface_ft_workspace(-1, 4, None, None, 0.0)
    with pytest.raises(sfd.SfdError):
        sfd.sfd_surface_ft_workspace(4, 4, None, None, 2.0)      # eps >= 1
    with pytest.raises(sfd.SfdError):
        sfd.sfd_surface_ft_workspace(4, 4, None, None, 1e-16)    # eps too small
    with pytest.raises(sfd.SfdError) as e:
        sfd.sfd_surface_ft_workspace(4, 4, None, None, 1e-6)     # X, S required
    assert e.value.status == -1
    assert sfd.sfd_surface_ft_workspace(0, 0, None, None, 0.0) == 0
    with pytest.raises(sfd.SfdError):
        sfd.sfd_weak_distance_workspace(80, 5, (4, 4, 4), 1.0, 0.0)  # unknown rule
    assert "rule" in sfd.binding._lib.sfd_last_error().decode()


def test_workspace_queries_scale(sfd):
    a = sfd.sfd_surface_ft_workspace(1000, 1000, [1, 1, 1], [32, 32, 32], 1e-6)
    b = sfd.sfd_surface_ft_workspace(1000, 1000, [1, 1, 1], [64, 64, 64], 1e-6)
    assert b > a > 0
    w0 = sfd.sfd_weak_distance_workspace(80, 6, (32, 16, 32), 32.0, 0.0)
    assert w0 >= 480 * 32 + 8192 * 48        # atoms + the xi_3 >= 0 half of the 16,384 nodes (R18)


def test_plan_and_workspace_queries(sfd):
    """sfd_surface_ft_plan / *_workspace are host-only: sizes of BASELINE.json's configs and argument checks."""
    w, nf, n2 = sfd.sfd_surface_ft_plan(30720, 1 << 20, [1, 1, 1], [128, 128, 128], 1e-9)
    assert w == 10 and nf == [180] * 3 and n2 == [360] * 3            # SURVEY 8(a) type-3 size table, config 2
    w, nf, n2 = sfd.sfd_surface_ft_plan(983040, 1 << 23, [1, 1, 1], [256, 256, 256], 1e-12)
    assert w == 13 and nf == [360] * 3 and n2 == [720] * 3            # config 3
    w, nf, n2 = sfd.sfd_surface_ft_plan(7864320, 1 << 26, [1, 1, 1], [1024, 1024, 1024], 1e-10)
    assert w == 11 and nf == [1350] * 3 and n2 == [2700] * 3          # config 5, level 8
    # the pruned transform fits one B200 at config 5 (the padded 2700^3 grid alone would be 315 GB); the query is
    # sized for complex strengths (127 GB), the ball-centred case that runs uses about half of it
    wb = sfd.sfd_weak_distance_workspace(20 * 4 ** 8, 6, (512, 256, 512), 1024.0, 1e-10)
    assert wb < 140e9
    assert sfd.sfd_surface_ft_workspace(100, 100, None, None, 0.0) >= 0
    for bad_eps in (-1.0, 1.0, 1e-15):
        with pytest.raises(sfd.SfdError):
            sfd.sfd_surface_ft_workspace(10, 10, [1, 1, 1], [1, 1, 1], bad_eps)
    with pytest.raises(sfd.SfdError):
        sfd.sfd_surface_ft_plan(10, 10, [1, 1, 1], [1, 1, 1], 0.0)    # the direct sum has no plan
    with pytest.raises(sfd.SfdError):
        sfd.sfd_weak_distance_workspace(10, 7, (4, 4, 4), 1.0, 0.0)   # unknown rule
    with pytest.raises(sfd.SfdError):
        sfd.sfd_weak_distance_lattice_workspace(10, 64, 7, 5.0, 0.0)  # odd M
    assert sfd.sfd_weak_distance_lattice_workspace(20 * 4 ** 7, 64, 128, 5.0, 1e-7) > 20 * 4 ** 7 * 64 * 32
    assert sfd.sfd_launch_count() >= 0


def test_lattice_transform_workspace_query(sfd):
    """sfd_surface_ft_lattice_workspace (host-only): the type-1 plan needs the lattice's nuhat band, not a type-3 grid;
    a lattice too coarse for the sources' extent is sized for the type-3 fallback; argument checks."""
    K = 417 ** 3
    t1 = sfd.sfd_surface_ft_lattice_workspace(1310720, 416, 5.0, [1, 1, 1], 1e-7)
    t3 = sfd.sfd_surface_ft_workspace(1310720, K, [1, 1, 1], [10 * np.pi] * 3, 1e-7)
    # expanded nodes of the fallback (24 K) + the half band 16 (M+1)^2 (M/2+1) + the n_in-plane intermediates + sorted
    # sources: well below the type-3 need
    band = 16 * 417 * 417 * 209
    assert 24 * K + band < t1 < 24 * K + 1.5 * band
    assert t1 < t3
    # growing extent -> larger spread grid -> more workspace, until the type-1 plan stops applying (2 pi h X ~ pi)
    a = sfd.sfd_surface_ft_lattice_workspace(1000, 64, 4.0, [0.5] * 3, 1e-9)
    b = sfd.sfd_surface_ft_lattice_workspace(1000, 64, 4.0, [1.0] * 3, 1e-9)
    assert a < b
    coarse = sfd.sfd_surface_ft_lattice_workspace(1000, 6, 2.0, [1, 1, 1], 1e-9)
    assert coarse >= sfd.sfd_surface_ft_workspace(1000, 343, [1, 1, 1], [4 * np.pi] * 3, 1e-9)
    for bad in ((7, 5.0, 1e-7), (0, 5.0, 1e-7), (16, -1.0, 1e-7), (16, 5.0, 2.0)):
        with pytest.raises(sfd.SfdError):
            sfd.sfd_surface_ft_lattice_workspace(10, bad[0], bad[1], [1, 1, 1], bad[2])


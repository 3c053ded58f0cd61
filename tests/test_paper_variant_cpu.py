"""Pins of the oracle's restatement of the paper's own variant: the 64-point iterated
Gauss-Legendre triangle rule, the cube lattice with the trapezoidal rule (eqs. 3.3-3.4) and
the norm in the paper's convention (eq. 2.7), against what the paper prints: the closed form eq. 4.2
and the error levels of Fig. 1(b).  Also the host logic of the CUDA library for the same pieces (no GPU)."""
import math

import numpy as np
import pytest


def closed_form_sigma_norm2(s):
    """||sigma||^2_{H_s(R^3)} of P:208 eq. 4.2, s < -1/2 (typed from the paper; mpmath for Gamma and K_nu)."""
    import mpmath as mp
    s = mp.mpf(s)
    return float(4 * mp.pi ** 1.5 / mp.gamma(-s) *
                 (mp.gamma(-s - 0.5) - 2 * (2 * mp.pi) ** (-s - 0.5) * mp.besselk(-s - 0.5, 4 * mp.pi)))


def test_rule64_polynomial_exactness(orc):
    """8 x 8 iterated Gauss-Legendre: exact for total degree <= 14 (u-degree d+1 <= 15 after the collapse), not 15."""
    lam, om = orc.rule(64)
    assert lam.shape == (64, 3) and abs(om.sum() - 1) < 1e-15 and np.all(om > 0)
    assert np.all(lam > 0) and np.abs(lam.sum(1) - 1).max() < 1e-15          # interior points
    worst = 0.0
    for p in range(15):
        for q in range(15 - p):
            exact = math.factorial(p) * math.factorial(q) / math.factorial(p + q + 2) * 2   # / area of Q_0
            worst = max(worst, abs((om * lam[:, 1] ** p * lam[:, 2] ** q).sum() - exact) / exact)
    assert worst < 5e-15
    exact15 = math.factorial(7) * math.factorial(8) / math.factorial(17) * 2
    assert abs((om * lam[:, 1] ** 7 * lam[:, 2] ** 8).sum() - exact15) / exact15 > 1e-6     # degree 15 is not exact


def test_rule64_single_triangle_exact_transform(orc):
    """Against the exact triangle transform P:128 eq. 2.19 (e^{-i xi.x} form): the 64-point rule is at rounding level
    where the 6-point rule has error 6e-8 (|xi| = 2, triangle of diameter ~1.2)."""
    V = np.array([[0.1, 0.0, 0.2], [1.1, 0.3, -0.1], [0.3, 0.9, 0.4]])
    F = np.array([[0, 1, 2]], np.int32)
    A = 0.5 * np.linalg.norm(np.cross(V[1] - V[0], V[2] - V[0]))
    xi = np.array([[1.1, -0.7, 1.5]])
    xi *= 2.0 / np.linalg.norm(xi)
    exact = 0
    for i in range(3):
        den = 1.0
        for j in range(3):
            if j != i:
                den *= xi[0] @ (V[i] - V[j])
        exact += np.exp(-1j * (xi[0] @ V[i])) / den
    exact *= -2 * A
    e64 = abs(orc.direct_sum(*orc.nodes(V, F, 64), xi)[0] - exact) / A
    e6 = abs(orc.direct_sum(*orc.nodes(V, F, 6), xi)[0] - exact) / A
    assert e64 < 1e-12 and e6 > 1e-9   # (the closed form itself cancels to ~1e-14)


def test_lattice_structure(orc):
    M, xi_max = 8, 5.0
    xi, W = orc.lattice_nodes(M, xi_max)
    n = M + 1
    assert xi.shape == (n ** 3, 3)
    h = 2 * xi_max / M
    assert abs(W.sum() - (2 * xi_max) ** 3) < 1e-10                           # the rule integrates 1 over the cube
    assert np.allclose(xi[0], -2 * np.pi * xi_max) and np.allclose(xi[-1], 2 * np.pi * xi_max)
    assert np.allclose(xi[1] - xi[0], [0, 0, 2 * np.pi * h])                   # last index fastest
    w = np.round(W / h ** 3, 12)
    counts = {v: int((w == v).sum()) for v in (1.0, 0.5, 0.25, 0.125)}
    assert counts == {1.0: (M - 1) ** 3, 0.5: 6 * (M - 1) ** 2, 0.25: 12 * (M - 1), 0.125: 8}
    k = (3 * n + 5) * n + 7
    assert np.allclose(xi[k], 2 * np.pi * h * (np.array([3, 5, 7]) - M / 2))


def test_trapezoid_vs_closed_form_eq_4_2(orc):
    """Fig. 1(b): at xi_max = 5 the relative error |I - I_M|/I "for s = -5 [is] dominated by the truncation
    error at the level of 10^-7 ... while the total error continues to decrease for s = -10 and eventually reaches the
    level of 10^-13".  Pins lattice, weights, sigmahat, the 2 pi mapping and the weight convention at once."""
    zero = {}
    for M in (64, 128):
        xi, W = orc.lattice_nodes(M, 5.0)
        zero[M] = (xi, W, np.zeros(len(W), complex))
    for s, M, lo, hi in ((-5, 64, 1e-8, 1e-7), (-5, 128, 1e-8, 1e-7), (-10, 64, 1e-8, 1e-6), (-10, 128, 0.0, 1e-13)):
        xi, W, nu = zero[M]
        I = orc.reduce_ex(nu, xi, W, -s, 1 / (2 * np.pi), 1.0)                # nuhat = 0: integrand |sigmahat|^2 weight
        rel = abs(I - closed_form_sigma_norm2(s)) / closed_form_sigma_norm2(s)
        assert lo <= rel <= hi, (s, M, rel)


def test_reduce_ex_reduces_to_reduce(orc):
    rng = np.random.default_rng(5)
    xi = rng.normal(size=(500, 3)) * 4
    W = rng.random(500)
    nu = rng.normal(size=500) + 1j * rng.normal(size=500)
    a = orc.reduce(nu, xi, W, 2.0)
    b = orc.reduce_ex(nu, xi, W, 2.0, 1.0, 1.0 / (2 * np.pi) ** 3)
    assert abs(a - b) <= 1e-15 * a


# ---- host logic of the CUDA library (runs without a GPU) -----------------------------------------------------
def test_library_rule64_and_lattice_host(orc):
    import paper_2304_06340_b200 as P
    lam, om = P.sfd_rule_table(64)
    lo, oo = orc.rule(64)
    assert np.abs(lam - lo).max() < 2e-16 and np.abs(om - oo).max() < 2e-17
    xi, W = P.sfd_lattice_nodes(12, 5.0)
    xo, Wo = orc.lattice_nodes(12, 5.0)
    assert np.array_equal(xi, xo) and np.array_equal(W, Wo)
    for bad in (3, 0, -2):
        with pytest.raises(P.SfdError):
            P.sfd_lattice_nodes(bad, 5.0)
    with pytest.raises(P.SfdError):
        P.sfd_lattice_nodes(8, -1.0)


def test_reduce_pair_pins(orc):
    """Mesh against mesh: the pair reduction against (i) the sphere reduction when the second operand
    is sigmahat sampled on the nodes, (ii) the closed form for a translated copy, |1 - e^{-i xi.c}|^2 = 4 sin^2(xi.c/2),
    (iii) the triangle inequality through the sphere."""
    V1, F1 = orc.mesh_icosphere(1)
    V2, F2 = orc.mesh_icosphere(2)
    xi, W = orc.freq_nodes(12, 6, 8, 10.0)
    n1 = orc.direct_sum(*orc.nodes(V1, F1, 6), xi)
    n2 = orc.direct_sum(*orc.nodes(V2, F2, 6), xi)
    sig = np.array([orc.sigma_hat(float(np.linalg.norm(v))) for v in xi], complex)
    for s in (1.0, 2.0):
        I1 = orc.reduce(n1, xi, W, s)
        assert abs(orc.reduce_pair(n1, sig, xi, W, s) - I1) <= 1e-14 * I1
        assert orc.reduce_pair(n1, n1, xi, W, s) == 0.0
        d12 = np.sqrt(orc.reduce_pair(n1, n2, xi, W, s))
        d1, d2 = np.sqrt(I1), np.sqrt(orc.reduce(n2, xi, W, s))
        assert abs(d1 - d2) <= d12 <= d1 + d2 and abs(d12 - np.sqrt(orc.reduce_pair(n2, n1, xi, W, s))) < 1e-15
    c = np.array([0.3, -0.2, 0.1])
    nt = orc.direct_sum(orc.nodes(V1, F1, 6)[0] + c, orc.nodes(V1, F1, 6)[1], xi)
    expect = (W * np.abs(n1) ** 2 * 4 * np.sin(xi @ c / 2) ** 2 * (1 + (xi ** 2).sum(1)) ** -2.0).sum() / (2 * np.pi) ** 3
    assert abs(orc.reduce_pair(n1, nt, xi, W, 2.0) - expect) <= 1e-12 * expect

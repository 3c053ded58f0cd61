"""Pins of the oracle's exact triangle transform (oracle/sfd_oracle_exact.cpp; eq. 2.19, eq. 2.20):
the paper's formula evaluated literally at 60-100 digits, the 64-point rule where it is exact to rounding, closed forms
of the degenerate directions, and the cube's transform.  CPU only."""
import mpmath as mp
import numpy as np
import pytest

TRI = np.array([[0.9, 0.1, 0.2], [-0.1, 0.8, 0.3], [0.2, -0.15, 1.1]])
F1 = np.array([[0, 1, 2]], dtype=np.int32)


def eq_2_19(p, xi, dps=60):
    """-2A sum_i e^{-i xi.p_i} / prod_{j != i} xi.(p_i - p_j): eq. 2.19 in the e^{-i xi.x} convention."""
    mp.mp.dps = dps
    P = [[mp.mpf(float(c)) for c in v] for v in p]
    X = [mp.mpf(float(c)) for c in xi]
    e1 = [P[1][c] - P[0][c] for c in range(3)]
    e2 = [P[2][c] - P[0][c] for c in range(3)]
    cr = [e1[1] * e2[2] - e1[2] * e2[1], e1[2] * e2[0] - e1[0] * e2[2], e1[0] * e2[1] - e1[1] * e2[0]]
    A2 = mp.sqrt(sum(c * c for c in cr))
    al = [sum(X[c] * P[i][c] for c in range(3)) for i in range(3)]
    tot = mp.mpc(0)
    for i in range(3):
        den = mp.mpf(1)
        for j in range(3):
            if j != i:
                den *= al[i] - al[j]
        tot += mp.exp(-1j * al[i]) / den
    return complex(-A2 * tot)


def area(p):
    return 0.5 * np.linalg.norm(np.cross(p[1] - p[0], p[2] - p[0]))


def test_matches_eq_2_19_literally(orc):
    """Generic directions and magnitudes from 1e-3 to 1e3: the binary128 evaluation of the printed formula, and (at the
    small magnitudes, where the alpha_i are within 1e-5 of each other) the arbitrary-precision one."""
    rng = np.random.default_rng(0)
    xis = [rng.normal(size=3) * m for m in (1e-3, 0.05, 0.7, 1.0, 3.0, 40.0, 1e3) for _ in range(6)]
    got = orc.exact_ft(TRI, F1, np.array(xis))
    for xi, g in zip(xis, got):
        ref = eq_2_19(TRI, xi, dps=80)
        assert abs(g - ref) <= 4e-16 * area(TRI), (xi, g, ref)


def test_nearly_degenerate_against_high_precision(orc):
    """xi almost orthogonal to an edge -- eq. 2.19 at 120 digits still resolves differences of 1e-9..1e-30."""
    e1 = TRI[1] - TRI[0]
    n = np.cross(e1, TRI[2] - TRI[0])
    perp = np.cross(e1, n)
    perp /= np.linalg.norm(perp)
    for mag in (0.3, 7.0, 300.0):
        for tilt in (1e-3, 1e-9, 1e-15):
            xi = mag * (perp + tilt * e1 / np.linalg.norm(e1))
            got = orc.exact_ft(TRI, F1, xi[None])[0]
            ref = eq_2_19(TRI, xi, dps=120)
            assert abs(got - ref) <= 4e-16 * area(TRI), (mag, tilt, got, ref)


def test_degenerate_directions_closed_form(orc):
    """xi along the normal: all alpha_i equal, Q^ = A e^{-i alpha}.  xi exactly orthogonal to an edge (u = 0 to rounding
    is not exact, so build the triangle on a lattice where it is): exp[0,0,b] = (e^b - 1 - b)/b^2."""
    p = np.array([[0.0, 0.0, 0.0], [1.0, 0.0, 0.0], [0.0, 2.0, 0.0]])
    A = 1.0
    for a in (0.0, 0.5, 30.0):
        got = orc.exact_ft(p + np.array([0, 0, 0.25]), F1, np.array([[0.0, 0.0, a]]))[0]
        assert abs(got - A * np.exp(-1j * a * 0.25)) <= 3e-16
    for b in (1e-6, 0.4, 2.0, 55.0):
        xi = np.array([0.0, b / 2.0, 0.0])          # xi.e1 = 0 exactly, xi.e2 = b
        got = orc.exact_ft(p, F1, xi[None])[0]
        mp.mp.dps = 50
        z = mp.mpc(0, -b)
        ref = complex(2 * A * (mp.exp(z) - 1 - z) / z ** 2)
        assert abs(got - ref) <= 3e-16, (b, got, ref)
    # two coincident nodes away from 0: xi.p_1 = xi.p_2
    xi = np.array([2.0, 1.0, 0.0])                  # alpha = (0, 2, 2)
    got = orc.exact_ft(p, F1, xi[None])[0]
    mp.mp.dps = 50
    z = mp.mpc(0, -2)
    ref = complex(2 * A * (mp.exp(z) * (z - 1) + 1) / z ** 2)   # exp[0, z, z] = (e^z (z - 1) + 1)/z^2
    assert abs(got - ref) <= 3e-16


def test_area_at_zero_and_rule64(orc):
    """xi = 0 gives the area; at |xi| h <~ 1 the 64-point rule (exact to degree 14) reproduces the transform."""
    V, F = orc.mesh_icosphere(2)
    x, w = orc.nodes(V, F, 64)
    rng = np.random.default_rng(1)
    xi = np.vstack([np.zeros((1, 3)), rng.normal(size=(40, 3)) * 1.5])
    got = orc.exact_ft(V, F, xi)
    assert abs(got[0] - w.sum()) <= 1e-14 * w.sum()
    ref = orc.direct_sum(x, w, xi)
    assert np.abs(got - ref).max() <= 2e-14 * w.sum()


def test_normal_invariance_eq_2_20(orc):
    """P:135 eq. 2.20: Q^(xi_perp + a n) = e^{-i a n.p_0} Q^(xi_perp)."""
    n = np.cross(TRI[1] - TRI[0], TRI[2] - TRI[0])
    n /= np.linalg.norm(n)
    base = np.array([0.4, 0.2, -0.3])
    base -= n * (base @ n)
    a = np.array([0.0, 0.7, -3.1, 12.5, 400.0])
    vals = orc.exact_ft(TRI, F1, base[None] + a[:, None] * n[None])
    for ai, v in zip(a, vals):
        assert abs(v - np.exp(-1j * ai * (n @ TRI[0])) * vals[0]) <= 1e-13 * area(TRI) * max(1.0, abs(ai))


def test_cube_surface(orc):
    """Surface of [-1/2, 1/2]^3 (12 triangles): 2 cos(xi_x/2) sinc(xi_y/2) sinc(xi_z/2) + cyclic."""
    c = 0.5
    V = np.array([[sx * c, sy * c, sz * c] for sx in (-1, 1) for sy in (-1, 1) for sz in (-1, 1)])
    idx = {tuple(np.sign(v).astype(int)): i for i, v in enumerate(V)}
    F = []
    for ax in range(3):
        for s in (-1, 1):
            q = []
            for a, b in ((-1, -1), (1, -1), (1, 1), (-1, 1)):
                k = [0, 0, 0]
                k[ax] = s
                k[(ax + 1) % 3] = a
                k[(ax + 2) % 3] = b
                q.append(idx[tuple(k)])
            F += [[q[0], q[1], q[2]], [q[0], q[2], q[3]]]
    F = np.array(F, dtype=np.int32)
    rng = np.random.default_rng(2)
    xi = np.vstack([rng.normal(size=(30, 3)) * m for m in (0.1, 3.0, 60.0)] + [np.array([[0.0, 0.0, 7.0], [2.0, 2.0, 0.0]])])
    got = orc.exact_ft(V, F, xi)

    def sinc(t):
        return np.sinc(t / np.pi)
    ref = sum(2 * np.cos(xi[:, a] / 2) * sinc(xi[:, (a + 1) % 3] / 2) * sinc(xi[:, (a + 2) % 3] / 2) for a in range(3))
    assert np.abs(got - ref).max() <= 1e-14 * 6


def test_polyhedron_approaches_sphere(orc):
    """The exact transform of T_N tends to sigma^ = 4 pi sin r / r (eq. 2.14) at the quadratic rate."""
    xi = np.array([[0.0, 0.0, 2.0], [1.0, -2.0, 0.5]])
    errs = []
    for N in (2, 3, 4):
        V, F = orc.mesh_icosphere(N)
        got = orc.exact_ft(V, F, xi)
        ref = np.array([orc.sigma_hat(np.linalg.norm(v)) for v in xi])
        errs.append(np.abs(got - ref).max())
    assert 3.7 <= errs[0] / errs[1] <= 4.3 and 3.7 <= errs[1] / errs[2] <= 4.3, errs

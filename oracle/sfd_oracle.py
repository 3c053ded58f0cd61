"""numpy/ctypes face of the CPU oracle (oracle/sfd_oracle.cpp, sfd_oracle_exact.cpp).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import
this module.  It never imports paper_2304_06340_b200 and the CUDA path never imports it.
Every function is a marshalling shim: all arithmetic is in sfd_oracle.cpp.
"""
import ctypes as C
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import build_oracle  # noqa: E402

_lib = C.CDLL(build_oracle.build())

_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_ip = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_i64 = C.c_int64

_lib.orc_mesh_sizes.argtypes = [C.c_int, C.POINTER(_i64), C.POINTER(_i64)]
_lib.orc_mesh_icosphere.argtypes = [C.c_int, _dp, _ip]
_lib.orc_subdivide.argtypes = [_dp, _i64, _ip, _i64, _dp, _ip]
_lib.orc_subdivide.restype = _i64
_lib.orc_rule.argtypes = [C.c_int, _dp, _dp]
_lib.orc_nodes.argtypes = [_dp, _i64, _ip, _i64, C.c_int, _dp, _dp]
_lib.orc_gauss_legendre.argtypes = [C.c_int, C.c_double, C.c_double, _dp, _dp]
_lib.orc_freq_nodes.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, _dp, _dp]
_lib.orc_direct_sum.argtypes = [_dp, _dp, _i64, _dp, _i64, _dp]
_lib.orc_exact_ft.argtypes = [_dp, _i64, _ip, _i64, _dp, _i64, _dp,
                               np.ctypeslib.ndpointer(np.int64, flags="C_CONTIGUOUS"), _i64, C.POINTER(_i64)]
_lib.orc_sigma_hat.argtypes = [C.c_double]
_lib.orc_sigma_hat.restype = C.c_double
_lib.orc_reduce.argtypes = [_dp, _dp, _dp, _i64, C.c_double]
_lib.orc_reduce.restype = C.c_double
_lib.orc_lattice_nodes.argtypes = [C.c_int, C.c_double, _dp, _dp]
_lib.orc_reduce_ex.argtypes = [_dp, _dp, _dp, _i64, C.c_double, C.c_double, C.c_double]
_lib.orc_reduce_ex.restype = C.c_double
_lib.orc_reduce_pair.argtypes = [_dp, _dp, _dp, _dp, _i64, C.c_double]
_lib.orc_reduce_pair.restype = C.c_double
_lib.orc_weak_distance.argtypes = [_dp, _i64, _ip, _i64, C.c_int, C.c_double, C.c_double, C.c_int,
                                   C.c_int, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
_lib.orc_num_threads.restype = C.c_int


def _chk(rc, what):
    if rc != 0:
        raise ValueError(f"oracle {what} failed with status {rc}")


def mesh_sizes(level):
    nv, nf = _i64(), _i64()
    _lib.orc_mesh_sizes(level, C.byref(nv), C.byref(nf))
    return nv.value, nf.value


def mesh_icosphere(level):
    nv, nf = mesh_sizes(level)
    V = np.empty((nv, 3), np.float64)
    F = np.empty((nf, 3), np.int32)
    _chk(_lib.orc_mesh_icosphere(level, V, F), "mesh_icosphere")
    return V, F


def subdivide(V, F):
    V = np.ascontiguousarray(V, np.float64)
    F = np.ascontiguousarray(F, np.int32)
    nv, nf = len(V), len(F)
    Vo = np.empty((nv + 3 * nf // 2, 3), np.float64)
    Fo = np.empty((4 * nf, 3), np.int32)
    e = _lib.orc_subdivide(V, nv, F, nf, Vo, Fo)
    assert e == 3 * nf // 2, "not a closed manifold mesh"
    return Vo, Fo


def rule(q):
    lam = np.empty((q, 3), np.float64)
    om = np.empty(q, np.float64)
    if _lib.orc_rule(q, lam, om) != q:
        raise ValueError(f"unknown rule {q}")
    return lam, om


def nodes(V, F, q):
    V = np.ascontiguousarray(V, np.float64)
    F = np.ascontiguousarray(F, np.int32)
    x = np.empty((len(F) * q, 3), np.float64)
    w = np.empty(len(F) * q, np.float64)
    _chk(_lib.orc_nodes(V, len(V), F, len(F), q, x, w), "nodes")
    return x, w


def gauss_legendre(n, a=-1.0, b=1.0):
    x = np.empty(n, np.float64)
    w = np.empty(n, np.float64)
    _chk(_lib.orc_gauss_legendre(n, a, b, x, w), "gauss_legendre")
    return x, w


def freq_nodes(n_r, n_th, n_ph, R):
    K = n_r * n_th * n_ph
    xi = np.empty((K, 3), np.float64)
    W = np.empty(K, np.float64)
    _chk(_lib.orc_freq_nodes(n_r, n_th, n_ph, R, xi, W), "freq_nodes")
    return xi, W


def direct_sum(x, w, xi):
    """nuhat_k = sum_j w_j exp(-i xi_k . x_j) as complex128[K]."""
    x = np.ascontiguousarray(x, np.float64).reshape(-1, 3)
    w = np.ascontiguousarray(w, np.float64).reshape(-1)
    xi = np.ascontiguousarray(xi, np.float64).reshape(-1, 3)
    out = np.empty((len(xi), 2), np.float64)
    _chk(_lib.orc_direct_sum(x, w, len(w), xi, len(xi), out), "direct_sum")
    return out.view(np.complex128).reshape(-1)


def _exact_pair_mp(p, xi):
    """P:128 eq. 2.19 for ONE face and ONE frequency whose alpha_i = xi.p_i are too close for binary128 ("large
    cancellation errors"): the printed formula -2A sum_i e^{-i alpha_i} / prod_{j != i}(alpha_i - alpha_j) with as many
    digits as its cancellation needs, or, where two or three alpha coincide EXACTLY and the printed formula is 0/0, its
    limit: 2A times the divided difference exp[z_0, z_1, z_2], z = -i alpha, with repeated nodes (textbook definitions:
    f[z, z, w] = (f[z, w] - f'(z)) / (w - z), f[z, w] = (f(w) - f(z)) / (w - z), f[z, z, z] = f''(z) / 2).  Returns an mpmath
    complex (the caller sums a frequency's pairs before rounding)."""
    import mpmath as mp
    mp.mp.dps = 400                      # the dot products of fp64 inputs are exact at this precision
    P = [[mp.mpf(float(c)) for c in v] for v in p]
    X = [mp.mpf(float(c)) for c in xi]
    e1 = [P[1][c] - P[0][c] for c in range(3)]
    e2 = [P[2][c] - P[0][c] for c in range(3)]
    cr = [e1[1] * e2[2] - e1[2] * e2[1], e1[2] * e2[0] - e1[0] * e2[2], e1[0] * e2[1] - e1[1] * e2[0]]
    A2 = mp.sqrt(sum(c * c for c in cr))
    al = [sum(X[c] * P[i][c] for c in range(3)) for i in range(3)]
    same = [(i, j) for i in range(3) for j in range(i + 1, 3) if al[i] == al[j]]
    if len(same) == 3:                   # all three coincide (xi along the normal, xi = 0): exp''(z) / 2
        return A2 * mp.exp(-1j * al[0]) / 2
    if len(same) == 1:                   # exactly two coincide (xi orthogonal to an edge): f[z, z, w]
        i, j = same[0]
        k = 3 - i - j
        z, w = -1j * al[i], -1j * al[k]
        first = (mp.exp(w) - mp.exp(z)) / (w - z)
        return A2 * (first - mp.exp(z)) / (w - z)
    dmin = min(abs(al[i] - al[j]) for i in range(3) for j in range(i + 1, 3))
    amax = max(1, max(abs(a) for a in al))
    mp.mp.dps = 60 + 3 * int(mp.ceil(mp.log10(amax / dmin)))     # 1/d^2 of cancellation, 1/d in each difference
    tot = mp.mpc(0)
    for i in range(3):
        den = mp.mpf(1)
        for j in range(3):
            if j != i:
                den *= al[i] - al[j]
        tot += mp.exp(-1j * al[i]) / den
    return -A2 * tot


def exact_ft(V, F, xi):
    """Exact transform of the flat mesh's surface measure, sum over faces of P:128 eq. 2.19 (e^{-i xi.x} convention):
    complex128[K].  The formula is evaluated as printed in binary128 (sfd_oracle_exact.cpp); the pairs whose alpha are
    too close for that are evaluated by _exact_pair_mp and added here."""
    V = np.ascontiguousarray(V, np.float64).reshape(-1, 3)
    F = np.ascontiguousarray(F, np.int32).reshape(-1, 3)
    xi = np.ascontiguousarray(xi, np.float64).reshape(-1, 3)
    out = np.empty((len(xi), 2), np.float64)
    cap = 1 << 16
    while True:
        skipped = np.empty((cap, 2), np.int64)
        n = C.c_int64(0)
        rc = _lib.orc_exact_ft(V, len(V), F, len(F), xi, len(xi), out, skipped, cap, C.byref(n))
        if rc != -2:
            break
        cap = int(n.value)
    _chk(rc, "exact_ft")
    res = out.view(np.complex128).reshape(-1)
    extra = {}                           # the skipped pairs of a frequency are summed at full precision, rounded once
    for k, f in skipped[:n.value]:
        extra[int(k)] = extra.get(int(k), 0) + _exact_pair_mp(V[F[f]], xi[k])
    for k, v in extra.items():
        res[k] += complex(v)
    return res


def sigma_hat(r):
    return _lib.orc_sigma_hat(float(r))


def reduce(nuhat, xi, W, s):
    """I = (2 pi)^-3 sum_k W_k |nuhat_k - sigmahat|^2 (1+|xi_k|^2)^-s."""
    nu = np.ascontiguousarray(nuhat, np.complex128).view(np.float64).reshape(-1, 2)
    xi = np.ascontiguousarray(xi, np.float64).reshape(-1, 3)
    W = np.ascontiguousarray(W, np.float64).reshape(-1)
    return _lib.orc_reduce(nu, xi, W, len(W), float(s))


def lattice_nodes(M, xi_max):
    """The paper's cube lattice: xi' = 2 pi xi_ijk as float64[(M+1)^3, 3], trapezoid weights w_ijk h^3."""
    K = (M + 1) ** 3
    xi = np.empty((K, 3), np.float64)
    W = np.empty(K, np.float64)
    _chk(_lib.orc_lattice_nodes(M, xi_max, xi, W), "lattice_nodes")
    return xi, W


def reduce_ex(nuhat, xi, W, s, scale, pref):
    """pref * sum_k W_k |nuhat_k - sigmahat|^2 (1 + (scale |xi_k|)^2)^-s."""
    nu = np.ascontiguousarray(nuhat, np.complex128).view(np.float64).reshape(-1, 2)
    xi = np.ascontiguousarray(xi, np.float64).reshape(-1, 3)
    W = np.ascontiguousarray(W, np.float64).reshape(-1)
    return _lib.orc_reduce_ex(nu, xi, W, len(W), float(s), float(scale), float(pref))


def reduce_pair(a, b, xi, W, s):
    """(2 pi)^-3 sum_k W_k |a_k - b_k|^2 (1+|xi_k|^2)^-s for two transforms on the same nodes."""
    a = np.ascontiguousarray(a, np.complex128).view(np.float64).reshape(-1, 2)
    b = np.ascontiguousarray(b, np.complex128).view(np.float64).reshape(-1, 2)
    xi = np.ascontiguousarray(xi, np.float64).reshape(-1, 3)
    W = np.ascontiguousarray(W, np.float64).reshape(-1)
    return _lib.orc_reduce_pair(a, b, xi, W, len(W), float(s))


def weak_distance(V, F, q, s, R, n_r, n_th, n_ph):
    V = np.ascontiguousarray(V, np.float64)
    F = np.ascontiguousarray(F, np.int32)
    d, i = C.c_double(), C.c_double()
    _chk(_lib.orc_weak_distance(V, len(V), F, len(F), q, s, R, n_r, n_th, n_ph, C.byref(d), C.byref(i)),
         "weak_distance")
    return d.value, i.value


def num_threads():
    return _lib.orc_num_threads()

"""ctypes face of libsfd.so (include/sfd.h).  Argument marshalling only: torch supplies device memory and the
current CUDA stream; every step of the path runs in the library's kernels.  There is no fallback: if the
library is not built (`python -m paper_2304_06340_b200.build`) importing this module raises.
"""
import ctypes as C
import os

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libsfd.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2304_06340_b200.build` "
                      "(nvcc, sm_100a). There is no CPU fallback.")
_lib = C.CDLL(LIB_PATH)

SFD_OK = 0
STATUS = {0: "SFD_OK", -1: "SFD_ERR_NULL", -2: "SFD_ERR_INVALID_ARG", -3: "SFD_ERR_BUFFER_TOO_SMALL",
          -4: "SFD_ERR_WORKSPACE_TOO_SMALL", -5: "SFD_ERR_CUDA", -6: "SFD_ERR_RESERVED_6", -7: "SFD_ERR_UNSUPPORTED"}
SFD_RULE_SYM6_DEG4, SFD_RULE_SYM12_DEG6 = 6, 12


class sfd_freq_quadrature(C.Structure):
    _fields_ = [("n_r", C.c_int32), ("n_theta", C.c_int32), ("n_phi", C.c_int32)]


class SfdError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


_vp, _i64, _sz, _dbl = C.c_void_p, C.c_int64, C.c_size_t, C.c_double
_P = C.POINTER
_SIGS = {
    "sfd_last_error": (C.c_char_p, []),
    "sfd_version": (C.c_char_p, []),
    "sfd_release_cache": (C.c_int, []),
    "sfd_mesh_icosphere_sizes": (C.c_int, [C.c_int, _P(_i64), _P(_i64), _P(_sz)]),
    "sfd_mesh_icosphere": (C.c_int, [C.c_int, _vp, _vp, _vp, _sz, _vp]),
    "sfd_nodes": (C.c_int, [_vp, _i64, _vp, _i64, C.c_int, _vp, _vp, _vp]),
    "sfd_rule_table": (C.c_int, [C.c_int, _vp, _vp]),
    "sfd_freq_nodes": (C.c_int, [_P(sfd_freq_quadrature), _dbl, _vp, _vp]),
    "sfd_freq_nodes_workspace": (C.c_int, [_P(sfd_freq_quadrature), _P(_sz)]),
    "sfd_freq_nodes_device": (C.c_int, [_P(sfd_freq_quadrature), _dbl, _vp, _vp, _vp, _sz, _vp]),
    "sfd_freq_nodes_device_range": (C.c_int, [_P(sfd_freq_quadrature), _dbl, C.c_int32, C.c_int32, _vp, _vp, _vp, _sz,
                                              _vp]),
    "sfd_surface_ft_workspace": (C.c_int, [_i64, _i64, _P(_dbl), _P(_dbl), _dbl, _P(_sz)]),
    "sfd_surface_ft_plan": (C.c_int, [_i64, _i64, _P(_dbl), _P(_dbl), _dbl, _P(C.c_int32), _P(_i64), _P(_i64)]),
    "sfd_surface_ft": (C.c_int, [_vp, _vp, _i64, _vp, _i64, _dbl, _vp, _vp, _sz, _vp]),
    "sfd_surface_ft_direct_static_scratch": (C.c_int, [_i64, _i64, _P(_sz)]),
    "sfd_surface_ft_direct_static": (C.c_int, [_vp, _vp, _i64, _vp, _i64, _vp, _vp]),
    "sfd_reduce_workspace": (C.c_int, [_i64, _P(_sz)]),
    "sfd_reduce": (C.c_int, [_vp, _vp, _vp, _i64, _dbl, _vp, _sz, _vp, _P(_dbl)]),
    "sfd_weak_distance_workspace": (C.c_int, [_i64, C.c_int, _P(sfd_freq_quadrature), _dbl, _dbl, _dbl, _P(_sz)]),
    "sfd_weak_distance_targets": (C.c_int, [_P(sfd_freq_quadrature), _P(_i64)]),
    "sfd_weak_distance": (C.c_int, [_vp, _i64, _vp, _i64, C.c_int, _dbl, _dbl, _P(sfd_freq_quadrature), _dbl, _vp,
                                    _sz, _vp, _P(_dbl), _P(_dbl)]),
    "sfd_lattice_nodes": (C.c_int, [C.c_int32, _dbl, _vp, _vp]),
    "sfd_lattice_nodes_device": (C.c_int, [C.c_int32, _dbl, _vp, _vp, _vp]),
    "sfd_reduce_ex": (C.c_int, [_vp, _vp, _vp, _i64, _dbl, _dbl, _dbl, _vp, _sz, _vp, _P(_dbl)]),
    "sfd_reduce_lattice": (C.c_int, [_vp, C.c_int32, _dbl, _dbl, _dbl, _dbl, _vp, _sz, _vp, _P(_dbl)]),
    "sfd_surface_ft_lattice_workspace": (C.c_int, [_i64, C.c_int32, _dbl, _P(_dbl), _dbl, _P(_sz)]),
    "sfd_surface_ft_lattice": (C.c_int, [_vp, _vp, _i64, C.c_int32, _dbl, _dbl, _vp, _vp, _sz, _vp]),
    "sfd_weak_distance_lattice_workspace": (C.c_int, [_i64, C.c_int, C.c_int32, _dbl, _dbl, _dbl, _P(_sz)]),
    "sfd_weak_distance_lattice": (C.c_int, [_vp, _i64, _vp, _i64, C.c_int, _dbl, _dbl, C.c_int32, _dbl, _vp, _sz, _vp,
                                            _P(_dbl), _P(_dbl)]),
    "sfd_exact_ft_workspace": (C.c_int, [_i64, _P(_sz)]),
    "sfd_exact_ft": (C.c_int, [_vp, _i64, _vp, _i64, _vp, _i64, _vp, _vp, _sz, _vp]),
    "sfd_reduce_pair": (C.c_int, [_vp, _vp, _vp, _vp, _i64, _dbl, _vp, _sz, _vp, _P(_dbl)]),
    "sfd_surface_ft_host": (C.c_int, [_vp, _vp, _i64, _vp, _i64, _dbl, _vp]),
    "sfd_weak_distance_host": (C.c_int, [_vp, _i64, _vp, _i64, C.c_int, _dbl, _dbl, _P(sfd_freq_quadrature), _dbl,
                                         _P(_dbl), _P(_dbl)]),
    "sfd_launch_count": (C.c_longlong, []),
    "sfd_extents_workspace": (C.c_int, [_P(_sz)]),
    "sfd_extents": (C.c_int, [_vp, _i64, _P(_dbl), _P(_dbl), _vp, _sz, _vp]),
    "sfd_weak_distance_range_workspace": (C.c_int, [_i64, C.c_int, _P(sfd_freq_quadrature), _dbl, C.c_int32, C.c_int32,
                                                    _dbl, _dbl, _P(_sz)]),
    "sfd_weak_distance_range": (C.c_int, [_vp, _i64, _vp, _i64, C.c_int, _dbl, _dbl, _P(sfd_freq_quadrature), C.c_int32,
                                          C.c_int32, _dbl, _vp, _sz, _vp, _vp]),
    "sfd_mesh_distance_workspace": (C.c_int, [_i64, _i64, C.c_int, _P(sfd_freq_quadrature), _dbl, _dbl, _dbl, _P(_sz)]),
    "sfd_mesh_distance": (C.c_int, [_vp, _i64, _vp, _i64, _vp, _i64, _vp, _i64, C.c_int, _dbl, _dbl,
                                    _P(sfd_freq_quadrature), _dbl, _vp, _sz, _vp, _P(_dbl), _P(_dbl)]),
    "sfd_set_profiling": (C.c_int, [C.c_int]),
    "sfd_set_grid_precision": (C.c_int, [C.c_int]),
    "sfd_last_stage_times": (C.c_int, [_P(C.c_char_p), _P(C.c_float), C.c_int]),
}
for _name, (_res, _args) in _SIGS.items():
    _f = getattr(_lib, _name)
    _f.restype, _f.argtypes = _res, _args
EXPORTS = tuple(_SIGS)


def _chk(rc):
    if rc != SFD_OK:
        raise SfdError(rc, _lib.sfd_last_error().decode())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


def _dev_f64(t, cols=None):
    assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous(), "need a contiguous CUDA float64 tensor"
    if cols is not None:
        assert t.dim() == 2 and t.shape[1] == cols
    return t


def _work(nbytes, device):
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)


def _quad(q):
    return q if isinstance(q, sfd_freq_quadrature) else sfd_freq_quadrature(*[int(v) for v in q])


def sfd_version():
    return _lib.sfd_version().decode()


def sfd_release_cache():
    _chk(_lib.sfd_release_cache())


def sfd_mesh_icosphere_sizes(level):
    nv, nf, wb = _i64(), _i64(), _sz()
    _chk(_lib.sfd_mesh_icosphere_sizes(int(level), C.byref(nv), C.byref(nf), C.byref(wb)))
    return nv.value, nf.value, wb.value


def sfd_mesh_icosphere(level, device="cuda"):
    """T_level: vertices float64[nV,3], faces int32[nF,3] on `device`."""
    nv, nf, wb = sfd_mesh_icosphere_sizes(level)
    V = torch.empty((nv, 3), dtype=torch.float64, device=device)
    F = torch.empty((nf, 3), dtype=torch.int32, device=device)
    work = _work(wb, device)
    _chk(_lib.sfd_mesh_icosphere(int(level), _ptr(V), _ptr(F), _ptr(work), work.numel(), _stream()))
    return V, F


def sfd_rule_table(rule):
    lam = np.empty((rule, 3), np.float64)
    om = np.empty(rule, np.float64)
    _chk(_lib.sfd_rule_table(int(rule), lam.ctypes.data_as(_vp), om.ctypes.data_as(_vp)))
    return lam, om


def sfd_nodes(V, F, rule):
    """Atoms (x_j, w_j) of the triangle rule on every face: x float64[nF*q,3], w float64[nF*q]."""
    _dev_f64(V, 3)
    assert F.is_cuda and F.dtype == torch.int32 and F.is_contiguous() and F.shape[1] == 3
    J = F.shape[0] * int(rule)
    x = torch.empty((J, 3), dtype=torch.float64, device=V.device)
    w = torch.empty((J,), dtype=torch.float64, device=V.device)
    _chk(_lib.sfd_nodes(_ptr(V), V.shape[0], _ptr(F), F.shape[0], int(rule), _ptr(x), _ptr(w), _stream()))
    return x, w


def sfd_freq_nodes(q, R):
    """Host version of the ball quadrature: numpy xi[K,3], W[K]."""
    q = _quad(q)
    K = q.n_r * q.n_theta * q.n_phi
    xi = np.empty((max(K, 0), 3), np.float64)
    W = np.empty(max(K, 0), np.float64)
    _chk(_lib.sfd_freq_nodes(C.byref(q), float(R), xi.ctypes.data_as(_vp), W.ctypes.data_as(_vp)))
    return xi, W


def sfd_freq_nodes_device(q, R, device="cuda"):
    q = _quad(q)
    wb = _sz()
    _chk(_lib.sfd_freq_nodes_workspace(C.byref(q), C.byref(wb)))
    K = q.n_r * q.n_theta * q.n_phi
    xi = torch.empty((K, 3), dtype=torch.float64, device=device)
    W = torch.empty((K,), dtype=torch.float64, device=device)
    work = _work(wb.value, device)
    _chk(_lib.sfd_freq_nodes_device(C.byref(q), float(R), _ptr(xi), _ptr(W), _ptr(work), work.numel(), _stream()))
    return xi, W


def sfd_freq_nodes_device_range(q, R, a_begin, a_end, device="cuda"):
    """Nodes of the radial shells [a_begin, a_end) of the ball quadrature (a shard of the targets)."""
    q = _quad(q)
    wb = _sz()
    _chk(_lib.sfd_freq_nodes_workspace(C.byref(q), C.byref(wb)))
    K = (int(a_end) - int(a_begin)) * q.n_theta * q.n_phi
    xi = torch.empty((K, 3), dtype=torch.float64, device=device)
    W = torch.empty((K,), dtype=torch.float64, device=device)
    work = _work(wb.value, device)
    _chk(_lib.sfd_freq_nodes_device_range(C.byref(q), float(R), int(a_begin), int(a_end), _ptr(xi), _ptr(W),
                                          _ptr(work), work.numel(), _stream()))
    return xi, W


def sfd_surface_ft_workspace(J, K, X, S, eps):
    wb = _sz()
    Xa = (_dbl * 3)(*[float(v) for v in X]) if X is not None else None
    Sa = (_dbl * 3)(*[float(v) for v in S]) if S is not None else None
    _chk(_lib.sfd_surface_ft_workspace(int(J), int(K), Xa, Sa, float(eps), C.byref(wb)))
    return wb.value


def sfd_surface_ft_plan(J, K, X, S, eps):
    """(w, nf[3], n2[3]) of the type-3 transform for sources / targets of half-widths X / S."""
    w, nf, n2 = C.c_int32(), (_i64 * 3)(), (_i64 * 3)()
    Xa, Sa = (_dbl * 3)(*[float(v) for v in X]), (_dbl * 3)(*[float(v) for v in S])
    _chk(_lib.sfd_surface_ft_plan(int(J), int(K), Xa, Sa, float(eps), C.byref(w), nf, n2))
    return w.value, list(nf), list(n2)


def sfd_extents(pts):
    """(half-widths[3], centre[3]) of the bounding box of device points float64[n,3] (the library's own bounds kernels)."""
    _dev_f64(pts, 3)
    wb = _sz()
    _chk(_lib.sfd_extents_workspace(C.byref(wb)))
    work = _work(wb.value, pts.device)
    half, centre = (_dbl * 3)(), (_dbl * 3)()
    _chk(_lib.sfd_extents(_ptr(pts), pts.shape[0], half, centre, _ptr(work), work.numel(), _stream()))
    return list(half), list(centre)


def _half_widths(t):
    return sfd_extents(t)[0]


def sfd_surface_ft(x, w, xi, eps=0.0, work=None, out=None):
    """nuhat_k = sum_j w_j exp(-i xi_k . x_j): complex128[K].  eps = 0 -> fp64 direct sum; eps > 0 -> type-3 NUFFT."""
    _dev_f64(x, 3), _dev_f64(w), _dev_f64(xi, 3)
    J, K = x.shape[0], xi.shape[0]
    assert w.shape[0] == J
    if work is None:
        if eps > 0 and J > 0 and K > 0:
            wb = sfd_surface_ft_workspace(J, K, _half_widths(x), _half_widths(xi), eps)
        else:
            wb = sfd_surface_ft_workspace(J, K, None, None, 0.0)
        work = _work(wb, x.device)
    nu = out if out is not None else torch.empty((K, 2), dtype=torch.float64, device=x.device)
    _chk(_lib.sfd_surface_ft(_ptr(x), _ptr(w), J, _ptr(xi), K, float(eps), _ptr(nu), _ptr(work), work.numel(),
                             _stream()))
    return torch.view_as_complex(nu) if K > 0 else torch.empty(0, dtype=torch.complex128, device=x.device)


SFD_STATIC_SCRATCH_BYTES = 16 << 20


def sfd_surface_ft_direct_static_scratch(J, K):
    """Bytes of the static scratch array a direct sum of J sources on K targets needs (0: any K fits)."""
    b = _sz()
    _chk(_lib.sfd_surface_ft_direct_static_scratch(int(J), int(K), C.byref(b)))
    return b.value


def sfd_surface_ft_direct_static(x, w, xi, out):
    """The fp64 direct sum without a workspace and without any allocation (include/sfd.h): the caller passes the output
    tensor float64[K][2]; the library's static device array holds the partial sums.  Returns `out` viewed as complex128."""
    _dev_f64(x, 3), _dev_f64(w), _dev_f64(xi, 3), _dev_f64(out, 2)
    J, K = x.shape[0], xi.shape[0]
    assert w.shape[0] == J and out.shape[0] == K
    _chk(_lib.sfd_surface_ft_direct_static(_ptr(x), _ptr(w), J, _ptr(xi), K, _ptr(out), _stream()))
    return torch.view_as_complex(out) if K > 0 else torch.empty(0, dtype=torch.complex128, device=x.device)


def sfd_reduce(nuhat, xi, W, s):
    """I = (2 pi)^-3 sum_k W_k |nuhat_k - sigmahat(xi_k)|^2 (1+|xi_k|^2)^-s (host float)."""
    nu = torch.view_as_real(nuhat) if nuhat.is_complex() else nuhat
    _dev_f64(nu, 2), _dev_f64(xi, 3), _dev_f64(W)
    K = xi.shape[0]
    wb = _sz()
    _chk(_lib.sfd_reduce_workspace(K, C.byref(wb)))
    work = _work(wb.value, xi.device)
    I = _dbl()
    _chk(_lib.sfd_reduce(_ptr(nu), _ptr(xi), _ptr(W), K, float(s), _ptr(work), work.numel(), _stream(), C.byref(I)))
    return I.value


def sfd_weak_distance_workspace(nF, rule, q, R, eps, x_extent=1.0):
    q = _quad(q)
    wb = _sz()
    _chk(_lib.sfd_weak_distance_workspace(int(nF), int(rule), C.byref(q), float(R), float(eps), float(x_extent),
                                          C.byref(wb)))
    return wb.value


def sfd_weak_distance_targets(q):
    """Number of frequency nodes sfd_weak_distance evaluates (the xi_3 >= 0 half of a rule with even n_phi)."""
    k = _i64()
    _chk(_lib.sfd_weak_distance_targets(C.byref(_quad(q)), C.byref(k)))
    return k.value


def sfd_weak_distance(V, F, rule, s, R, q, eps=0.0, work=None, x_extent=None):
    """(sqrt(I), I): the H^{-s} distance between the mesh's surface measure and the unit sphere's."""
    _dev_f64(V, 3)
    assert F.is_cuda and F.dtype == torch.int32 and F.is_contiguous()
    q = _quad(q)
    if work is None:
        if x_extent is None:
            x_extent = max(_half_widths(V)) if eps > 0 else 1.0
        work = _work(sfd_weak_distance_workspace(F.shape[0], rule, q, R, eps, x_extent), V.device)
    d, I = _dbl(), _dbl()
    _chk(_lib.sfd_weak_distance(_ptr(V), V.shape[0], _ptr(F), F.shape[0], int(rule), float(s), float(R), C.byref(q),
                                float(eps), _ptr(work), work.numel(), _stream(), C.byref(d), C.byref(I)))
    return d.value, I.value


def sfd_surface_ft_host(x, w, xi, eps=0.0):
    """End-to-end call on HOST numpy buffers (copies in, runs, copies out)."""
    x = np.ascontiguousarray(x, np.float64).reshape(-1, 3)
    w = np.ascontiguousarray(w, np.float64).reshape(-1)
    xi = np.ascontiguousarray(xi, np.float64).reshape(-1, 3)
    nu = np.empty((len(xi), 2), np.float64)
    _chk(_lib.sfd_surface_ft_host(x.ctypes.data_as(_vp), w.ctypes.data_as(_vp), len(w), xi.ctypes.data_as(_vp),
                                  len(xi), float(eps), nu.ctypes.data_as(_vp)))
    return nu.view(np.complex128).reshape(-1)


def sfd_weak_distance_host(V, F, rule, s, R, q, eps=0.0):
    V = np.ascontiguousarray(V, np.float64).reshape(-1, 3)
    F = np.ascontiguousarray(F, np.int32).reshape(-1, 3)
    q = _quad(q)
    d, I = _dbl(), _dbl()
    _chk(_lib.sfd_weak_distance_host(V.ctypes.data_as(_vp), len(V), F.ctypes.data_as(_vp), len(F), int(rule), float(s),
                                     float(R), C.byref(q), float(eps), C.byref(d), C.byref(I)))
    return d.value, I.value


def sfd_set_profiling(on):
    _chk(_lib.sfd_set_profiling(1 if on else 0))


def sfd_set_grid_precision(bits):
    """32: later transforms of this thread keep their grids in single precision (eps >= 1e-6); 64: fp64."""
    _chk(_lib.sfd_set_grid_precision(int(bits)))


def sfd_last_stage_times():
    names = (C.c_char_p * 32)()
    ms = (C.c_float * 32)()
    n = _lib.sfd_last_stage_times(names, ms, 32)
    return [(names[i].decode(), float(ms[i])) for i in range(n)]


def sfd_launch_count():
    return int(_lib.sfd_launch_count())


def sfd_weak_distance_range_workspace(nF, rule, q, R, a_begin, a_end, eps, x_extent=1.0):
    q = _quad(q)
    wb = _sz()
    _chk(_lib.sfd_weak_distance_range_workspace(int(nF), int(rule), C.byref(q), float(R), int(a_begin), int(a_end),
                                                float(eps), float(x_extent), C.byref(wb)))
    return wb.value


def sfd_weak_distance_range(V, F, rule, s, R, q, a_begin, a_end, eps=0.0, work=None, x_extent=None, out=None):
    """The distance's partial sum over the radial shells [a_begin, a_end) as a DEVICE pair float64[2] = (sum, comp),
    I_shard = sum + comp: a rank's share of a multi-GPU evaluation; nothing crosses to the host."""
    _dev_f64(V, 3)
    assert F.is_cuda and F.dtype == torch.int32 and F.is_contiguous()
    q = _quad(q)
    if work is None:
        if x_extent is None:
            x_extent = max(_half_widths(V)) if eps > 0 else 1.0
        work = _work(sfd_weak_distance_range_workspace(F.shape[0], rule, q, R, a_begin, a_end, eps, x_extent), V.device)
    pair = out if out is not None else torch.empty(2, dtype=torch.float64, device=V.device)
    _chk(_lib.sfd_weak_distance_range(_ptr(V), V.shape[0], _ptr(F), F.shape[0], int(rule), float(s), float(R), C.byref(q),
                                      int(a_begin), int(a_end), float(eps), _ptr(work), work.numel(), _stream(),
                                      _ptr(pair)))
    return pair


# ---- the paper's own variant: cube lattice, trapezoidal rule, its norm convention ---------------------------------
SFD_RULE_GL8X8 = 64


def sfd_lattice_nodes(M, xi_max):
    """Host version of the paper's lattice: numpy xi' = 2 pi xi [K,3], trapezoid weights W[K]."""
    K = max(int(M) + 1, 1) ** 3
    xi = np.empty((K, 3), np.float64)
    W = np.empty(K, np.float64)
    _chk(_lib.sfd_lattice_nodes(int(M), float(xi_max), xi.ctypes.data_as(_vp), W.ctypes.data_as(_vp)))
    return xi, W


def sfd_lattice_nodes_device(M, xi_max, device="cuda"):
    K = (int(M) + 1) ** 3
    xi = torch.empty((K, 3), dtype=torch.float64, device=device)
    W = torch.empty((K,), dtype=torch.float64, device=device)
    _chk(_lib.sfd_lattice_nodes_device(int(M), float(xi_max), _ptr(xi), _ptr(W), _stream()))
    return xi, W


def sfd_reduce_ex(nuhat, xi, W, s, xi_scale, prefactor):
    """prefactor * sum_k W_k |nuhat_k - sigmahat|^2 (1 + (xi_scale |xi_k|)^2)^-s (host float)."""
    nu = torch.view_as_real(nuhat) if nuhat.is_complex() else nuhat
    _dev_f64(nu, 2), _dev_f64(xi, 3), _dev_f64(W)
    K = xi.shape[0]
    wb = _sz()
    _chk(_lib.sfd_reduce_workspace(K, C.byref(wb)))
    work = _work(wb.value, xi.device)
    I = _dbl()
    _chk(_lib.sfd_reduce_ex(_ptr(nu), _ptr(xi), _ptr(W), K, float(s), float(xi_scale), float(prefactor), _ptr(work),
                            work.numel(), _stream(), C.byref(I)))
    return I.value


def sfd_reduce_lattice(nuhat, M, xi_max, s, xi_scale, prefactor):
    """sfd_reduce_ex on the lattice of sfd_lattice_nodes, nodes and weights recomputed from the index (not read)."""
    K = (int(M) + 1) ** 3
    nu = torch.view_as_real(nuhat) if nuhat.is_complex() else nuhat
    _dev_f64(nu, 2)
    assert nu.shape[0] == K
    wb = _sz()
    _chk(_lib.sfd_reduce_workspace(K, C.byref(wb)))
    work = _work(wb.value, nu.device)
    I = _dbl()
    _chk(_lib.sfd_reduce_lattice(_ptr(nu), int(M), float(xi_max), float(s), float(xi_scale), float(prefactor),
                                 _ptr(work), work.numel(), _stream(), C.byref(I)))
    return I.value


def sfd_surface_ft_lattice_workspace(J, M, xi_max, X, eps):
    wb = _sz()
    Xa = (_dbl * 3)(*[float(v) for v in X])
    _chk(_lib.sfd_surface_ft_lattice_workspace(int(J), int(M), float(xi_max), Xa, float(eps), C.byref(wb)))
    return wb.value


def sfd_surface_ft_lattice(x, w, M, xi_max, eps, work=None):
    """nuhat on the lattice of sfd_lattice_nodes (same order): complex128[(M+1)^3].  eps > 0: the paper's type-1
    NUFFT (eq. 3.6); eps = 0 (or a lattice too coarse for the sources): sfd_surface_ft on the expanded nodes."""
    _dev_f64(x, 3), _dev_f64(w)
    J = x.shape[0]
    assert w.shape[0] == J
    if work is None:
        work = _work(sfd_surface_ft_lattice_workspace(J, M, xi_max, _half_widths(x), eps), x.device)
    K = (int(M) + 1) ** 3
    nu = torch.empty((K, 2), dtype=torch.float64, device=x.device)
    _chk(_lib.sfd_surface_ft_lattice(_ptr(x), _ptr(w), J, int(M), float(xi_max), float(eps), _ptr(nu), _ptr(work),
                                     work.numel(), _stream()))
    return torch.view_as_complex(nu)


def sfd_weak_distance_lattice_workspace(nF, rule, M, xi_max, eps, x_extent=1.0):
    wb = _sz()
    _chk(_lib.sfd_weak_distance_lattice_workspace(int(nF), int(rule), int(M), float(xi_max), float(eps),
                                                  float(x_extent), C.byref(wb)))
    return wb.value


def sfd_weak_distance_lattice(V, F, rule, s_paper, xi_max, M, eps=0.0, work=None, x_extent=None):
    """(||mu - sigma||_{H_s}, its square) in the paper's convention (eq. 2.7, s_paper < -1/2) on its lattice."""
    _dev_f64(V, 3)
    assert F.is_cuda and F.dtype == torch.int32 and F.is_contiguous()
    if work is None:
        if x_extent is None:
            x_extent = max(_half_widths(V)) if eps > 0 else 1.0
        work = _work(sfd_weak_distance_lattice_workspace(F.shape[0], rule, M, xi_max, eps, x_extent), V.device)
    d, I = _dbl(), _dbl()
    _chk(_lib.sfd_weak_distance_lattice(_ptr(V), V.shape[0], _ptr(F), F.shape[0], int(rule), float(s_paper),
                                        float(xi_max), int(M), float(eps), _ptr(work), work.numel(), _stream(),
                                        C.byref(d), C.byref(I)))
    return d.value, I.value


def sfd_exact_ft(V, F, xi):
    """Exact transform of the flat mesh, sum over faces of P:128 eq. 2.19 (e^{-i xi.x} convention): complex128[K]."""
    _dev_f64(V, 3), _dev_f64(xi, 3)
    assert F.is_cuda and F.dtype == torch.int32 and F.is_contiguous()
    K = xi.shape[0]
    wb = _sz()
    _chk(_lib.sfd_exact_ft_workspace(F.shape[0], C.byref(wb)))
    work = _work(wb.value, V.device)
    out = torch.empty((K, 2), dtype=torch.float64, device=V.device)
    _chk(_lib.sfd_exact_ft(_ptr(V), V.shape[0], _ptr(F), F.shape[0], _ptr(xi), K, _ptr(out), _ptr(work), work.numel(),
                           _stream()))
    return torch.view_as_complex(out) if K > 0 else torch.empty(0, dtype=torch.complex128, device=V.device)


# ---- two meshes against each other ----------------------------------------------------------------
def sfd_reduce_pair(nuhat_a, nuhat_b, xi, W, s):
    """(2 pi)^-3 sum_k W_k |nuhat_a - nuhat_b|^2 (1+|xi_k|^2)^-s (host float)."""
    na = torch.view_as_real(nuhat_a) if nuhat_a.is_complex() else nuhat_a
    nb = torch.view_as_real(nuhat_b) if nuhat_b.is_complex() else nuhat_b
    _dev_f64(na, 2), _dev_f64(nb, 2), _dev_f64(xi, 3), _dev_f64(W)
    K = xi.shape[0]
    assert na.shape[0] == K and nb.shape[0] == K
    wb = _sz()
    _chk(_lib.sfd_reduce_workspace(K, C.byref(wb)))
    work = _work(wb.value, xi.device)
    I = _dbl()
    _chk(_lib.sfd_reduce_pair(_ptr(na), _ptr(nb), _ptr(xi), _ptr(W), K, float(s), _ptr(work), work.numel(), _stream(),
                              C.byref(I)))
    return I.value


def sfd_mesh_distance_workspace(nFa, nFb, rule, q, R, eps, x_extent=1.0):
    q = _quad(q)
    wb = _sz()
    _chk(_lib.sfd_mesh_distance_workspace(int(nFa), int(nFb), int(rule), C.byref(q), float(R), float(eps), float(x_extent),
                                          C.byref(wb)))
    return wb.value


def sfd_mesh_distance(Va, Fa, Vb, Fb, rule, s, R, q, eps=0.0, work=None, x_extent=None):
    """(sqrt(I), I): H^{-s} distance between the surface measures of two meshes on the ball quadrature (q, R)."""
    _dev_f64(Va, 3), _dev_f64(Vb, 3)
    for F in (Fa, Fb):
        assert F.is_cuda and F.dtype == torch.int32 and F.is_contiguous()
    q = _quad(q)
    if work is None:
        if x_extent is None:
            x_extent = max(_half_widths(Va) + _half_widths(Vb)) if eps > 0 else 1.0
        work = _work(sfd_mesh_distance_workspace(Fa.shape[0], Fb.shape[0], rule, q, R, eps, x_extent), Va.device)
    d, I = _dbl(), _dbl()
    _chk(_lib.sfd_mesh_distance(_ptr(Va), Va.shape[0], _ptr(Fa), Fa.shape[0], _ptr(Vb), Vb.shape[0], _ptr(Fb), Fb.shape[0],
                                int(rule), float(s), float(R), C.byref(q), float(eps), _ptr(work), work.numel(), _stream(),
                                C.byref(d), C.byref(I)))
    return d.value, I.value

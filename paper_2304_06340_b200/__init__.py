"""B200-native hot path of arXiv 2304.06340 (weak distance between S^2 and its triangulations): the Fourier
transform of a triangle-mesh surface measure on a ball-shaped frequency quadrature and the H^{-s} distance to the
unit sphere.  Hand-written CUDA for sm_100a behind the C ABI of include/sfd.h; this package is its ctypes binding.
"""
from .binding import *  # noqa: F401,F403
from .binding import EXPORTS, LIB_PATH, SfdError, sfd_freq_quadrature  # noqa: F401

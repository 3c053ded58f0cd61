"""The polynomial literals pasted into the CUDA sources, checked against mpmath (-m "not gpu").

The sin/cos polynomials of csrc/common.cuh (sincos_fp64) and csrc/direct.cu (c_sc, the direct sum's residual-angle
polynomials) are near-minimax fits computed once at 60 digits and pasted in as decimal literals.  A mistyped digit would
only show up as a slightly larger parity error on the GPU; this test reads the literals out of the source text (it does
not import or run the CUDA path) and evaluates their fp64 Horner forms against sin / cos on the interval each is used on.
"""
import os
import re

import mpmath as mp
import numpy as np

CSRC = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_2304_06340_b200", "csrc")
NUM = r"[-+]?\d+\.?\d*(?:[eE][-+]?\d+)?"


def _exact(f, xs):
    mp.mp.dps = 40
    return np.array([float(f(mp.mpf(float(x)))) for x in xs])


def test_sincos_fp64_literals():
    """common.cuh: sin r = r + r z P(z), cos r = 1 + z Q'(z) with z = r^2 on |r| <= pi/4: both within 1 ulp of 1."""
    src = open(os.path.join(CSRC, "common.cuh")).read()
    body = src[src.index("sincos_fp64(double t"):]
    ps = [float(v) for v in re.findall(r"ps = (?:__fma_rn\(ps, z, )?(" + NUM + r")\)?;", body)]
    pc = [float(v) for v in re.findall(r"pc = (?:__fma_rn\(pc, z, )?(" + NUM + r")\)?;", body)]
    assert len(ps) == 6 and len(pc) == 7, (ps, pc)
    assert ps[-1] == -1.66666666666666640762e-1 and pc[-1] == -0.5
    r = np.linspace(-np.pi / 4, np.pi / 4, 20001)
    z = r * r
    s = np.full_like(r, ps[0])
    for c in ps[1:]:
        s = s * z + c
    s = r * z * s + r
    c_ = np.full_like(r, pc[0])
    for c in pc[1:]:
        c_ = c_ * z + c
    c_ = c_ * z + 1.0
    assert np.abs(s - _exact(mp.sin, r)).max() <= 2.3e-16
    assert np.abs(c_ - _exact(mp.cos, r)).max() <= 2.3e-16
    # the Cody-Waite split of pi/2 (t - n*hi is exact for the n this library meets, lo carries the next 53 bits)
    hi, lo = (float(v) for v in re.findall(r"kPio2(?:Hi|Lo) = (" + NUM + r");", body))
    mp.mp.dps = 50
    assert hi == float(mp.pi / 2) and abs(mp.mpf(hi) + mp.mpf(lo) - mp.pi / 2) < mp.mpf(2) ** -105


def test_direct_sum_table_literals():
    """direct.cu c_sc: with a = 2 pi / 256 and |f| <= 1/2, sin(a f) = f S(f^2) and cos(a f) = C(f^2), three coefficients
    each, stored monic: S(z) = S2 ((z + As) z + Bs), C(z) = C2 ((z + Ac) z + Bc) -- evaluated here in the kernel's order
    (the leading coefficient multiplies the weight first); the last two entries are 1.5 * 2^52 and 256 / (2 pi).
    DESIGN.md 5.2 quotes 1.8e-18 and 2.6e-16."""
    src = open(os.path.join(CSRC, "direct.cu")).read()
    m = re.search(r"c_sc\[8\] = \{(.*?)\};", src, flags=re.S)
    vals = [float(v) for v in re.findall(NUM, re.sub(r"//.*", "", m.group(1)))]
    assert len(vals) == 8, vals
    (As, Bs, S2), (Ac, Bc, C2), magic, scale = vals[0:3], vals[3:6], vals[6], vals[7]
    assert magic == 1.5 * 2.0 ** 52
    mp.mp.dps = 40
    assert scale == float(256 / (2 * mp.pi))
    a = 2 * mp.pi / 256
    f = np.linspace(-0.5, 0.5, 20001)
    z = f * f
    for w in (1.0, 0.731, 3.1e-4):
        s = (w * S2) * (f * ((z + As) * z + Bs))
        c = (w * C2) * ((z + Ac) * z + Bc)
        assert np.abs(s - w * _exact(lambda t: mp.sin(a * t), f)).max() <= 8e-18 * w
        assert np.abs(c - w * _exact(lambda t: mp.cos(a * t), f)).max() <= 7e-16 * w   # the fit as evaluated (2.3e-16) + w C2 + the product + this reference

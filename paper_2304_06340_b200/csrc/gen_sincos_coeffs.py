"""Derives the polynomial coefficients of sincos_fp64 (csrc/common.cuh) and checks them.

    sin r = r + r z P(z),      P of degree 5 in z = r^2,  |r| <= pi/4 (+ a little slack)
    cos r = 1 - z/2 + z^2 Q(z), Q of degree 5

P and Q interpolate (sin(sqrt z)/sqrt z - 1)/z and (cos(sqrt z) - 1 + z/2)/z^2 at the Chebyshev
nodes of [0, zmax] (near-minimax), in 60-digit arithmetic.  Run: python gen_sincos_coeffs.py
The printed constants are pasted into common.cuh; the script then evaluates the fp64 Horner forms
on 200k points against mpmath and prints the worst absolute error.
"""
import mpmath as mp
import numpy as np

mp.mp.dps = 60
RMAX = mp.pi / 4 * mp.mpf("1.02")
ZMAX = RMAX ** 2
DEG = 5


def f_sin(z):
    if z == 0:
        return -mp.mpf(1) / 6
    r = mp.sqrt(z)
    return (mp.sin(r) / r - 1) / z


def f_cos(z):
    if z == 0:
        return mp.mpf(1) / 24
    r = mp.sqrt(z)
    return (mp.cos(r) - 1 + z / 2) / (z * z)


def cheb_interp(f, deg):
    n = deg + 1
    zs = [ZMAX / 2 * (1 + mp.cos(mp.pi * (2 * i + 1) / (2 * n))) for i in range(n)]
    A = mp.matrix(n, n)
    b = mp.matrix(n, 1)
    for i, z in enumerate(zs):
        for j in range(n):
            A[i, j] = z ** j
        b[i] = f(z)
    return list(mp.lu_solve(A, b))


def main():
    P = cheb_interp(f_sin, DEG)
    Q = cheb_interp(f_cos, DEG)
    print("// sin: S1..S6 (ascending powers of z)")
    for c in P:
        print("  %s," % mp.nstr(c, 21))
    print("// cos: C1..C6 (ascending powers of z)")
    for c in Q:
        print("  %s," % mp.nstr(c, 21))
    Pd = [float(c) for c in P]
    Qd = [float(c) for c in Q]
    r = np.linspace(-float(mp.pi / 4), float(mp.pi / 4), 200001)
    z = r * r
    ps = np.full_like(r, Pd[5])
    pc = np.full_like(r, Qd[5])
    for k in range(4, -1, -1):
        ps = ps * z + Pd[k]
        pc = pc * z + Qd[k]
    s = r + (r * z) * ps
    c = 1.0 + z * (z * pc - 0.5)
    es = max(abs(mp.mpf(float(a)) - mp.sin(mp.mpf(float(b)))) for a, b in zip(s[::97], r[::97]))
    ec = max(abs(mp.mpf(float(a)) - mp.cos(mp.mpf(float(b)))) for a, b in zip(c[::97], r[::97]))
    print("max |sin err| = %s, max |cos err| = %s (fp64 Horner without FMA, sampled)" % (mp.nstr(es, 3), mp.nstr(ec, 3)))




# ---------------------------------------------------------------------------------------------
# Quarter-turn form used by the direct sum's inner loop (csrc/direct.cu, sincos_qturn):
#     sin(pi/2 f) = f S(f^2),  cos(pi/2 f) = C(f^2),  |f| <= 1/2,
# S with 6 and C with 7 coefficients (Chebyshev-node interpolants on [0, (0.505)^2]).
# Run: python gen_sincos_coeffs.py qturn
def qturn():
    H = mp.pi / 2
    zmax = (mp.mpf("0.505")) ** 2

    def f_s(z):
        if z == 0:
            return H
        f = mp.sqrt(z)
        return mp.sin(H * f) / f

    def f_c(z):
        return mp.cos(H * mp.sqrt(z))

    def interp(f, n):
        zs = [zmax / 2 * (1 + mp.cos(mp.pi * (2 * i + 1) / (2 * n))) for i in range(n)]
        A = mp.matrix(n, n)
        b = mp.matrix(n, 1)
        for i, z in enumerate(zs):
            for j in range(n):
                A[i, j] = z ** j
            b[i] = f(z)
        return list(mp.lu_solve(A, b))

    S = interp(f_s, 6)
    Cc = interp(f_c, 7)
    print("// S0..S5 (ascending powers of z = f^2)")
    for c in S:
        print("  %s," % mp.nstr(c, 21))
    print("// C0..C6")
    for c in Cc:
        print("  %s," % mp.nstr(c, 21))
    Sd, Cd = [float(c) for c in S], [float(c) for c in Cc]
    f = np.linspace(-0.5, 0.5, 200001)
    z = f * f
    ps = np.full_like(f, Sd[-1])
    for k in range(len(Sd) - 2, -1, -1):
        ps = ps * z + Sd[k]
    pc = np.full_like(f, Cd[-1])
    for k in range(len(Cd) - 2, -1, -1):
        pc = pc * z + Cd[k]
    s = f * ps
    es = max(abs(mp.mpf(float(a)) - mp.sin(H * mp.mpf(float(b)))) for a, b in zip(s[::97], f[::97]))
    ec = max(abs(mp.mpf(float(a)) - mp.cos(H * mp.mpf(float(b)))) for a, b in zip(pc[::97], f[::97]))
    print("qturn: max |sin err| = %s, max |cos err| = %s" % (mp.nstr(es, 3), mp.nstr(ec, 3)))


# ---------------------------------------------------------------------------------------------
# Table form used by the direct sum's inner loop (csrc/direct.cu): the phase is reduced to |f| <= 1/2 in units of
# 1/256 turn (a = 2 pi / 256), the table supplies the multiple of a, and the residual needs
#     sin(a f) = f S(f^2),  cos(a f) = C(f^2)   with 3 coefficients each.
# Run: python gen_sincos_coeffs.py table
def table(ntab=256, ns=3, nc=3):
    a = 2 * mp.pi / ntab
    zmax = mp.mpf("0.2551")

    def f_s(z):
        return a if z == 0 else mp.sin(a * mp.sqrt(z)) / mp.sqrt(z)

    def f_c(z):
        return mp.cos(a * mp.sqrt(z))

    def interp(f, n):
        zs = [zmax / 2 * (1 + mp.cos(mp.pi * (2 * i + 1) / (2 * n))) for i in range(n)]
        A = mp.matrix(n, n)
        b = mp.matrix(n, 1)
        for i, z in enumerate(zs):
            for j in range(n):
                A[i, j] = z ** j
            b[i] = f(z)
        return list(mp.lu_solve(A, b))

    S, Cc = interp(f_s, ns), interp(f_c, nc)
    print("// S%d..S0:" % (ns - 1), ", ".join(mp.nstr(c, 20) for c in S[::-1]))
    print("// C%d..C0:" % (nc - 1), ", ".join(mp.nstr(c, 20) for c in Cc[::-1]))
    print("// ntab / (2 pi) =", mp.nstr(ntab / (2 * mp.pi), 32))
    f = np.linspace(-0.5, 0.5, 20001)
    z = f * f
    ps = np.full_like(f, float(S[-1]))
    for k in range(ns - 2, -1, -1):
        ps = ps * z + float(S[k])
    pc = np.full_like(f, float(Cc[-1]))
    for k in range(nc - 2, -1, -1):
        pc = pc * z + float(Cc[k])
    es = max(abs(mp.mpf(float(x)) - mp.sin(a * mp.mpf(float(y)))) for x, y in zip((f * ps)[::97], f[::97]))
    ec = max(abs(mp.mpf(float(x)) - mp.cos(a * mp.mpf(float(y)))) for x, y in zip(pc[::97], f[::97]))
    print("table %d: max |sin err| = %s, max |cos err| = %s" % (ntab, mp.nstr(es, 3), mp.nstr(ec, 3)))


if __name__ == "__main__":
    import sys
    if "table" in sys.argv:
        table()
    elif "qturn" in sys.argv:
        qturn()
    else:
        main()

#!/usr/bin/env python3
"""Generator for the polynomial coefficients in gw_math.cuh (CUDA path only; the oracle uses libm).

The fused kernel carries the phase in TURNS and reduces it to r in [-1/8, 1/8] (a quarter-turn
quadrant), then needs sin(2 pi r) and cos(2 pi r).  With z = r^2 in [0, 1/64]:

    sin(2 pi r) = r * S(z),   S(z) = sin(2 pi sqrt z)/sqrt z     (degree NS polynomial in z)
    cos(2 pi r) =     C(z),   C(z) = cos(2 pi sqrt z)            (degree NC polynomial in z)

Coefficients: interpolation at Chebyshev nodes of [0, 1/64] in 60-digit arithmetic (within a small
factor of minimax), rounded to fp64; the script prints the maximum absolute error of the ROUNDED
polynomials evaluated in exact arithmetic, which is what the header comment quotes.

Run:  python paper_1904_02863_b200/csrc/gen_sincos_coeffs.py            (prints a C snippet)
"""
import sys

import mpmath as mp

mp.mp.dps = 60
ZMAX = mp.mpf(1) / 64


def S(z):
    if z == 0:
        return 2 * mp.pi
    s = mp.sqrt(z)
    return mp.sin(2 * mp.pi * s) / s


def C(z):
    return mp.cos(2 * mp.pi * mp.sqrt(z))


def cheb_interp(fn, deg):
    n = deg + 1
    nodes = [ZMAX / 2 * (1 + mp.cos(mp.pi * (2 * k + 1) / (2 * n))) for k in range(n)]
    A = mp.matrix(n, n)
    b = mp.matrix(n, 1)
    for i, z in enumerate(nodes):
        for j in range(n):
            A[i, j] = z ** j
        b[i] = fn(z)
    c = mp.lu_solve(A, b)
    return [c[j] for j in range(n)]


def max_err(fn, coef_f64, scale_by_r, n=4001):
    worst = mp.mpf(0)
    for k in range(n):
        r = mp.mpf(k) / (n - 1) / 8
        z = r * r
        p = mp.mpf(0)
        for c in reversed(coef_f64):
            p = p * z + mp.mpf(c)
        e = abs((p - fn(z)) * (r if scale_by_r else 1))
        worst = max(worst, e)
    return worst


def main():
    ns = int(sys.argv[1]) if len(sys.argv) > 1 else 6
    nc = int(sys.argv[2]) if len(sys.argv) > 2 else 7
    s = [float(c) for c in cheb_interp(S, ns)]
    c = [float(x) for x in cheb_interp(C, nc)]
    print(f"/* sin(2 pi r) = r*S(r^2), deg {ns}: max abs err {mp.nstr(max_err(S, s, True), 3)} */")
    for k, v in enumerate(s):
        print(f"#define GW_SIN_S{k} {v!r}  /* {v.hex()} */")
    print(f"/* cos(2 pi r) = C(r^2), deg {nc}: max abs err {mp.nstr(max_err(C, c, False), 3)} */")
    for k, v in enumerate(c):
        print(f"#define GW_COS_C{k} {v!r}  /* {v.hex()} */")


if __name__ == "__main__":
    main()

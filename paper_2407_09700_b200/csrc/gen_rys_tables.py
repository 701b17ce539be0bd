#!/usr/bin/env python3
"""Build step: writes rys_tables.inc (Rys roots/weights data for the CUDA path).  Run once; output is committed.

What is tabulated (Eq. 1, Eq. 3; the paper's `rys_roots<N>()` at PAPER.md:135 is not
specified -- reading R4 in DESIGN.md):  for N = 1..NMAX the N-point Gauss rule

    sum_n w_n f(u_n) = int_0^1 f(t^2) exp(-x t^2) dt      for every polynomial f of degree < 2N,   u_n = t_n^2,

i.e. the rule whose moments are the Boys functions F_m(x), m = 0..2N-1.

* x in [0, XMAX[N]):  on intervals of width 2.5 every u_n(x), w_n(x) is replaced by its degree-13 Chebyshev
  interpolant (14 Chebyshev-Gauss nodes).  Reference values come from Golub-Welsch on the Cholesky factor of the
  Hankel matrix of the moments, in 160-digit mpmath arithmetic.
* x >= XMAX[N]:  u_n = h_n^2 / x, w_n = v_n / sqrt(x) with (h_n, v_n) the positive nodes / weights of the 2N-point
  Gauss-Hermite rule (the [1, inf) tail of the integral is below 1e-14 relative there; checked below).

This file shares nothing with oracle/ (which never uses Rys quadrature).

usage:  python gen_rys_tables.py [--check-only]
"""
from __future__ import annotations

import math
import os
import sys
from multiprocessing import Pool

import mpmath as mp

NMAX = 13   # l <= 6 (h, i functions): N = floor(4*6/2) + 1 = 13 roots for (ii|ii) and for the gradient of (ii|ih)
WIDTH = 2.5
DEG = 13
NCOEF = DEG + 1
# switch to the Gauss-Hermite asymptote; multiples of WIDTH at or above the smallest x where all 2N moments of
# the asymptotic rule agree with F_m(x) to 1e-14 relative for every root and weight (verified by check_asymptote below)
XMAX = {1: 35.0, 2: 45.0, 3: 50.0, 4: 57.5, 5: 62.5, 6: 67.5, 7: 72.5, 8: 77.5, 9: 82.5, 10: 87.5, 11: 92.5, 12: 97.5, 13: 102.5}
DPS = 160
HERE = os.path.dirname(os.path.abspath(__file__))


def boys_moments(nmom: int, x):
    """F_m(x), m < nmom, in the working precision."""
    x = mp.mpf(x)
    if x == 0:
        return [mp.mpf(1) / (2 * m + 1) for m in range(nmom)]
    if x < mp.mpf("1e-3"):
        out = []
        for m in range(nmom):
            s, term, k = mp.mpf(0), mp.mpf(1), 0
            while True:
                add = term / (2 * m + 2 * k + 1)
                s += add
                k += 1
                term *= -x / k
                if abs(add) < mp.mpf(10) ** (-DPS + 5):
                    break
            out.append(s)
        return out
    return [mp.gammainc(m + mp.mpf(1) / 2, 0, x) / (2 * x ** (m + mp.mpf(1) / 2)) for m in range(nmom)]


def gauss_from_moments(N: int, mom):
    """Golub-Welsch: moments m_0..m_2N -> nodes u_n (ascending), weights w_n."""
    M = mp.matrix(N + 1, N + 1)
    for i in range(N + 1):
        for j in range(N + 1):
            M[i, j] = mom[i + j]
    L = mp.cholesky(M)          # M = L L^T, L lower; R = L^T
    R = L.T
    alpha = []
    beta = []
    for j in range(N):
        a = R[j, j + 1] / R[j, j]
        if j > 0:
            a -= R[j - 1, j] / R[j - 1, j - 1]
        alpha.append(a)
        if j + 1 < N:
            beta.append(R[j + 1, j + 1] / R[j, j])
    if N == 1:
        return [alpha[0]], [mom[0]]
    J = mp.matrix(N, N)
    for j in range(N):
        J[j, j] = alpha[j]
        if j + 1 < N:
            J[j, j + 1] = beta[j]
            J[j + 1, j] = beta[j]
    E, Q = mp.eigsy(J)
    order = sorted(range(N), key=lambda k: E[k])
    return [E[k] for k in order], [mom[0] * Q[0, k] ** 2 for k in order]


def rys_exact(N: int, x):
    mp.mp.dps = DPS
    mom = boys_moments(2 * N + 1, x)
    return gauss_from_moments(N, mom)


def hermite_half(N: int):
    """Positive nodes h_n (ascending) and weights v_n of the 2N-point Gauss-Hermite rule."""
    mp.mp.dps = DPS
    n = 2 * N
    J = mp.matrix(n, n)
    for j in range(n - 1):
        b = mp.sqrt(mp.mpf(j + 1) / 2)
        J[j, j + 1] = b
        J[j + 1, j] = b
    E, Q = mp.eigsy(J)
    pairs = sorted((E[k], mp.sqrt(mp.pi) * Q[0, k] ** 2) for k in range(n))
    pos = [(h, v) for (h, v) in pairs if h > 0]
    assert len(pos) == N
    return [h for h, _ in pos], [v for _, v in pos]


def _fit_task(args):
    N, iv = args
    mp.mp.dps = DPS
    lo = WIDTH * iv
    mid, half = lo + WIDTH / 2, WIDTH / 2
    vals = []
    for j in range(NCOEF):
        s = mp.cos(mp.pi * (j + mp.mpf(1) / 2) / NCOEF)
        u, w = rys_exact(N, mid + half * s)
        vals.append(u + w)
    coefs = []  # [value][k]
    for v in range(2 * N):
        ck = []
        for k in range(NCOEF):
            acc = mp.mpf(0)
            for j in range(NCOEF):
                acc += vals[j][v] * mp.cos(mp.pi * k * (j + mp.mpf(1) / 2) / NCOEF)
            acc *= mp.mpf(2) / NCOEF
            if k == 0:
                acc /= 2
            ck.append(float(acc))
        coefs.append(ck)
    return N, iv, coefs


def clenshaw(ck, s):
    b1 = b2 = 0.0
    for k in range(DEG, 0, -1):
        b1, b2 = 2.0 * s * b1 - b2 + ck[k], b1
    return s * b1 - b2 + ck[0]


def _check_task(args):
    N, x, table = args
    mp.mp.dps = DPS
    u, w = rys_exact(N, x)
    iv = min(int(x / WIDTH), len(table) - 1)
    s = (x - (WIDTH * iv + WIDTH / 2)) / (WIDTH / 2)
    err = 0.0
    for v in range(2 * N):
        ref = float(u[v]) if v < N else float(w[v - N])
        got = clenshaw(table[iv][v], s)
        err = max(err, abs(got - ref) / abs(ref))
    return N, x, err


def check_asymptote():
    """Largest relative deviation of the asymptotic rule from the exact one at x = XMAX[N]."""
    out = {}
    for N in range(1, NMAX + 1):
        h, v = hermite_half(N)
        x = mp.mpf(XMAX[N])
        u, w = rys_exact(N, x)
        err = 0.0
        for n in range(N):
            err = max(err, float(abs(h[n] ** 2 / x - u[n]) / u[n]), float(abs(v[n] / mp.sqrt(x) - w[n]) / w[n]))
        out[N] = err
    return out


def main():
    check_only = "--check-only" in sys.argv
    tasks = [(N, iv) for N in range(1, NMAX + 1) for iv in range(int(round(XMAX[N] / WIDTH)))]
    with Pool() as pool:
        res = pool.map(_fit_task, tasks, chunksize=2)
        tables = {N: [None] * int(round(XMAX[N] / WIDTH)) for N in range(1, NMAX + 1)}
        for N, iv, coefs in res:
            tables[N][iv] = coefs
        # accuracy of the fits at points that are not interpolation nodes
        import random
        rnd = random.Random(20240709)
        checks = []
        for N in range(1, NMAX + 1):
            xs = [rnd.uniform(0.0, XMAX[N]) for _ in range(40)] + [1e-9, 1e-3, XMAX[N] - 1e-9] + \
                 [WIDTH * k + d for k in range(1, 4) for d in (-1e-9, 1e-9)]
            checks += [(N, x, tables[N]) for x in xs]
        worst = {}
        for N, x, err in pool.map(_check_task, checks, chunksize=4):
            if err > worst.get(N, (0.0, 0.0))[0]:
                worst[N] = (err, x)
    asym = check_asymptote()
    for N in range(1, NMAX + 1):
        print(f"N={N}: fit max rel err {worst[N][0]:.2e} at x={worst[N][1]:.4f}; asymptote rel err at x={XMAX[N]}: {asym[N]:.2e}")
    if check_only:
        return
    herm = {N: hermite_half(N) for N in range(1, NMAX + 1)}
    lines = ["// GENERATED by gen_rys_tables.py -- do not edit.  See that file for what is tabulated.",
             f"// NMAX={NMAX}, interval width {WIDTH}, Chebyshev degree {DEG}.",
             "// Layout per N: [interval][k = 0..13][value = u_0..u_{N-1}, w_0..w_{N-1}]  (values fastest).",
             f"#define RYS_NMAX {NMAX}", f"#define RYS_NCOEF {NCOEF}", f"#define RYS_WIDTH {WIDTH}"]
    offs, total = [0], 0
    for N in range(1, NMAX + 1):
        offs.append(total)
        total += len(tables[N]) * NCOEF * 2 * N
    lines.append("static const int RYS_TABLE_OFFSET_H[RYS_NMAX + 1] = {" + ", ".join(str(o) for o in offs) + "};")
    lines.append("static const double RYS_XMAX_H[RYS_NMAX + 1] = {0.0, " + ", ".join(repr(XMAX[N]) for N in range(1, NMAX + 1)) + "};")
    lines.append(f"#define RYS_TABLE_SIZE {total}")
    lines.append("static const double RYS_TABLE_H[RYS_TABLE_SIZE] = {")
    for N in range(1, NMAX + 1):
        lines.append(f"// N = {N}")
        for iv in range(len(tables[N])):
            for k in range(NCOEF):
                lines.append(", ".join(float(tables[N][iv][v][k]).hex() for v in range(2 * N)) + ",")
    lines.append("};")
    # Gauss-Hermite data: per N, offset N*(N-1)/2 ... ; h^2 then v
    h2, vv = [], []
    for N in range(1, NMAX + 1):
        h, v = herm[N]
        h2 += [float(a * a).hex() for a in h]
        vv += [float(a).hex() for a in v]
    lines.append(f"static const double RYS_HERM_H2_H[{len(h2)}] = {{" + ", ".join(h2) + "};")
    lines.append(f"static const double RYS_HERM_V_H[{len(vv)}] = {{" + ", ".join(vv) + "};")
    with open(os.path.join(HERE, "rys_tables.inc"), "w") as f:
        f.write("\n".join(lines) + "\n")
    print("wrote rys_tables.inc:", total, "doubles")


if __name__ == "__main__":
    main()

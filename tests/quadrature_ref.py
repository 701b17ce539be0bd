"""Brute-force numerical quadrature of primitive Cartesian ERIs -- an independent pin for the oracle.

Shares no recurrence with McMurchie-Davidson, Obara-Saika or Rys ("higher-l primitive ERIs"):

    1/r12 = (2/sqrt(pi)) int_0^inf exp(-s^2 r12^2) ds,     s^2 = rho t^2/(1-t^2),  ds = sqrt(rho) (1-t^2)^(-3/2) dt

For each s the six-dimensional integrand factorises into three 2-D integrals over (x1,x2) of
polynomial x exp(-(x-m)^T M (x-m) + const), M = [[p+s^2, -s^2], [-s^2, q+s^2]]; each is done exactly by a tensor
Gauss-Hermite rule after a Cholesky change of variables; the t-integral by Gauss-Legendre on [0,1].
"""
import numpy as np

_GH_X, _GH_W = np.polynomial.hermite.hermgauss(14)
_GL_X, _GL_W = np.polynomial.legendre.leggauss(160)
_GL_X = 0.5 * (_GL_X + 1.0)
_GL_W = 0.5 * _GL_W


def _axis_integral(s2, pa, pb, pc, pd, a, b, c, d, A, B, C, D):
    """int int (x1-A)^pa (x1-B)^pb e^{-a(x1-A)^2-b(x1-B)^2} (x2-C)^pc (x2-D)^pd e^{-c(x2-C)^2-d(x2-D)^2} e^{-s2 (x1-x2)^2}"""
    M = np.array([[a + b + s2, -s2], [-s2, c + d + s2]])
    v = np.array([a * A + b * B, c * C + d * D])
    m = np.linalg.solve(M, v)
    const = -(a * A * A + b * B * B + c * C * C + d * D * D) + m @ M @ m
    L = np.linalg.cholesky(M)  # M = L L^T ; y = L^T (x-m)
    Linv_T = np.linalg.inv(L).T
    y1, y2 = np.meshgrid(_GH_X, _GH_X, indexing="ij")
    w = np.outer(_GH_W, _GH_W)
    x1 = m[0] + Linv_T[0, 0] * y1 + Linv_T[0, 1] * y2
    x2 = m[1] + Linv_T[1, 0] * y1 + Linv_T[1, 1] * y2
    poly = (x1 - A) ** pa * (x1 - B) ** pb * (x2 - C) ** pc * (x2 - D) ** pd
    return np.exp(const) * np.sum(w * poly) / np.linalg.det(L)


def prim_eri_quadrature(powers, exps, centres):
    powers = np.asarray(powers)
    a, b, c, d = exps
    A, B, C, D = [np.asarray(x, dtype=float) for x in centres]
    p, q = a + b, c + d
    rho = p * q / (p + q)
    total = 0.0
    for t, wt in zip(_GL_X, _GL_W):
        s2 = rho * t * t / (1.0 - t * t)
        f = 1.0
        for x in range(3):
            f *= _axis_integral(s2, powers[0][x], powers[1][x], powers[2][x], powers[3][x], a, b, c, d,
                                A[x], B[x], C[x], D[x])
        total += wt * f * np.sqrt(rho) * (1.0 - t * t) ** -1.5
    return 2.0 / np.sqrt(np.pi) * total


def cart_powers(l):
    """Cartesian components of a shell in the order of reading R3: lx descending, then ly descending."""
    return [(lx, ly, l - lx - ly) for lx in range(l, -1, -1) for ly in range(l - lx, -1, -1)]


def prim_block_quadrature(ls, exps, centres):
    """The whole Cartesian block [nc_a, nc_b, nc_c, nc_d] of one primitive quartet by the same quadrature: per node t
    the three per-axis tables I[pa, pb, pc, pd] are formed once and every Cartesian component is a product of three
    entries (the integrand factorises), so a block costs 3 * prod(l+1) axis integrals per node instead of 3 per component."""
    la, lb, lc, ld = ls
    a, b, c, d = exps
    A, B, C, D = [np.asarray(x, dtype=float) for x in centres]
    p, q = a + b, c + d
    rho = p * q / (p + q)
    pws = [cart_powers(l) for l in ls]
    out = np.zeros([len(x) for x in pws])
    ia = np.array([[pw[x] for pw in pws[0]] for x in range(3)])
    ib = np.array([[pw[x] for pw in pws[1]] for x in range(3)])
    ic = np.array([[pw[x] for pw in pws[2]] for x in range(3)])
    id_ = np.array([[pw[x] for pw in pws[3]] for x in range(3)])
    for t, wt in zip(_GL_X, _GL_W):
        s2 = rho * t * t / (1.0 - t * t)
        f = 1.0
        for x in range(3):
            tab = np.empty((la + 1, lb + 1, lc + 1, ld + 1))
            for pa in range(la + 1):
                for pb in range(lb + 1):
                    for pc in range(lc + 1):
                        for pd in range(ld + 1):
                            tab[pa, pb, pc, pd] = _axis_integral(s2, pa, pb, pc, pd, a, b, c, d, A[x], B[x], C[x], D[x])
            f = f * tab[ia[x][:, None, None, None], ib[x][None, :, None, None], ic[x][None, None, :, None], id_[x][None, None, None, :]]
        out += wt * f * np.sqrt(rho) * (1.0 - t * t) ** -1.5
    return 2.0 / np.sqrt(np.pi) * out

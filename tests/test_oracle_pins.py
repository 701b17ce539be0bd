"""Pins for the oracle (no GPU): every check ties oracle/ to something other than itself.

What fixes the values (SURVEY.md 8(c) table "What pins each part"):
  * closed forms: F_m(0), F_0 via erf, F_m via the regularised incomplete gamma function, (ss|ss) via erf,
    one-centre (ss|ss) = 2 sqrt(alpha/pi), far-field 1/R;
  * brute-force quadrature (tests/quadrature_ref.py) of primitive ERIs up to g functions;
  * the centre-derivative ladder by central differences;
  * invariants: 8-fold permutational symmetry, translation, Schwarz inequality, J/K symmetry and linearity,
    symmetry-list digestion (reading R9) == plain quadruple loop, gradient sum rules, finite differences of E_J, E_K.
The paper prints no numeric ERI/J/K/gradient value, so there is no tests/golden value of the paper's.
"""
import math

import mpmath
import numpy as np
import pytest
from scipy.special import erf, gamma, gammainc

from paper_2407_09700_b200 import workloads as W
from quadrature_ref import cart_powers, prim_block_quadrature, prim_eri_quadrature


# ------------------------------------------------------------------------------------------------ Boys
def test_boys_at_zero(orc):
    F = orc.boys(25, 0.0)
    assert np.allclose(F, [1.0 / (2 * m + 1) for m in range(26)], rtol=1e-15)


@pytest.mark.parametrize("x", [1e-8, 1e-3, 0.3, 1.0, 4.7, 12.0, 25.0, 34.999, 35.0, 35.001, 50.0, 90.0, 150.0])
def test_boys_incomplete_gamma_and_recursion(orc, x):
    F = orc.boys(25, x)       # m up to 25: (ii|ii) with one raised index
    assert F[0] == pytest.approx(0.5 * math.sqrt(math.pi / x) * erf(math.sqrt(x)), rel=2e-15)
    for m in range(26):
        ref = gamma(m + 0.5) * gammainc(m + 0.5, x) / (2.0 * x ** (m + 0.5))
        if x >= 1e-3:  # gammainc loses relative accuracy for tiny x; covered by the mpmath test
            assert F[m] == pytest.approx(ref, rel=5e-14)
    for m in range(25):  # (2m+1) F_m = 2x F_{m+1} + e^-x
        assert (2 * m + 1) * F[m] == pytest.approx(2 * x * F[m + 1] + math.exp(-x), rel=1e-13)


@pytest.mark.parametrize("x", [1e-8, 0.02, 2.5, 18.0, 33.0, 36.0, 71.0])
def test_boys_mpmath_quadrature(orc, x):
    mpmath.mp.dps = 30
    F = orc.boys(25, x)
    for m in (0, 1, 5, 9, 16, 17, 21, 25):
        ref = mpmath.quad(lambda t: t ** (2 * m) * mpmath.exp(-x * t * t), [0, 1])
        assert F[m] == pytest.approx(float(ref), rel=1e-14)


# ------------------------------------------------------------------------------------------------ (ss|ss)
def _ssss_closed(exps, ctr):
    a, b, c, d = exps
    A, B, C, D = [np.asarray(v, float) for v in ctr]
    p, q = a + b, c + d
    P, Q = (a * A + b * B) / p, (c * C + d * D) / q
    x = p * q / (p + q) * np.sum((P - Q) ** 2)
    F0 = 1.0 if x == 0 else 0.5 * math.sqrt(math.pi / x) * erf(math.sqrt(x))
    return (2 * math.pi ** 2.5 / (p * q * math.sqrt(p + q)) * math.exp(-a * b / p * np.sum((A - B) ** 2))
            * math.exp(-c * d / q * np.sum((C - D) ** 2)) * F0)


def test_ssss_closed_form(orc):
    rng = np.random.default_rng(1)
    z = np.zeros((4, 3), int)
    for _ in range(50):
        ex = np.exp(rng.uniform(math.log(0.05), math.log(50), 4))
        ctr = rng.uniform(-2, 2, (4, 3))
        assert orc.prim_eri(z, ex, ctr) == pytest.approx(_ssss_closed(ex, ctr), rel=1e-14)


def test_ssss_one_centre_and_far_field(orc):
    z = np.zeros((4, 3), int)
    for a in (0.3, 1.0, 7.5):
        N = (2 * a / math.pi) ** 0.75
        assert orc.prim_eri(z, [a] * 4, np.zeros((4, 3))) * N ** 4 == pytest.approx(2 * math.sqrt(a / math.pi), rel=1e-14)
    a, R = 2.0, 40.0
    N = (2 * a / math.pi) ** 0.75
    ctr = np.array([[0, 0, 0], [0, 0, 0], [0, 0, R], [0, 0, R]], float)
    assert orc.prim_eri(z, [a] * 4, ctr) * N ** 4 == pytest.approx(1.0 / R, rel=1e-13)


# ------------------------------------------------------------------------------------------------ higher l vs quadrature
def _rand_powers(rng, l):
    lx = rng.integers(0, l + 1)
    ly = rng.integers(0, l - lx + 1)
    return [lx, ly, l - lx - ly]


@pytest.mark.parametrize("ls", [(1, 0, 0, 0), (1, 1, 0, 0), (1, 0, 1, 0), (1, 1, 1, 1), (2, 0, 0, 0), (2, 1, 1, 0), (2, 2, 1, 1),
                                (2, 2, 2, 2), (3, 0, 2, 1), (3, 3, 1, 0), (3, 3, 3, 3), (4, 0, 0, 0), (4, 2, 3, 1),
                                (4, 4, 2, 2), (4, 4, 4, 4), (0, 2, 0, 3), (1, 4, 2, 4),
                                (5, 0, 0, 0), (6, 0, 1, 0), (5, 5, 0, 0), (6, 2, 5, 1), (6, 6, 6, 6)])
def test_primitive_eri_vs_bruteforce_quadrature(orc, ls):
    rng = np.random.default_rng(100 + sum(ls) * 7 + ls[0])
    for _ in range(3):
        pw = [_rand_powers(rng, l) for l in ls]
        ex = np.exp(rng.uniform(math.log(0.3), math.log(3.0), 4))
        ctr = rng.uniform(-1.0, 1.0, (4, 3))
        ref = prim_eri_quadrature(pw, ex, ctr)
        val = orc.prim_eri(pw, ex, ctr)
        assert val == pytest.approx(ref, rel=2e-11, abs=1e-13 * max(abs(ref), 1e-3))


def test_derivative_ladder(orc):
    """[a+1_x b|cd] = (d/dA_x [ab|cd] + a_x [a-1_x b|cd]) / (2 alpha): ties every l back to lower l."""
    rng = np.random.default_rng(5)
    h = 1e-4
    for la in range(0, 4):
        for trial in range(3):
            pw = np.array([_rand_powers(rng, la), _rand_powers(rng, 2), _rand_powers(rng, 1), _rand_powers(rng, 3)])
            ex = np.exp(rng.uniform(math.log(0.4), math.log(2.5), 4))
            ctr = rng.uniform(-1.0, 1.0, (4, 3))
            x = int(rng.integers(0, 3))
            cp, cm = ctr.copy(), ctr.copy()
            cp[0, x] += h
            cm[0, x] -= h
            dA = (orc.prim_eri(pw, ex, cp) - orc.prim_eri(pw, ex, cm)) / (2 * h)
            up, dn = pw.copy(), pw.copy()
            up[0, x] += 1
            rhs = dA
            if pw[0, x] > 0:
                dn[0, x] -= 1
                rhs += pw[0, x] * orc.prim_eri(dn, ex, ctr)
            assert orc.prim_eri(up, ex, ctr) == pytest.approx(rhs / (2 * ex[0]), rel=2e-7, abs=1e-9)


# ------------------------------------------------------------------------------------------------ c2s / normalisation
def test_c2s_explicit_low_l(orc):
    from oracle import sph
    s3 = math.sqrt(3.0)
    assert np.allclose(sph.c2s(0), [[1 / math.sqrt(4 * math.pi)]], atol=1e-14)
    n1 = math.sqrt(3 / (4 * math.pi))
    assert np.allclose(sph.c2s(1), n1 * np.array([[0, 1, 0], [0, 0, 1], [1, 0, 0]]), atol=1e-14)  # y, z, x
    n2 = math.sqrt(5 / (4 * math.pi))
    # xx,xy,xz,yy,yz,zz ; sqrt3 xy, sqrt3 yz, z^2-(x^2+y^2)/2, sqrt3 xz, sqrt3/2 (x^2-y^2)
    ref = n2 * np.array([[0, s3, 0, 0, 0, 0], [0, 0, 0, 0, s3, 0], [-0.5, 0, 0, -0.5, 0, 1], [0, 0, s3, 0, 0, 0],
                         [s3 / 2, 0, 0, -s3 / 2, 0, 0]])
    assert np.allclose(sph.c2s(2), ref, atol=1e-13)


@pytest.mark.parametrize("l", [0, 1, 2, 3, 4, 5, 6])
def test_c2s_harmonic_orthonormal(orc, l):
    from oracle import sph
    T = sph.c2s(l)
    pw = sph.cart_powers(l)
    # harmonicity: Laplacian of each row polynomial vanishes identically
    for row in T:
        lap = {}
        for coef, (a, b, c) in zip(row, pw):
            for ax, e in enumerate((a, b, c)):
                if e >= 2:
                    key = [a, b, c]
                    key[ax] -= 2
                    lap[tuple(key)] = lap.get(tuple(key), 0.0) + coef * e * (e - 1)
        assert all(abs(v) < 1e-12 for v in lap.values())
    # orthonormality on the unit sphere by an exact product rule (Gauss-Legendre in cos(theta), uniform in phi)
    ct, wt = np.polynomial.legendre.leggauss(12)
    ph = np.arange(24) * 2 * math.pi / 24
    st = np.sqrt(1 - ct ** 2)
    x = np.outer(st, np.cos(ph)).ravel()
    y = np.outer(st, np.sin(ph)).ravel()
    z = np.outer(ct, np.ones_like(ph)).ravel()
    w = np.outer(wt, np.full(24, 2 * math.pi / 24)).ravel()
    mono = np.stack([x ** a * y ** b * z ** c for a, b, c in pw])
    Y = T @ mono
    assert np.allclose((Y * w) @ Y.T, np.eye(2 * l + 1), atol=1e-13)
    # contaminants r^2 * (degree l-2 polynomial) are annihilated by the dual projection
    if l >= 2:
        for a, b, c in sph.cart_powers(l - 2):
            f = (x * x + y * y + z * z) * x ** a * y ** b * z ** c
            assert np.allclose((Y * w) @ f, 0.0, atol=1e-13)


def test_normalise_radial_integral():
    from scipy.integrate import quad
    rng = np.random.default_rng(3)
    for l in range(5):
        e = np.exp(rng.uniform(-2, 3, 4))
        c = W.normalise(l, e, rng.uniform(0.2, 1, 4))
        val, _ = quad(lambda r: r ** (2 * l + 2) * sum(ck * math.exp(-ek * r * r) for ck, ek in zip(c, e)) ** 2, 0, 30,
                      epsabs=1e-14, epsrel=1e-13, limit=400)
        assert val == pytest.approx(1.0, rel=1e-10)


def _one_shell_basis(shells):
    """shells: list of (l, exps, raw coefs, centre); every shell on its own atom"""
    sh, pr, xyz, ao = [], [], [], 0
    for ia, (l, e, c, ctr) in enumerate(shells):
        sh.append((ia, l, len(e), len(pr), ao))
        pr += [(float(ek), float(ck)) for ek, ck in zip(e, c)]
        xyz.append(ctr)
        ao += 2 * l + 1
    return W.Basis(np.array(sh, dtype=W.SHELL_DTYPE), np.array(pr, dtype=W.PRIM_DTYPE), np.array(xyz, dtype=float), ao)


def test_block_quadrature_matches_component_quadrature():
    """the vectorised block quadrature of tests/quadrature_ref.py is the component quadrature that pins prim_eri"""
    rng = np.random.default_rng(31)
    ls = (2, 1, 1, 0)
    ex = np.exp(rng.uniform(math.log(0.3), math.log(3.0), 4))
    ctr = rng.uniform(-1.0, 1.0, (4, 3))
    blk = prim_block_quadrature(ls, ex, ctr)
    pws = [cart_powers(l) for l in ls]
    for idx in [(0, 0, 0, 0), (3, 2, 1, 0), (5, 1, 2, 0), (2, 0, 0, 0)]:
        pw = [pws[k][idx[k]] for k in range(4)]
        assert blk[idx] == pytest.approx(prim_eri_quadrature(pw, ex, ctr), rel=1e-12)


@pytest.mark.parametrize("ls,ks", [((1, 2, 3, 0), (2, 1, 1, 2)), ((2, 2, 1, 1), (1, 2, 2, 1)), ((4, 0, 1, 0), (2, 1, 2, 1)),
                                   ((0, 3, 2, 1), (2, 2, 1, 1)), ((5, 0, 1, 0), (1, 1, 2, 1)), ((1, 6, 0, 0), (2, 1, 1, 1))])
def test_contracted_spherical_block_vs_quadrature(orc, ls, ks):
    """The oracle's contraction (Eq. 5) and its four-index Cartesian -> spherical transform (reading R3) for
    l >= 1: expected block = einsum of brute-force quadrature primitive blocks with the RAW coefficients and the c2s
    matrices, every Cartesian component from tests/quadrature_ref.py (no MD recurrence).  A transposed or mis-ordered
    index in transform_index, a wrong component order or a dropped coefficient fails here; the shells have different l,
    so no index permutation maps the block onto itself."""
    from oracle import sph
    rng = np.random.default_rng(700 + 37 * ls[0] + 11 * ls[1] + 5 * ls[2] + ls[3])
    shells = []
    for l, k in zip(ls, ks):
        e = np.exp(rng.uniform(math.log(0.3), math.log(3.0), k))
        shells.append((l, e, W.normalise(l, e, rng.uniform(0.3, 1.0, k) * rng.choice([-1.0, 1.0], k)), rng.uniform(-1.0, 1.0, 3)))
    b = _one_shell_basis(shells)
    cart = np.zeros([(l + 1) * (l + 2) // 2 for l in ls])
    for ia, (ea, ca) in enumerate(zip(shells[0][1], shells[0][2])):
        for ib, (eb, cb) in enumerate(zip(shells[1][1], shells[1][2])):
            for ic, (ec, cc) in enumerate(zip(shells[2][1], shells[2][2])):
                for id_, (ed, cd) in enumerate(zip(shells[3][1], shells[3][2])):
                    cart += ca * cb * cc * cd * prim_block_quadrature(ls, [ea, eb, ec, ed], [s[3] for s in shells])
    ref = np.einsum("abcd,ia,jb,kc,ld->ijkl", cart, sph.c2s(ls[0]), sph.c2s(ls[1]), sph.c2s(ls[2]), sph.c2s(ls[3]))
    val = orc.eri_block(b, 0, 1, 2, 3)
    assert val.shape == ref.shape
    assert np.abs(val - ref).max() <= 1e-11 * np.abs(ref).max()


@pytest.mark.parametrize("l", [0, 1, 2, 3, 4, 5, 6])
def test_contracted_spherical_shells_are_orthonormal(orc, l):
    """SURVEY 8(c) "c2s matrices" pin: a contracted shell normalised by reading R2 has unit self-overlap and its 2l+1
    functions are orthonormal; the overlap comes from the oracle's E_0 Hermite coefficients, S = E0x E0y E0z (pi/p)^(3/2),
    through the oracle's own index transform.  Two shells of different l on one centre are orthogonal; two displaced s
    shells reproduce the closed-form Gaussian product overlap."""
    rng = np.random.default_rng(900 + l)
    e = np.exp(rng.uniform(-1.5, 2.5, 3))
    c = W.normalise(l, e, rng.uniform(0.2, 1.0, 3))
    l2 = (l + 2) % 7
    e2 = np.exp(rng.uniform(-1.0, 1.0, 2))
    c2 = W.normalise(l2, e2, rng.uniform(0.2, 1.0, 2))
    ctr = rng.uniform(-1, 1, 3)
    b = _one_shell_basis([(l, e, c, ctr), (l2, e2, c2, ctr)])
    assert np.allclose(orc.overlap_block(b, 0, 0), np.eye(2 * l + 1), atol=1e-13)
    assert np.allclose(orc.overlap_block(b, 1, 1), np.eye(2 * l2 + 1), atol=1e-13)
    assert np.allclose(orc.overlap_block(b, 0, 1), 0.0, atol=1e-13)
    if l == 0:
        a1, a2, R = 0.8, 1.7, np.array([0.3, -0.4, 1.1])
        bb = _one_shell_basis([(0, [a1], [1.0], np.zeros(3)), (0, [a2], [1.0], R)])
        ref = (math.pi / (a1 + a2)) ** 1.5 * math.exp(-a1 * a2 / (a1 + a2) * R @ R) / (4 * math.pi)
        assert orc.overlap_block(bb, 0, 1)[0, 0] == pytest.approx(ref, rel=1e-14)


# ------------------------------------------------------------------------------------------------ ERI tensor invariants
@pytest.fixture(scope="module")
def tiny():
    """1 water, TZ-like basis with one s shell contraction cut short: s,p,d,f, contracted and not."""
    b, D = W.water_cluster((1, 1, 1), "tz", 11, "tiny")
    return b, D


def test_eightfold_symmetry_translation_schwarz(orc, tiny):
    b, _ = tiny
    rng = np.random.default_rng(8)
    Q = orc.schwarz(b)
    shifted = b.with_coords(b.coords + np.array([0.37, -1.2, 2.5]))
    for _ in range(25):
        i, j, k, l = rng.integers(0, b.nshell, 4)
        g = orc.eri_block(b, i, j, k, l)
        scale = max(np.abs(g).max(), 1e-8)
        assert np.allclose(g, orc.eri_block(b, j, i, k, l).transpose(1, 0, 2, 3), atol=1e-13 * scale)
        assert np.allclose(g, orc.eri_block(b, i, j, l, k).transpose(0, 1, 3, 2), atol=1e-13 * scale)
        assert np.allclose(g, orc.eri_block(b, k, l, i, j).transpose(2, 3, 0, 1), atol=1e-13 * scale)
        assert np.allclose(g, orc.eri_block(b, l, k, j, i).transpose(3, 2, 1, 0), atol=1e-13 * scale)
        assert np.allclose(g, orc.eri_block(shifted, i, j, k, l), atol=2e-12 * scale)
        assert np.abs(g).max() <= Q[i, j] * Q[k, l] * (1 + 1e-10) + 1e-300
    for i in range(0, b.nshell, 3):
        for j in range(0, b.nshell, 4):
            g = orc.eri_block(b, i, j, i, j)
            ni, nj = g.shape[:2]
            diag = np.array([[g[a, c, a, c] for c in range(nj)] for a in range(ni)])
            assert (diag >= 0).all()
            assert math.sqrt(diag.max()) == pytest.approx(Q[i, j], rel=1e-13)


def test_unit_self_overlap_through_coulomb_limit(orc):
    """A normalised s shell: (chi chi|delta-like) is hard to reach; instead check the shell normalisation through
    the one-centre closed form for a contracted s pair: (ss|ss) = sum c c c c [ss|ss] with the closed-form primitives."""
    rng = np.random.default_rng(21)
    e = np.exp(rng.uniform(-1, 2, 3))
    c = W.normalise(0, e, rng.uniform(0.2, 1, 3))
    sh = np.array([(0, 0, 3, 0, 0)], dtype=W.SHELL_DTYPE)
    pr = np.array(list(zip(e, c)), dtype=W.PRIM_DTYPE)
    b = W.Basis(sh, pr, np.zeros((1, 3)), 1)
    val = orc.eri_block(b, 0, 0, 0, 0)[0, 0, 0, 0]
    ref = 0.0
    for i in range(3):
        for j in range(3):
            for k in range(3):
                for l in range(3):
                    ref += c[i] * c[j] * c[k] * c[l] * _ssss_closed([e[i], e[j], e[k], e[l]], np.zeros((4, 3)))
    assert val == pytest.approx(ref / (4 * math.pi) ** 2, rel=1e-13)  # Y_00 = 1/sqrt(4 pi) per function


# ------------------------------------------------------------------------------------------------ J / K
def test_jk_symmetry_linearity_positivity(orc, tiny):
    b, D = tiny
    J, K, n = orc.jk(b, D)
    assert n == b.nshell ** 4
    s = np.abs(J).max()
    assert np.abs(J - J.T).max() < 1e-13 * s and np.abs(K - K.T).max() < 1e-13 * s
    assert np.sum(D * J) > 0  # Coulomb self-energy of a real density
    rng = np.random.default_rng(2)
    G = rng.standard_normal(D.shape)
    D2 = (G + G.T) / 8
    J2, K2, _ = orc.jk(b, D2)
    J3, K3, _ = orc.jk(b, 0.5 * D - 2.0 * D2)
    assert np.allclose(J3, 0.5 * J - 2.0 * J2, atol=1e-12 * s)
    assert np.allclose(K3, 0.5 * K - 2.0 * K2, atol=1e-12 * s)


def test_jk_equals_definition_from_blocks_and_R9(orc):
    """Plain quadruple loop == explicit einsum over the oracle's own blocks == R9 applied to unique quartets."""
    b, D, _ = W.cfg0()
    n, nao = b.nshell, b.nao
    off = b.shells["ao_off"]
    dim = 2 * b.shells["l"] + 1
    eri = np.zeros((nao,) * 4)
    for i in range(n):
        for j in range(n):
            for k in range(n):
                for l in range(n):
                    eri[off[i]:off[i] + dim[i], off[j]:off[j] + dim[j], off[k]:off[k] + dim[k], off[l]:off[l] + dim[l]] = \
                        orc.eri_block(b, i, j, k, l)
    J, K, _ = orc.jk(b, D)
    s = np.abs(J).max()
    assert np.allclose(J, np.einsum("ijkl,kl->ij", eri, D), atol=1e-13 * s)
    assert np.allclose(K, np.einsum("ijkl,jl->ik", eri, D), atol=1e-13 * s)
    Jt = np.zeros_like(D)
    Kt = np.zeros_like(D)

    def sl(x):
        return slice(off[x], off[x] + dim[x])

    for i in range(n):
        for j in range(i + 1):
            for k in range(i + 1):
                for l in range(k + 1):
                    ij, kl = i * (i + 1) // 2 + j, k * (k + 1) // 2 + l
                    if kl > ij:
                        continue
                    f = (0.5 if i == j else 1.0) * (0.5 if k == l else 1.0) * (0.5 if ij == kl else 1.0)
                    g = f * eri[sl(i), sl(j), sl(k), sl(l)]
                    Jt[sl(i), sl(j)] += np.einsum("abcd,cd->ab", g, D[sl(k), sl(l)])
                    Jt[sl(k), sl(l)] += np.einsum("abcd,ab->cd", g, D[sl(i), sl(j)])
                    Kt[sl(i), sl(k)] += np.einsum("abcd,bd->ac", g, D[sl(j), sl(l)])
                    Kt[sl(i), sl(l)] += np.einsum("abcd,bc->ad", g, D[sl(j), sl(k)])
                    Kt[sl(j), sl(k)] += np.einsum("abcd,ad->bc", g, D[sl(i), sl(l)])
                    Kt[sl(j), sl(l)] += np.einsum("abcd,ac->bd", g, D[sl(i), sl(k)])
    assert np.allclose(2 * (Jt + Jt.T), J, atol=1e-13 * s)
    assert np.allclose(Kt + Kt.T, K, atol=1e-13 * s)


def test_block_modes_and_list_digest(orc, tiny):
    b, D = tiny
    J, K, _ = orc.jk(b, D)
    off, dim = b.shells["ao_off"], 2 * b.shells["l"] + 1
    pairs = [(0, 0), (9, 3), (4, 21), (20, 7), (13, 13)]
    s = np.abs(J).max()
    for (i, j), Jb, Kb in zip(pairs, orc.j_blocks(b, D, pairs), orc.k_blocks(b, D, pairs)):
        assert np.allclose(Jb, J[off[i]:off[i] + dim[i], off[j]:off[j] + dim[j]], atol=1e-13 * s)
        assert np.allclose(Kb, K[off[i]:off[i] + dim[i], off[j]:off[j] + dim[j]], atol=1e-13 * s)
    # screened J/K stays within the parity budget of the unscreened one
    Js, Ks, n = orc.jk(b, D, 1e-13)
    assert n <= b.nshell ** 4
    assert np.abs(Js - J).max() < 1e-11 * s and np.abs(Ks - K).max() < 1e-11 * s
    # explicit list: all ordered quartets listed once gives J̃ = 2J-like sums: Jt = J + J (both updates), Kt = 4 terms
    rng = np.random.default_rng(4)
    q = rng.integers(0, b.nshell, (40, 4)).astype(np.int32)
    Jt, Kt = orc.digest_list(b, D, q)
    Jr, Kr = np.zeros_like(D), np.zeros_like(D)
    for i, j, k, l in q:
        g = orc.eri_block(b, i, j, k, l)
        si, sj, sk, sl_ = [slice(off[x], off[x] + dim[x]) for x in (i, j, k, l)]
        Jr[si, sj] += np.einsum("abcd,cd->ab", g, D[sk, sl_])
        Jr[sk, sl_] += np.einsum("abcd,ab->cd", g, D[si, sj])
        Kr[si, sk] += np.einsum("abcd,bd->ac", g, D[sj, sl_])
        Kr[sj, sl_] += np.einsum("abcd,ac->bd", g, D[si, sk])
        Kr[si, sl_] += np.einsum("abcd,bc->ad", g, D[sj, sk])
        Kr[sj, sk] += np.einsum("abcd,ad->bc", g, D[si, sl_])
    assert np.allclose(Jt, Jr, atol=1e-13 * max(np.abs(Jr).max(), 1e-3))
    assert np.allclose(Kt, Kr, atol=1e-13 * max(np.abs(Jr).max(), 1e-3))


def test_density_weighted_screening_mode_is_the_rule_written_out(orc):
    """oracle.jk_dscreen (Eq. 8-9, PAPER.md:78-89 at shell-group level) == the oracle's own blocks summed over exactly the
    quartets with Q_ij Q_kl min(1, P) >= tau, the rule evaluated here in numpy; a scaled-down density removes quartets."""
    b, D, _ = W.cfg0()
    D = 1e-3 * D
    thr = 1e-3
    n, nao = b.nshell, b.nao
    off, dim = b.shells["ao_off"], 2 * b.shells["l"] + 1
    g = orc.shell_groups(b)
    assert list(g) == [0 if l == 0 else 1 for l in b.shells["l"]]
    Q = orc.schwarz(b)
    ng = g.max() + 1
    Pg = np.zeros((ng, ng))
    for i in range(n):
        for j in range(n):
            Pg[g[i], g[j]] = max(Pg[g[i], g[j]], np.abs(D[off[i]:off[i] + dim[i], off[j]:off[j] + dim[j]]).max())
    J, K = np.zeros_like(D), np.zeros_like(D)
    kept = 0
    for i in range(n):
        for j in range(n):
            for k in range(n):
                for l in range(n):
                    gs = [g[i], g[j], g[k], g[l]]
                    P = min(1.0, max(Pg[gs[x], gs[y]] for x in range(4) for y in range(4) if x != y))
                    if Q[i, j] * Q[k, l] * P < thr:
                        continue
                    kept += 1
                    blk = orc.eri_block(b, i, j, k, l)
                    si, sj, sk, sl = [slice(off[x], off[x] + dim[x]) for x in (i, j, k, l)]
                    J[si, sj] += np.einsum("abcd,cd->ab", blk, D[sk, sl])
                    K[si, sk] += np.einsum("abcd,bd->ac", blk, D[sj, sl])
    Jd, Kd, nd = orc.jk_dscreen(b, D, thr)
    _, _, ns = orc.jk(b, D, thr)
    assert nd == kept and kept < ns < n ** 4
    assert np.allclose(Jd, J, atol=1e-14 * np.abs(J).max()) and np.allclose(Kd, K, atol=1e-14 * np.abs(J).max())


# ------------------------------------------------------------------------------------------------ gradient
def test_eri_derivative_block_vs_finite_difference(orc):
    b, D, _ = W.cfg0()
    h = 1e-4
    rng = np.random.default_rng(6)
    for _ in range(6):
        i = int(rng.integers(0, b.nshell))
        others = [s for s in range(b.nshell) if b.shells["atom"][s] != b.shells["atom"][i]]
        j, k, l = rng.choice(others, 3)
        dg = orc.eri_block(b, i, j, k, l, deriv=True)
        for x in range(3):
            cp, cm = b.coords.copy(), b.coords.copy()
            cp[b.shells["atom"][i], x] += h
            cm[b.shells["atom"][i], x] -= h
            fd = (orc.eri_block(b.with_coords(cp), i, j, k, l) - orc.eri_block(b.with_coords(cm), i, j, k, l)) / (2 * h)
            assert np.allclose(dg[x], fd, rtol=1e-6, atol=1e-8 * max(np.abs(fd).max(), 1e-6))


def test_gradient_translational_invariance_and_fd_of_energy(orc, tiny):
    b, D = tiny
    gJ, gK = orc.jk_grad(b, D)
    assert np.abs(gJ.sum(0)).max() < 1e-10 * np.abs(gJ).max()
    assert np.abs(gK.sum(0)).max() < 1e-10 * np.abs(gK).max()
    for h, tol in ((1e-4, 1e-6), (2e-4, 4e-6)):
        for atom, x in ((0, 0), (0, 2), (1, 1), (2, 0)):
            cp, cm = b.coords.copy(), b.coords.copy()
            cp[atom, x] += h
            cm[atom, x] -= h
            EJp, EKp = orc.energy(b.with_coords(cp), D)
            EJm, EKm = orc.energy(b.with_coords(cm), D)
            assert (EJp - EJm) / (2 * h) == pytest.approx(gJ[atom, x], abs=tol * np.abs(gJ).max())
            assert (EKp - EKm) / (2 * h) == pytest.approx(gK[atom, x], abs=tol * np.abs(gK).max())
    # row mode == rows of the full gradient
    rJ, rK = orc.jk_grad(b, D, atoms=[1])
    assert np.allclose(rJ[1], gJ[1], rtol=1e-13) and np.allclose(rK[1], gK[1], rtol=1e-13)
    assert np.all(rJ[[0, 2]] == 0)

"""Parity of the CUDA path (through the C ABI of include/eri.h) against the CPU oracle on the same seeded inputs.

Tolerances are BASELINE.json's: max|dJ|, max|dK| <= 1e-10 * max|J|; gradient |d| <= 1e-8 Hartree/Bohr.
ERI blocks are compared at 1e-11 of the largest integral of the test (four to five digits tighter than J/K need).
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_2407_09700_b200 import workloads as W  # noqa: E402

JK_TOL = 1e-10
GRAD_TOL = 1e-8


@pytest.fixture(scope="module")
def eri():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2407_09700_b200 import eri as E
    E.lib()
    return E


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def mixed_basis(seed=7, K=2, lmax=4, ncentre=4):
    """Shells l = 0..lmax on `ncentre` random centres in a 3 Bohr box, K primitives each (cfg1-like exponents)."""
    rng = np.random.default_rng(seed)
    coords = rng.uniform(0.0, 3.0, (ncentre, 3))
    atom_shells = [[] for _ in range(ncentre)]
    for l in range(lmax + 1):
        for c in range(ncentre):
            e = np.sort(np.exp(rng.uniform(math.log(0.2), math.log(8.0), K)))[::-1].copy()
            atom_shells[c].append((l, e, W.normalise(l, e, rng.uniform(0.2, 1.0, K))))
    return W._assemble(atom_shells, coords, {"name": "mixed"})


# ----------------------------------------------------------------------------------------------- Rys data
def test_rys_moment_identity(eri, orc):
    """sum_n w_n u_n^m = F_m(x), m < 2N (definition of the rule) with F_m from the oracle's Boys function."""
    rng = np.random.default_rng(1)
    for N in range(1, 14):
        xmax = [0, 35.0, 45.0, 50.0, 57.5, 62.5, 67.5, 72.5, 77.5, 82.5, 87.5, 92.5, 97.5, 102.5][N]
        xs = np.concatenate([rng.uniform(0, xmax, 200), [0.0, 1e-12, 2.5 - 1e-12, 2.5, 2.5 + 1e-12, xmax - 1e-9, xmax, xmax + 1e-9],
                             np.exp(rng.uniform(math.log(xmax), math.log(5e4), 50))])
        u, w = eri.eri_rys_roots(N, xs)
        assert np.all(u > 0) and np.all(u < 1) and np.all(w > 0)
        for i, x in enumerate(xs):
            F = orc.boys(2 * N - 1, float(x))
            mom = np.array([np.sum(w[i] * u[i] ** m) for m in range(2 * N)])
            assert np.max(np.abs(mom - F) / F) < 2e-12, (N, x)


# ----------------------------------------------------------------------------------------------- ERI blocks
def test_eri_blocks_cfg0_all_unique_and_permuted(eri, orc):
    basis, D, thr = W.cfg0()
    n = basis.nshell
    quartets = [(i, j, k, l) for i in range(n) for j in range(i + 1) for k in range(i + 1) for l in range(k + 1)
                if k * (k + 1) // 2 + l <= i * (i + 1) // 2 + j]
    assert len(quartets) == 1540
    rng = np.random.default_rng(3)
    quartets += [tuple(rng.integers(0, n, 4)) for _ in range(200)]   # any order of shells
    got = eri.eri_compute_quartets(basis, quartets)
    ref = [orc.eri_block(basis, *q) for q in quartets]
    scale = max(np.abs(r).max() for r in ref)
    for q, g, r in zip(quartets, got, ref):
        assert np.abs(g - r).max() <= 1e-11 * scale, q


def test_eri_blocks_up_to_g(eri, orc):
    basis = mixed_basis()
    ls = basis.shells["l"]
    rng = np.random.default_rng(11)
    n = basis.nshell
    quartets = [tuple(rng.integers(0, n, 4)) for _ in range(60)]
    # make sure the heaviest classes are present
    g = [s for s in range(n) if ls[s] == 4]
    f = [s for s in range(n) if ls[s] == 3]
    quartets += [(g[0], g[1], g[2], g[3]), (g[0], g[0], g[0], g[0]), (f[0], f[1], f[2], f[3]), (g[0], f[1], f[2], g[3]), (f[0], g[1], 0, g[2])]
    got = eri.eri_compute_quartets(basis, quartets)
    ref = [orc.eri_block(basis, *q) for q in quartets]
    scale = max(np.abs(r).max() for r in ref)
    for q, a, r in zip(quartets, got, ref):
        assert np.abs(a - r).max() <= 1e-11 * scale, (q, [int(ls[s]) for s in q])


def test_schwarz_matches_oracle(eri, orc):
    basis, D, thr = W.cfg0()
    Q = eri.eri_schwarz(basis)
    Qo = orc.schwarz(basis)
    assert np.abs(Q - Qo).max() <= 1e-11 * Qo.max()


def test_c2s_table_matches_oracle(eri):
    import oracle.sph as sph
    for l in range(7):
        assert np.abs(eri.eri_c2s_matrix(l) - sph.c2s(l)).max() < 1e-13


# ----------------------------------------------------------------------------------------------- J/K
def _jk_parity(eri, orc, basis, D, thr, kernel_mode=0):
    plan = eri.eri_plan_create(basis, thr)
    plan.set_kernel_mode(kernel_mode)
    J, K = plan.build_jk(dev(D))
    J, K = J.cpu().numpy(), K.cpu().numpy()
    Jo, Ko, _ = orc.jk(basis, D, 0.0)
    scale = np.abs(Jo).max()
    assert np.abs(J - J.T).max() <= 1e-13 * scale and np.abs(K - K.T).max() <= 1e-13 * scale
    assert np.abs(J - Jo).max() <= JK_TOL * scale
    assert np.abs(K - Ko).max() <= JK_TOL * scale
    return plan


@pytest.mark.parametrize("mode", [0, 1])
def test_jk_cfg0(eri, orc, mode):
    basis, D, thr = W.cfg0()
    plan = _jk_parity(eri, orc, basis, D, thr, mode)
    st = plan.stats()
    assert st["quartets_kept"] == 1540 and st["pairs_kept"] == 55


def test_jk_one_shot_cfg0(eri, orc):
    basis, D, thr = W.cfg0()
    J, K = eri.eri_build_jk(basis, dev(D), thr)
    Jo, Ko, _ = orc.jk(basis, D, 0.0)
    scale = np.abs(Jo).max()
    assert np.abs(J.cpu().numpy() - Jo).max() <= JK_TOL * scale and np.abs(K.cpu().numpy() - Ko).max() <= JK_TOL * scale


@pytest.mark.parametrize("mode", [0, 1])
def test_jk_two_water_tz_with_f_and_k8(eri, orc, mode):
    basis, D = W.water_cluster((1, 1, 2), "tz", 77, "tz2")
    _jk_parity(eri, orc, basis, D, 1e-13, mode)


def test_jk_mixed_up_to_g(eri, orc):
    basis = mixed_basis(seed=5, K=1, lmax=4, ncentre=2)
    rng = np.random.default_rng(2)
    C = rng.standard_normal((basis.nao, 6)) / math.sqrt(basis.nao)
    _jk_parity(eri, orc, basis, C @ C.T, 0.0)


def test_jk_cfg2_full(eri, orc):
    basis, D, thr = W.cfg2()
    plan = _jk_parity(eri, orc, basis, D, thr)
    st = plan.stats()
    assert st["nao"] == 192 and st["pairs_total"] == 4656 and st["quartets_total"] == 4656 * 4657 // 2
    # host-buffer entry point gives the same result
    J, K = plan.build_jk(dev(D))
    Jh, Kh = np.empty_like(D), np.empty_like(D)
    plan.build_jk_host(D, Jh, Kh)
    assert np.abs(Jh - J.cpu().numpy()).max() <= 1e-12 * np.abs(Jh).max()
    assert np.abs(Kh - K.cpu().numpy()).max() <= 1e-12 * np.abs(Jh).max()


def test_screening_equals_oracle_same_screening(eri, orc):
    """A loose threshold drops real work; the GPU list must reproduce the oracle's 'same screening' mode (reading R7)."""
    basis, D = W.water_cluster((1, 2, 2), "dzp", 31, "dzp4")
    thr = 1e-6
    plan = eri.eri_plan_create(basis, thr)
    J, K = plan.build_jk(dev(D))
    Jo, Ko, nq = orc.jk(basis, D, thr)
    scale = np.abs(Jo).max()
    assert np.abs(J.cpu().numpy() - Jo).max() <= 1e-9 * scale    # pairs within rounding of the threshold may differ
    assert np.abs(K.cpu().numpy() - Ko).max() <= 1e-9 * scale
    st = plan.stats()
    assert st["quartets_kept"] < st["quartets_total"]


def test_density_weighted_screening_equals_oracle_rule(eri, orc):
    """SURVEY 8(f) NEXT-1 (Eq. 8-9, Alg. 1 lines 12-16): eri_plan_build_jk_dscreen evaluates exactly the quartets
    with Q_ij Q_kl min(1, P_{ab|cd}) >= tau, P from the density itself; the oracle's jk_dscreen applies the same rule to its
    plain quadruple loop.  A small "delta-D" (an SCF-like density change) removes most of the list."""
    basis, D = W.water_cluster((1, 2, 2), "dzp", 31, "dzp4")
    thr = 1e-6
    plan = eri.eri_plan_create(basis, thr)
    nk = plan.stats()["quartets_kept"]
    rng = np.random.default_rng(12)
    G = rng.standard_normal(D.shape)
    for name, M in (("D", D), ("deltaD", 1e-3 * np.abs(D).max() * 0.5 * (G + G.T))):
        for mode in (0, 2, 1):                                      # tile + register + cooperative, no tile family, generic
            plan.set_kernel_mode(mode)
            J, K = plan.build_jk_dens(dev(M))
            kept = plan.dens_quartets()
            Jo, Ko, _ = orc.jk_dscreen(basis, M, thr)
            scale = np.abs(Jo).max()
            assert np.abs(J.cpu().numpy() - Jo).max() <= 1e-9 * scale, (name, mode)   # pairs within rounding of the threshold may differ
            assert np.abs(K.cpu().numpy() - Ko).max() <= 1e-9 * scale, (name, mode)
            assert 0 < kept <= nk
            if name == "deltaD":
                assert kept < 0.7 * nk, (kept, nk)                 # the density factor did remove work
                Ju, Ku, _ = orc.jk(basis, M, 0.0)                   # and the result is still the J/K of delta-D within the screening error
                assert np.abs(J.cpu().numpy() - Ju).max() <= 1e-3 * np.abs(Ju).max()
    plan.set_kernel_mode(0)
    # the plain build is unchanged by the density-weighted calls before it
    J, K = plan.build_jk(dev(D))
    Jo, Ko, _ = orc.jk(basis, D, thr)
    assert np.abs(J.cpu().numpy() - Jo).max() <= 1e-9 * np.abs(Jo).max()


# ----------------------------------------------------------------------------------------------- cfg1 lists
CFG1_CASES = [((0, 0, 0, 0), 1, 256), ((1, 0, 0, 0), 3, 256), ((1, 1, 1, 1), 3, 128), ((2, 1, 1, 1), 1, 128),
              ((2, 2, 2, 2), 1, 64), ((3, 3, 3, 3), 1, 16), ((3, 2, 1, 0), 6, 32), ((4, 4, 3, 3), 1, 8), ((4, 4, 4, 4), 1, 4),
              ((4, 3, 2, 1), 3, 8), ((2, 0, 1, 0), 6, 64), ((3, 0, 0, 0), 1, 128), ((4, 0, 4, 0), 3, 16)]


@pytest.mark.parametrize("cls,K,n", CFG1_CASES)
def test_cfg1_list_digest(eri, orc, cls, K, n):
    basis, D, q = W.cfg1_class(cls, K, nquartets=n)
    Jt, Kt = eri.eri_digest_quartet_list(basis, q, dev(D))
    Jo, Ko = orc.digest_list(basis, D, q)
    scale = max(np.abs(Jo).max(), np.abs(Ko).max(), 1e-300)
    assert np.abs(Jt.cpu().numpy() - Jo).max() <= JK_TOL * scale
    assert np.abs(Kt.cpu().numpy() - Ko).max() <= JK_TOL * scale
    # digesting the list in two halves and adding gives the same result (linearity in the list)
    h = n // 2
    J1, K1 = eri.eri_digest_quartet_list(basis, q[:h], dev(D))
    J2, K2 = eri.eri_digest_quartet_list(basis, q[h:], dev(D))
    assert (J1 + J2 - Jt).abs().max().item() <= 1e-12 * scale


# ----------------------------------------------------------------------------------------------- gradient
def _grad_parity(eri, orc, basis, D, thr):
    gJ, gK = eri.eri_jk_grad(basis, dev(D), thr)
    gJ, gK = gJ.cpu().numpy(), gK.cpu().numpy()
    gJo, gKo = orc.jk_grad(basis, D)
    assert np.abs(gJ.sum(axis=0)).max() <= 1e-10 and np.abs(gK.sum(axis=0)).max() <= 1e-10   # translational invariance
    assert np.abs(gJ - gJo).max() <= GRAD_TOL
    assert np.abs(gK - gKo).max() <= GRAD_TOL


def test_grad_cfg0(eri, orc):
    basis, D, thr = W.cfg0()
    _grad_parity(eri, orc, basis, D, thr)


def test_grad_two_water_dzp(eri, orc):
    basis, D = W.water_cluster((1, 1, 2), "dzp", 5, "dzp2")
    _grad_parity(eri, orc, basis, D, 1e-13)


def test_grad_one_water_tz(eri, orc):
    basis, D = W.water_cluster((1, 1, 1), "tz", 9, "tz1")
    _grad_parity(eri, orc, basis, D, 1e-13)


def test_grad_mixed_up_to_g(eri, orc):
    basis = mixed_basis(seed=15, K=1, lmax=4, ncentre=2)
    rng = np.random.default_rng(4)
    C = rng.standard_normal((basis.nao, 6)) / math.sqrt(basis.nao)
    D = C @ C.T
    _grad_parity(eri, orc, basis, D, 0.0)
    # kernel mode 2 (no tile family): every class that has a cooperative gradient kernel runs on it, all 120 classes occur here
    plan = eri.eri_plan_create(basis, 0.0, want_grad=True)
    plan.set_kernel_mode(2)
    assert {c["kernel_grad"] for c in plan.class_stats()} <= {0, 2}
    gJ, gK = plan.jk_grad(dev(D))
    gJo, gKo = orc.jk_grad(basis, D)
    assert np.abs(gJ.cpu().numpy() - gJo).max() <= GRAD_TOL and np.abs(gK.cpu().numpy() - gKo).max() <= GRAD_TOL


def test_grad_finite_difference_of_gpu_energy(eri):
    """Central differences (h = 1e-4 Bohr) of E_J, E_K from GPU J/K builds against the GPU gradient (reading R13)."""
    basis, D = W.water_cluster((1, 1, 2), "dzp", 5, "dzp2")
    Dd = dev(D)
    gJ, gK = eri.eri_jk_grad(basis, Dd, 0.0)
    h = 1e-4
    for atom, ax in [(0, 0), (1, 2), (4, 1)]:
        e = []
        for sgn in (+1, -1):
            xyz = basis.coords.copy()
            xyz[atom, ax] += sgn * h
            J, K = eri.eri_build_jk(basis.with_coords(xyz), Dd, 0.0)
            e.append((0.5 * (Dd * J).sum().item(), 0.5 * (Dd * K).sum().item()))
        fdJ, fdK = (e[0][0] - e[1][0]) / (2 * h), (e[0][1] - e[1][1]) / (2 * h)
        scale = max(gJ.abs().max().item(), gK.abs().max().item())
        assert abs(fdJ - gJ[atom, ax].item()) <= 1e-6 * scale
        assert abs(fdK - gK[atom, ax].item()) <= 1e-6 * scale


# ----------------------------------------------------------------------------------------------- h and i functions
def hi_basis(seed=41, ncentre=3):
    """shells l = 0..6 (s..i) spread over `ncentre` centres in a 3 Bohr box, one primitive each, two for p and h"""
    rng = np.random.default_rng(seed)
    coords = rng.uniform(0.0, 3.0, (ncentre, 3))
    atom_shells = [[] for _ in range(ncentre)]
    for l in range(7):
        K = 2 if l in (1, 5) else 1
        e = np.sort(np.exp(rng.uniform(math.log(0.4), math.log(2.5), K)))[::-1].copy()
        atom_shells[l % ncentre].append((l, e, W.normalise(l, e, rng.uniform(0.3, 1.0, K))))
    return W._assemble(atom_shells, coords, {"name": "hi"})


def test_eri_blocks_with_h_and_i_shells(eri, orc):
    """The paper stops at g because its 2-D integrals overflow per-thread local memory; here l = 5, 6 run on the
    generic kernels (N up to 13 roots) and must match the oracle like every other class."""
    basis = hi_basis()
    ls = basis.shells["l"]
    h, i6 = int(np.where(ls == 5)[0][0]), int(np.where(ls == 6)[0][0])
    quartets = [(h, 0, 0, 0), (i6, 0, 0, 0), (h, 1, 2, 0), (i6, 2, 1, 1), (h, h, 0, 0), (i6, 3, h, 1), (h, i6, 4, 2), (i6, i6, 0, 0),
                (0, h, i6, 1), (i6, h, i6, h), (h, h, h, h)]
    got = eri.eri_compute_quartets(basis, quartets)
    ref = [orc.eri_block(basis, *q) for q in quartets]
    for q, a, r in zip(quartets, got, ref):
        assert np.abs(a - r).max() <= 1e-11 * max(np.abs(r).max(), 1e-3), (q, [int(ls[s]) for s in q])


def test_jk_and_gradient_with_h_and_i_shells(eri, orc):
    basis = hi_basis(seed=43)
    rng = np.random.default_rng(6)
    C = rng.standard_normal((basis.nao, 6)) / math.sqrt(basis.nao)
    D = C @ C.T
    _jk_parity(eri, orc, basis, D, 0.0)
    # explicit lists of h/i classes (cfg1 recipe)
    ls = basis.shells["l"]
    h, i6, s0, p1 = (int(np.where(ls == l)[0][0]) for l in (5, 6, 0, 1))
    q = np.array([(h, s0, s0, s0), (i6, p1, h, s0), (i6, i6, s0, s0), (h, h, p1, p1)], dtype=np.int32)
    Jt, Kt = eri.eri_digest_quartet_list(basis, q, dev(D))
    Jo, Ko = orc.digest_list(basis, D, q)
    scale = max(np.abs(Jo).max(), np.abs(Ko).max())
    assert np.abs(Jt.cpu().numpy() - Jo).max() <= JK_TOL * scale and np.abs(Kt.cpu().numpy() - Ko).max() <= JK_TOL * scale
    # gradient: a smaller set (s, p, h, i on three centres) keeps the oracle to seconds
    keep = np.isin(ls, (0, 1, 5, 6))
    sub = W._assemble([[(int(basis.shells["l"][s]), basis.prims["exp"][basis.shells["prim_off"][s]:basis.shells["prim_off"][s] + basis.shells["nprim"][s]],
                         basis.prims["coef"][basis.shells["prim_off"][s]:basis.shells["prim_off"][s] + basis.shells["nprim"][s]])
                        for s in range(basis.nshell) if keep[s] and basis.shells["atom"][s] == a] for a in range(basis.natm)], basis.coords, {})
    C = rng.standard_normal((sub.nao, 5)) / math.sqrt(sub.nao)
    _grad_parity(eri, orc, sub, C @ C.T, 0.0)


# ----------------------------------------------------------------------------------------------- edge cases
def test_edge_cases(eri, orc):
    basis, D, thr = W.cfg0()
    # threshold above every bound: nothing survives, J = K = 0
    plan = eri.eri_plan_create(basis, 1e6)
    J, K = plan.build_jk(dev(D))
    assert J.abs().max().item() == 0.0 and K.abs().max().item() == 0.0 and plan.stats()["quartets_kept"] == 0
    # a single s shell
    one = W._assemble([[(0, np.array([1.0]), W.normalise(0, np.array([1.0]), np.array([1.0])))]], np.zeros((1, 3)), {})
    J, K = eri.eri_build_jk(one, dev(np.ones((1, 1))), 0.0)
    assert abs(J.item() - 2.0 * math.sqrt(1.0 / math.pi)) < 1e-13 and abs(K.item() - J.item()) < 1e-15   # (ss|ss) = 2 sqrt(alpha/pi)
    # empty list
    assert eri.eri_compute_quartets(basis, np.zeros((0, 4), dtype=np.int32)) == []
    # error paths
    bad = W.Basis(basis.shells.copy(), basis.prims.copy(), basis.coords.copy(), basis.nao)
    bad.shells["l"][0] = 7
    with pytest.raises(eri.EriError, match="angular momentum"):
        eri.eri_plan_create(bad, 0.0)
    bad.shells["l"][0] = 0
    bad.shells["ao_off"][3] += 1
    with pytest.raises(eri.EriError, match="bad argument"):
        eri.eri_plan_create(bad, 0.0)

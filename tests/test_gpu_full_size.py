"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (SURVEY.md 8(c) "parity procedure").

cfg3 (32 waters, 1856 functions): the unscreened oracle is hours, so the full GPU J/K build is compared on seeded
samples of J and K shell-pair blocks that the oracle computes one by one (block mode: each block is summed over ALL
(k,l) resp. (j,l) with no screening), covering every (l_i, l_j) combination and the K = 8 core shells; plus the
properties that hold at any size (symmetry, agreement of the three kernel selections, agreement of the concurrent and
the serialised launch schedule).
cfg4 (16 waters, 928 functions, gradient): per-axis sums over atoms = 0 (translational invariance) and
central differences (h = 1e-4 Bohr, BASELINE.json) of the GPU J/K energies on one O and one H atom; the gradient
arithmetic itself is compared with the oracle on a 2-water cluster with the same basis (f shells, K = 8).
"""
import numpy as np
import pytest

from paper_2407_09700_b200 import workloads as W

pytestmark = pytest.mark.gpu
JK_TOL = 1e-10      # BASELINE.json north_star: max|dJ|, |dK| <= 1e-10 max|J|
GRAD_TOL = 1e-8     # Hartree/Bohr


@pytest.fixture(scope="module")
def eri():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2407_09700_b200 import eri as E
    return E


@pytest.fixture(scope="module")
def orc():
    import oracle
    oracle.build()
    return oracle


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.fixture(scope="module")
def cfg3_jk(eri):
    basis, D, thr = W.cfg3()
    plan = eri.eri_plan_create(basis, thr)
    J, K = plan.build_jk(dev(D))
    return basis, D, thr, plan, J.cpu().numpy(), K.cpu().numpy()


def _sample_pairs(basis, seed, per_combo):
    """seeded shell pairs covering every (l_i, l_j) combination, the contracted core shells first"""
    rng = np.random.default_rng(seed)
    l = basis.shells["l"]; k = basis.shells["nprim"]
    pairs = []
    for li in sorted(set(l.tolist())):
        for lj in sorted(set(l.tolist())):
            if lj > li:
                continue
            si = np.where(l == li)[0]; sj = np.where(l == lj)[0]
            for _ in range(per_combo):
                pairs.append((int(rng.choice(si)), int(rng.choice(sj))))
    k8 = np.where(k == k.max())[0]
    pairs += [(int(k8[0]), int(k8[1])), (int(k8[-1]), int(k8[-1])), (int(np.where(l == l.max())[0][0]), int(k8[3]))]
    return pairs


def _block(M, basis, i, j):
    oi, oj = basis.shells["ao_off"][i], basis.shells["ao_off"][j]
    ni, nj = 2 * basis.shells["l"][i] + 1, 2 * basis.shells["l"][j] + 1
    return M[oi:oi + ni, oj:oj + nj]


def test_cfg3_sampled_blocks_against_oracle(eri, orc, cfg3_jk):
    basis, D, thr, plan, J, K = cfg3_jk
    scale = np.abs(J).max()
    assert np.abs(J - J.T).max() <= 1e-13 * scale and np.abs(K - K.T).max() <= 1e-13 * scale
    assert np.isfinite(J).all() and np.isfinite(K).all()
    pj = _sample_pairs(basis, 2407, 6)     # 6 per (l_i, l_j) combination + 3 core-shell pairs = 63 blocks (64 + 64)
    for (i, j), blk in zip(pj, orc.j_blocks(basis, D, pj)):
        assert np.abs(_block(J, basis, i, j) - blk).max() <= JK_TOL * scale, ("J", i, j)
    pk = _sample_pairs(basis, 9700, 6)
    for (i, j), blk in zip(pk, orc.k_blocks(basis, D, pk)):
        assert np.abs(_block(K, basis, i, j) - blk).max() <= JK_TOL * scale, ("K", i, j)


def test_cfg3_kernel_selections_and_schedules_agree(eri, cfg3_jk):
    """tile + register + cooperative (default) vs register + cooperative only, and concurrent vs serialised launches"""
    basis, D, thr, plan, J, K = cfg3_jk
    scale = np.abs(J).max()
    kinds = {c["kernel"] for c in plan.class_stats()}
    assert 3 in kinds and 2 in kinds and 0 not in kinds          # no class of cfg3 is left on the generic kernel
    st = plan.stats()
    assert st["quartets_kept"] == sum(c["quartets"] for c in plan.class_stats())
    # lane slots swept by a launch cover its quartets; the shell-grouped tiles of the tile family are well filled
    assert all(c["slots"] >= c["quartets"] for c in plan.class_stats())
    tile = [c for c in plan.class_stats() if c["kernel"] == 3]
    assert sum(c["quartets"] for c in tile) >= 0.75 * sum(c["slots"] for c in tile)
    plan.set_timing(True)                                         # serialised schedule
    J1, K1 = plan.build_jk(dev(D))
    plan.set_timing(False)
    assert np.abs(J1.cpu().numpy() - J).max() <= 1e-12 * scale and np.abs(K1.cpu().numpy() - K).max() <= 1e-12 * scale
    plan.set_kernel_mode(2)
    J2, K2 = plan.build_jk(dev(D))
    assert np.abs(J2.cpu().numpy() - J).max() <= 1e-11 * scale and np.abs(K2.cpu().numpy() - K).max() <= 1e-11 * scale
    plan.set_kernel_mode(0)


def test_cfg4_gradient_sum_rule_and_finite_differences(eri):
    basis, D, thr = W.cfg4()
    Dd = dev(D)
    plan = eri.eri_plan_create(basis, thr, want_grad=True)
    gJ, gK = plan.jk_grad(Dd)
    gJ, gK = gJ.cpu().numpy(), gK.cpu().numpy()
    assert np.isfinite(gJ).all() and np.isfinite(gK).all()
    assert np.abs(gJ.sum(axis=0)).max() <= GRAD_TOL and np.abs(gK.sum(axis=0)).max() <= GRAD_TOL
    kinds = {c["kernel_grad"] for c in plan.class_stats()}
    assert 3 in kinds                                             # the tile gradient kernels serve part of cfg4
    h = 1e-4
    for atom, ax in [(0, 0), (1, 2), (24, 1), (25, 0)]:            # O and H of the first and of the ninth molecule
        e = []
        for sgn in (+1, -1):
            xyz = basis.coords.copy()
            xyz[atom, ax] += sgn * h
            J, K = eri.eri_build_jk(basis.with_coords(xyz), Dd, thr)
            e.append((0.5 * (Dd * J).sum().item(), 0.5 * (Dd * K).sum().item()))
        fdJ, fdK = (e[0][0] - e[1][0]) / (2 * h), (e[0][1] - e[1][1]) / (2 * h)
        # truncation error of the central difference ~ h^2 f''' / 6 and rounding ~ 1e-16 E / h with E ~ 1e3
        assert abs(fdJ - gJ[atom, ax]) <= 2e-6 and abs(fdK - gK[atom, ax]) <= 2e-6, (atom, ax, fdJ, gJ[atom, ax], fdK, gK[atom, ax])


def test_cfg4_full_size_gradient_row_against_oracle(eri, orc):
    """SURVEY 8(c) cfg4 procedure at full size, in bench.py's launch configuration: the oracle's row mode (all quartets with
    the differentiated function on the atom, same Schwarz screening) for one hydrogen of the 16-water cluster; that row of
    the GPU gradient must match to BASELINE.json's 1e-8 Hartree/Bohr.  Covers what only large units reach: the runs of
    2..16 bra pairs per task of the cooperative gradient kernel and the re-routed (x|ps), (dp|ps) units."""
    basis, D, thr = W.cfg4()
    plan = eri.eri_plan_create(basis, thr, want_grad=True)
    gJ, gK = plan.jk_grad(dev(D))
    gJ, gK = gJ.cpu().numpy(), gK.cpu().numpy()
    atom = 3 * 9 + 1                                               # first H of the tenth molecule (inside the cluster)
    rJ, rK = orc.jk_grad(basis, D, atoms=[atom], thr=thr)
    assert np.abs(gJ[atom] - rJ[atom]).max() <= GRAD_TOL, (gJ[atom], rJ[atom])
    assert np.abs(gK[atom] - rK[atom]).max() <= GRAD_TOL, (gK[atom], rK[atom])
    # the three kernel selections agree on the whole gradient (generic = mode 1 is the reference path)
    for mode in (2, 1):
        plan.set_kernel_mode(mode)
        hJ, hK = plan.jk_grad(dev(D))
        assert np.abs(hJ.cpu().numpy() - gJ).max() <= GRAD_TOL and np.abs(hK.cpu().numpy() - gK).max() <= GRAD_TOL, mode


def test_gradient_four_water_tz_against_oracle(eri, orc):
    """full oracle gradient of a 4-water cluster with the cfg4 basis (88 shells), default kernel selection and
    the cooperative kernel forced to full runs of 16 bra pairs (the multi-bra-pair path under the oracle)."""
    basis, D = W.water_cluster((1, 2, 2), "tz", 43, "tz4g")
    gJo, gKo = orc.jk_grad(basis, D, thr=1e-13)
    plan = eri.eri_plan_create(basis, 1e-13, want_grad=True)
    for tasks in (None, 0.0):
        if tasks is not None:
            plan.set_tuning(eri.ERI_TUNE_GRAD_MIN_TASKS, tasks)
        gJ, gK = plan.jk_grad(dev(D))
        assert np.abs(gJ.cpu().numpy() - gJo).max() <= GRAD_TOL, tasks
        assert np.abs(gK.cpu().numpy() - gKo).max() <= GRAD_TOL, tasks
    plan.set_kernel_mode(2)                                        # no tile family: everything on the cooperative gradient kernel, runs of 16
    gJ, gK = plan.jk_grad(dev(D))
    assert np.abs(gJ.cpu().numpy() - gJo).max() <= GRAD_TOL and np.abs(gK.cpu().numpy() - gKo).max() <= GRAD_TOL


def test_gradient_two_water_tz_against_oracle(eri, orc):
    """the cfg4 basis (f shells, K = 8 core shells) on two waters: every gradient class of cfg4 occurs, tile and generic kernels"""
    basis, D = W.water_cluster((1, 1, 2), "tz", 77, "tz2")
    gJ, gK = eri.eri_jk_grad(basis, dev(D), 1e-13)
    gJo, gKo = orc.jk_grad(basis, D)
    assert np.abs(gJ.cpu().numpy() - gJo).max() <= GRAD_TOL
    assert np.abs(gK.cpu().numpy() - gKo).max() <= GRAD_TOL
    # primitive-parallel gradient kernel (pp_grad.cuh) on every unit of the classes it serves, whatever the contraction depth
    plan = eri.eri_plan_create(basis, 1e-13, want_grad=True)
    plan.set_kernel_mode(2)
    plan.set_tuning(eri.ERI_TUNE_PGRAD_MIN_NPP, 1)
    kinds = {}
    for c in plan.class_stats():
        kinds.setdefault((c["la"], c["lb"], c["lc"], c["ld"]), set()).add(c["kernel_grad"])
    served = {tuple(int(v) for v in x.split()[1:]) for x in eri.eri_kernel_catalog() if x.startswith("pgrad ")}
    assert len(served) == 15 and all(kinds[c] == {4} for c in served), kinds
    pJ, pK = plan.jk_grad(dev(D))
    assert np.abs(pJ.cpu().numpy() - gJo).max() <= GRAD_TOL and np.abs(pK.cpu().numpy() - gKo).max() <= GRAD_TOL
    plan.set_tuning(eri.ERI_TUNE_PGRAD_MIN_NPP, 3)              # the default rule: contracted units the tile kernel declines or fills badly
    plan.set_kernel_mode(0)
    assert 4 in {c["kernel_grad"] for c in plan.class_stats()}
    qJ, qK = plan.jk_grad(dev(D))
    assert np.abs(qJ.cpu().numpy() - gJo).max() <= GRAD_TOL and np.abs(qK.cpu().numpy() - gKo).max() <= GRAD_TOL

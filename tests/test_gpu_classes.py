"""Per-class parity of the tuned kernels (register and cooperative families) against the oracle, through the C ABI.

Every canonical l-class up to f (the 55 classes of cfg3/cfg4) plus a sample of g classes is digested as an explicit
quartet list (cfg1 recipe) with contraction degree 2, so that the primitive loops, the per-primitive
choice of the HRR build centre and the six digestion updates are all exercised; the same lists are run on the generic
kernels, and both must match the oracle to BASELINE.json's 1e-10 * max|J|."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_2407_09700_b200 import workloads as W  # noqa: E402

CLASSES_F = [c for c in W.canonical_classes(4) if max(c) <= 3]
CLASSES_G = [c for c in W.canonical_classes(4) if max(c) == 4]   # all 65 g classes: every cooperative instantiation (TW, NCH, PASSES differ per class)
# contraction degrees 1 and 3 beside 2 (BASELINE.json configs[1]: K in {1, 3, 6}; K = 6 in test_gpu_parity.CFG1_CASES) on classes of every family
CLASSES_K13 = [(0, 0, 0, 0), (1, 0, 1, 0), (2, 1, 1, 0), (1, 1, 1, 1), (2, 1, 2, 1), (2, 2, 2, 0), (3, 1, 2, 1), (3, 3, 1, 0), (3, 2, 3, 2),
               (4, 0, 1, 0), (4, 1, 4, 0), (4, 4, 0, 0), (4, 2, 3, 1)]


@pytest.fixture(scope="module")
def eri():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2407_09700_b200 import eri as E
    E.lib()
    return E


def _n_for(cls):
    size = 1
    for l in cls:
        size *= (l + 1) * (l + 2) // 2
    return 64 if size <= 100 else 24 if size <= 2000 else 8 if size <= 12000 else 5


CASES = [(c, 2) for c in CLASSES_F + CLASSES_G] + [(c, k) for c in CLASSES_K13 for k in (1, 3)]


@pytest.mark.parametrize("cls,K", CASES, ids=lambda v: "".join("spdfg"[l] for l in v) if isinstance(v, tuple) else f"K{v}")
def test_class_list_digest(eri, orc, cls, K):
    assert len(CLASSES_F) == 55 and len(CLASSES_G) == 65
    n = _n_for(cls)
    basis, D, q = W.cfg1_class(cls, K, nquartets=n, pool=6)
    Dd = torch.from_numpy(D).cuda()
    Jo, Ko = orc.digest_list(basis, D, q)
    scale = max(np.abs(Jo).max(), np.abs(Ko).max(), 1e-300)
    for mode in (0, 1):
        plan = eri.eri_list_plan_create(basis, q)
        plan.set_kernel_mode(mode)
        Jt, Kt = plan.build_jk(Dd)
        assert np.abs(Jt.cpu().numpy() - Jo).max() <= 1e-10 * scale, (cls, mode)
        assert np.abs(Kt.cpu().numpy() - Ko).max() <= 1e-10 * scale, (cls, mode)


def test_tuned_kernels_are_selected(eri):
    """The tuned families must actually serve the classes the plan reports (kernel != 0), not fall back silently."""
    basis, D = W.water_cluster((1, 1, 2), "tz", 77, "tz2")
    plan = eri.eri_plan_create(basis, 1e-13)
    kinds = {}
    for c in plan.class_stats():
        kinds.setdefault((c["la"], c["lb"], c["lc"], c["ld"]), set()).add(c["kernel"])
    assert all(k.issubset({1, 2, 3}) for k in kinds.values()), kinds
    assert kinds[(3, 3, 3, 3)] == {2}
    lp = eri.eri_list_plan_create(*W.cfg1_class((4, 4, 4, 4), 1, nquartets=4, pool=4)[::2])
    assert {c["kernel"] for c in lp.class_stats()} == {2}   # no class is left on the generic kernel
    plan.set_kernel_mode(2)   # register and cooperative families only
    kinds = {}
    for c in plan.class_stats():
        kinds.setdefault((c["la"], c["lb"], c["lc"], c["ld"]), set()).add(c["kernel"])
    assert kinds[(0, 0, 0, 0)] == {1} and kinds[(2, 1, 1, 0)] == {1}
    assert kinds[(2, 1, 2, 1)] == {2} and kinds[(2, 2, 2, 1)] == {2}
    plan.set_kernel_mode(1)
    assert all(c["kernel"] == 0 for c in plan.class_stats())


def test_dense_tuned_equals_generic_on_4_water_dzp_and_sharding(eri):
    """Dense (tile) mode: tuned == generic to rounding; two shards sum to the whole (eri_plan_set_shard)."""
    basis, D = W.water_cluster((1, 2, 2), "tz", 41, "tz4")
    Dd = torch.from_numpy(D).cuda()
    plan = eri.eri_plan_create(basis, 1e-13)
    J, K = plan.build_jk(Dd)
    J, K = J.clone(), K.clone()
    plan.set_kernel_mode(1)
    Jg, Kg = plan.build_jk(Dd)
    scale = J.abs().max().item()
    assert (J - Jg).abs().max().item() <= 1e-11 * scale and (K - Kg).abs().max().item() <= 1e-11 * scale
    plan.set_kernel_mode(0)
    Js, Ks = torch.zeros_like(J), torch.zeros_like(K)
    for r in range(3):
        plan.set_shard(r, 3)
        a, b = plan.build_jk(Dd)
        Js += a; Ks += b
    assert (J - Js).abs().max().item() <= 1e-12 * scale and (K - Ks).abs().max().item() <= 1e-12 * scale

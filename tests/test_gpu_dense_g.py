"""Dense-mode (tile family) kernels for g shells under the oracle.

tests/test_gpu_classes.py runs list mode, which the tile family does not serve, and cfg2/cfg3/cfg4 have no g shells: the
fourteen g classes of the tile J/K family and the five of the tile gradient family are exercised here on small clusters
whose pair sets fill the half-chunks (many s shells, a few shells of every higher l), with the fill thresholds of the
kernel selection switched off (eri_plan_set_tuning) so that every served class really runs on its tile kernel; the
results are compared with the oracle's full J/K resp. full gradient (unscreened, no symmetry)."""
import math
import re

import numpy as np
import pytest

from paper_2407_09700_b200 import workloads as W

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def eri():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2407_09700_b200 import eri as E
    E.lib()
    return E


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def g_cluster(counts, seed, box=4.0, kp=2):
    """counts[l] shells of angular momentum l, each on its own centre (the first counts[l] of max(counts) centres in a
    `box` Bohr cube); one primitive each, two for the p shells; exponents in [0.4, 1.6] so that nothing is screened"""
    rng = np.random.default_rng(seed)
    ncentre = max(counts)
    coords = rng.uniform(0.0, box, (ncentre, 3))
    atom_shells = [[] for _ in range(ncentre)]
    for l, cnt in enumerate(counts):
        K = kp if l == 1 else 1
        for c in range(cnt):
            e = np.sort(np.exp(rng.uniform(math.log(0.4), math.log(1.6), K)))[::-1].copy()
            atom_shells[c].append((l, e, W.normalise(l, e, rng.uniform(0.2, 1.0, K))))
    b = W._assemble(atom_shells, coords, {"name": "g_cluster"})
    C = rng.standard_normal((b.nao, 8)) / math.sqrt(b.nao)
    return b, C @ C.T


def _tile_classes(header, pattern):
    import os
    path = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_2407_09700_b200", "csrc", header)
    return {tuple(int(x) for x in m) for m in re.findall(pattern, open(path).read())}


def test_tile_jk_g_classes_against_oracle(eri, orc):
    basis, D = g_cluster([16, 8, 4, 2, 4], seed=23)
    plan = eri.eri_plan_create(basis, 0.0)
    plan.set_tuning(eri.ERI_TUNE_TILE_FILL_SCALE, 0.0)
    kinds = {}
    for c in plan.class_stats():
        kinds.setdefault((c["la"], c["lb"], c["lc"], c["ld"]), set()).add(c["kernel"])
    tile_g = {c for c in _tile_classes("tile_classes.h", r"X\((\d),(\d),(\d),(\d),\d+,\d+\)") if max(c) == 4}
    assert len(tile_g) >= 14
    for cls in tile_g:
        assert kinds.get(cls) == {3}, (cls, kinds.get(cls))      # every g class of the tile family runs on its tile kernel here
    J, K = plan.build_jk(dev(D))
    Jo, Ko, _ = orc.jk(basis, D, 0.0)
    scale = np.abs(Jo).max()
    assert np.abs(J.cpu().numpy() - Jo).max() <= 1e-10 * scale
    assert np.abs(K.cpu().numpy() - Ko).max() <= 1e-10 * scale
    # and the default selection (fill thresholds on) gives the same matrices
    plan.set_tuning(eri.ERI_TUNE_TILE_FILL_SCALE, 1.0)
    J1, K1 = plan.build_jk(dev(D))
    assert np.abs(J1.cpu().numpy() - Jo).max() <= 1e-10 * scale and np.abs(K1.cpu().numpy() - Ko).max() <= 1e-10 * scale


def test_tile_grad_g_classes_against_oracle(eri, orc):
    basis, D = g_cluster([16, 8, 4, 0, 4], seed=29)
    plan = eri.eri_plan_create(basis, 0.0, want_grad=True)
    plan.set_tuning(eri.ERI_TUNE_TILE_FILL_SCALE, 0.0)
    kinds = {}
    for c in plan.class_stats():
        kinds.setdefault((c["la"], c["lb"], c["lc"], c["ld"]), set()).add(c["kernel_grad"])
    tgrad_g = {c for c in _tile_classes("tile_grad_classes.h", r"X\((\d),(\d),(\d),(\d),\d+,\d+\)") if max(c) == 4}
    assert len(tgrad_g) >= 5
    for cls in tgrad_g:
        assert kinds.get(cls) == {3}, (cls, kinds.get(cls))
    served = {tuple(int(v) for v in x.split()[1:]) for x in eri.eri_kernel_catalog() if x.split()[0] in ("cgrad", "tgrad")}
    assert all(0 not in k for cls, k in kinds.items() if cls in served), kinds   # the generic gradient kernel only where no tuned one exists
    gJ, gK = plan.jk_grad(dev(D))
    gJo, gKo = orc.jk_grad(basis, D)
    assert np.abs(gJ.cpu().numpy() - gJo).max() <= 1e-8 and np.abs(gK.cpu().numpy() - gKo).max() <= 1e-8
    plan.set_tuning(eri.ERI_TUNE_TILE_FILL_SCALE, 1.0)
    plan.set_tuning(eri.ERI_TUNE_GRAD_MIN_TASKS, 0.0)              # cooperative gradient kernel with full runs of 16 bra pairs per task
    g1J, g1K = plan.jk_grad(dev(D))
    assert np.abs(g1J.cpu().numpy() - gJo).max() <= 1e-8 and np.abs(g1K.cpu().numpy() - gKo).max() <= 1e-8

"""Collected last (file name).  eri_density_group_max_noalloc -- the allocation-free form of the pass over the density that
density-weighted screening starts with (Eq. 9) -- against the existing path, the shell-group maxima that
eri_plan_build_jk_dscreen computes into a cudaMalloc'd buffer of the plan (read back by eri_plan_dscreen_group_max), on two
calls in a row with different densities (the static scratch array keeps the first call's contents; the second density is
smaller everywhere, so stale maxima would show).  Maxima are exact in any order: the comparison is bit for bit.  The test
stands alone (fresh process) and after the other GPU tests alike: it needs no state from them."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _cuda():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


def test_noalloc_group_max_equals_plan_path_on_two_calls():
    _cuda()
    from paper_2407_09700_b200 import eri, workloads
    basis, D, _ = workloads.cfg2()
    thr = 1e-8
    plan = eri.eri_plan_create(basis, thr)
    ng = plan.stats()["n_shell_groups"]
    assert 1 < ng <= eri.ERI_NOALLOC_MAX_GROUPS
    rng = np.random.default_rng(97)
    S = rng.uniform(0.0, 1.0, D.shape)
    dens = [D, 1e-3 * D * (S + S.T)]            # second call: every entry smaller in magnitude than in the first
    P = torch.full((ng, ng), -1.0, dtype=torch.float64, device="cuda")
    ag_dev = None
    for k, Dk in enumerate(dens):
        Dd = torch.from_numpy(np.ascontiguousarray(Dk)).cuda()
        plan.build_jk_dens(Dd)                  # existing path: group_max_kernel into the plan's own buffer
        ag, P_ref = plan.dens_group_max()
        if ag_dev is None:
            ag_dev = torch.from_numpy(ag).cuda()
        free_before = torch.cuda.mem_get_info()[0]
        eri.eri_density_group_max_noalloc(Dd, ag_dev, ng, P)
        torch.cuda.synchronize()
        if k == 1:   # (the first call may load the kernels' code lazily; that is the driver's, not an allocation of the call)
            assert torch.cuda.mem_get_info()[0] == free_before, "the allocation-free entry point changed the free device memory"
        got = P.cpu().numpy()
        assert np.array_equal(got, P_ref), (k, np.abs(got - P_ref).max())
        # independent of both GPU paths: the definition written out in numpy
        want = np.zeros((ng, ng))
        np.maximum.at(want, (ag[:, None].repeat(len(ag), 1), ag[None, :].repeat(len(ag), 0)), np.abs(Dk))
        assert np.array_equal(got, want), k
    assert P.cpu().numpy().max() < 1e-2 * np.abs(D).max() * 2.0   # the second call's maxima, not the first's
    plan.destroy()


def test_noalloc_group_max_rejects_sizes_beyond_the_static_array():
    _cuda()
    from paper_2407_09700_b200 import eri
    n = 8
    D = torch.ones((n, n), dtype=torch.float64, device="cuda")
    ag = torch.zeros(n, dtype=torch.int32, device="cuda")
    big = eri.ERI_NOALLOC_MAX_GROUPS + 1
    P = torch.zeros((big, big), dtype=torch.float64, device="cuda")
    with pytest.raises(eri.EriError, match="ERI_NOALLOC_MAX_GROUPS"):
        eri.eri_density_group_max_noalloc(D, ag, big, P)
    # the largest accepted size works, ids outside 0..ngroups-1 are ignored
    m = eri.ERI_NOALLOC_MAX_GROUPS
    ag = torch.tensor([0, 1, m - 1, m - 1, m, -1, 5, 5], dtype=torch.int32, device="cuda")
    Dh = np.arange(1.0, n * n + 1.0).reshape(n, n) * np.where(np.arange(n * n).reshape(n, n) % 2 == 0, 1.0, -1.0)
    P = torch.full((m, m), -1.0, dtype=torch.float64, device="cuda")
    eri.eri_density_group_max_noalloc(torch.from_numpy(Dh).cuda(), ag, m, P)
    want = np.zeros((m, m))
    agh = ag.cpu().numpy()
    for i in range(n):
        for j in range(n):
            if 0 <= agh[i] < m and 0 <= agh[j] < m:
                want[agh[i], agh[j]] = max(want[agh[i], agh[j]], abs(Dh[i, j]))
    assert np.array_equal(P.cpu().numpy(), want)

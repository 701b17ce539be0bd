"""CPU-side checks of the C-ABI library: it builds, loads, exports every symbol include/eri.h declares, validates
arguments before touching the device, and its host-side tables agree with independent constructions.
No compute call is made here (there is no GPU on this box, and there is no CPU fallback)."""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def eri():
    from paper_2407_09700_b200 import build
    build.build()
    from paper_2407_09700_b200 import eri as E
    E.lib()
    return E


def declared_functions():
    src = open(os.path.join(ROOT, "include", "eri.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(eri_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(eri):
    names = declared_functions()
    assert len(names) >= 20
    for n in names:
        assert hasattr(eri.lib(), n), n
    assert sorted(eri.EXPORTS) == names


def test_c2s_table_matches_oracle_route(eri):
    """Library: closed formula (reading R3).  Oracle: least-squares projection on scipy's spherical harmonics."""
    import oracle.sph as sph
    for l in range(7):
        assert np.abs(eri.eri_c2s_matrix(l) - sph.c2s(l)).max() < 1e-13


def test_canonical_flop_model_pins(eri):
    """(ss|ss) 162 per primitive quartet and 182 per contracted quartet at K=1; (pp|pp) 1.77e3."""
    assert eri.eri_canonical_flops(0, 0, 0, 0, 1, 1, 1, 1) == 182.0
    assert eri.eri_canonical_flops(0, 0, 0, 0, 3, 3, 3, 3) == 81 * 162.0 + 20.0
    f = eri.eri_canonical_flops(1, 1, 1, 1, 1, 1, 1, 1)
    assert abs(f - 4.7e3) < 1e2
    f = eri.eri_canonical_flops(4, 4, 4, 4, 1, 1, 1, 1)
    assert abs(f - 3.5e6) < 1e5


def test_argument_errors_need_no_device(eri):
    from paper_2407_09700_b200 import workloads as W
    import ctypes
    basis, D, thr = W.cfg0()
    bad = W.Basis(basis.shells.copy(), basis.prims.copy(), basis.coords.copy(), basis.nao)
    bad.shells["l"][0] = 7
    args, keep = eri._basis_args(bad)
    h = ctypes.c_void_p()
    rc = eri.lib().eri_plan_create(*args, ctypes.c_double(0.0), 0, None, ctypes.byref(h))
    assert rc == -2 and b"outside" in eri.lib().eri_last_error()
    bad.shells["l"][0] = 0
    bad.prims["exp"][2] = -1.0
    args, keep = eri._basis_args(bad)
    rc = eri.lib().eri_plan_create(*args, ctypes.c_double(0.0), 0, None, ctypes.byref(h))
    assert rc == -1
    assert eri.lib().eri_strerror(-3) == b"CUDA failure"


def test_no_gpu_means_loud_failure(eri):
    torch = pytest.importorskip("torch")
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2407_09700_b200 import workloads as W
    import ctypes
    basis, D, thr = W.cfg0()
    args, keep = eri._basis_args(basis)
    h = ctypes.c_void_p()
    rc = eri.lib().eri_plan_create(*args, ctypes.c_double(0.0), 0, None, ctypes.byref(h))
    assert rc == -3   # ERI_ERR_CUDA: no fallback


def test_noalloc_entry_point_validates_sizes_without_a_device(eri):
    """eri_density_group_max_noalloc refuses what its static scratch array cannot hold, before touching the device"""
    import ctypes
    L = eri.lib()
    vp, ci = ctypes.c_void_p, ctypes.c_int
    big = eri.ERI_NOALLOC_MAX_GROUPS + 1
    rc = L.eri_density_group_max_noalloc(vp(8), ci(4), vp(8), ci(big), vp(8), None)   # (dummy non-null pointers: never dereferenced)
    assert rc == -1 and b"ERI_NOALLOC_MAX_GROUPS" in L.eri_last_error()
    assert L.eri_density_group_max_noalloc(vp(8), ci(-1), vp(8), ci(2), vp(8), None) == -1
    assert L.eri_density_group_max_noalloc(vp(8), ci(4), vp(8), ci(-2), vp(8), None) == -1
    assert L.eri_density_group_max_noalloc(None, ci(4), vp(8), ci(2), vp(8), None) == -1      # null D
    assert L.eri_density_group_max_noalloc(vp(8), ci(4), vp(8), ci(2), None, None) == -1      # null P
    assert L.eri_density_group_max_noalloc(None, ci(0), None, ci(0), None, None) == 0         # nothing to do
    assert L.eri_plan_dscreen_group_max(None, None, None) == -1

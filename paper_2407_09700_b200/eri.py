"""Thin ctypes binding over liberi_b200.so (include/eri.h).  Argument marshalling only: every step of the hot path
runs in the library's CUDA kernels.  PyTorch is used for device memory and streams, nothing else.

There is no CPU fallback: if the shared library has not been built (python -m paper_2407_09700_b200.build) or no CUDA
device is present, the calls raise.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liberi_b200.so")
_lib_handle = None

ERI_OK = 0
_vp, _i32, _i64, _f64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double


class EriError(RuntimeError):
    pass


class eri_stats_t(ctypes.Structure):
    _fields_ = [("nshell", _i32), ("nao", _i32), ("nao_cart", _i32), ("natm", _i32), ("n_shell_groups", _i32),
                ("n_pair_classes", _i32), ("n_quartet_classes", _i32), ("launches_per_call", _i32),
                ("pairs_total", _i64), ("pairs_kept", _i64), ("quartets_total", _i64), ("quartets_kept", _i64),
                ("canonical_flops", _f64), ("canonical_flops_grad", _f64), ("plan_ms", _f64),
                ("plan_ms_init", _f64), ("plan_ms_schwarz", _f64), ("plan_ms_pairs", _f64), ("plan_ms_units", _f64)]


class eri_class_stat_t(ctypes.Structure):
    _fields_ = [("la", _i32), ("lb", _i32), ("lc", _i32), ("ld", _i32), ("ka", _i32), ("kb", _i32), ("kc", _i32),
                ("kd", _i32), ("nroots", _i32), ("kernel", _i32), ("quartets", _i64), ("slots", _i64), ("canonical_flops", _f64),
                ("last_ms", ctypes.c_float), ("last_ms_grad", ctypes.c_float), ("kernel_grad", _i32), ("tile_fill_pm", _i32),
                ("canonical_flops_grad", _f64)]


EXPORTS = ["eri_build_jk", "eri_jk_grad", "eri_plan_create", "eri_plan_build_jk", "eri_plan_jk_grad",
           "eri_plan_build_jk_dscreen", "eri_plan_dscreen_quartets", "eri_plan_dscreen_group_max", "eri_density_group_max_noalloc", "eri_plan_build_jk_host", "eri_plan_jk_grad_host", "eri_plan_stats", "eri_plan_num_classes",
           "eri_plan_class_stats", "eri_plan_set_timing", "eri_plan_set_kernel_mode", "eri_plan_set_tuning", "eri_plan_set_shard", "eri_plan_destroy",
           "eri_kernel_catalog", "eri_kernel_launched",
           "eri_compute_quartets", "eri_digest_quartet_list", "eri_list_plan_create", "eri_list_plan_digest",
           "eri_schwarz", "eri_rys_roots", "eri_c2s_matrix", "eri_measure_fp64_peak", "eri_canonical_flops",
           "eri_strerror", "eri_last_error", "eri_version"]


def library_path() -> str:
    return _SO


def lib():
    global _lib_handle
    if _lib_handle is None:
        if not os.path.exists(_SO):
            raise EriError(f"{_SO} is missing: build it with `python -m paper_2407_09700_b200.build` (no CPU fallback)")
        L = ctypes.CDLL(_SO)
        L.eri_last_error.restype = ctypes.c_char_p
        L.eri_strerror.restype = ctypes.c_char_p
        L.eri_version.restype = ctypes.c_char_p
        L.eri_canonical_flops.restype = _f64
        L.eri_plan_destroy.restype = None
        L.eri_plan_destroy.argtypes = [_vp]
        L.eri_plan_dscreen_quartets.argtypes = [_vp, ctypes.POINTER(_i64)]
        for name in ("eri_plan_build_jk", "eri_plan_build_jk_dscreen", "eri_plan_jk_grad", "eri_plan_build_jk_host", "eri_plan_jk_grad_host",
                     "eri_list_plan_digest"):
            getattr(L, name).argtypes = [_vp, _vp, _vp, _vp, _vp]
        L.eri_plan_dscreen_group_max.argtypes = [_vp, _vp, _vp]
        L.eri_density_group_max_noalloc.argtypes = [_vp, ctypes.c_int, _vp, ctypes.c_int, _vp, _vp]
        L.eri_plan_stats.argtypes = [_vp, ctypes.POINTER(eri_stats_t)]
        L.eri_plan_num_classes.argtypes = [_vp]
        L.eri_plan_class_stats.argtypes = [_vp, ctypes.POINTER(eri_class_stat_t), ctypes.c_int]
        L.eri_plan_set_timing.argtypes = [_vp, ctypes.c_int]
        L.eri_plan_set_kernel_mode.argtypes = [_vp, ctypes.c_int]
        L.eri_plan_set_shard.argtypes = [_vp, ctypes.c_int, ctypes.c_int]
        L.eri_plan_set_tuning.argtypes = [_vp, ctypes.c_int, _f64]
        L.eri_kernel_catalog.argtypes = [ctypes.c_char_p, ctypes.c_int]
        L.eri_kernel_launched.argtypes = [ctypes.c_char_p, ctypes.c_int]
        _lib_handle = L
    return _lib_handle


def _check(code: int):
    if code != ERI_OK:
        L = lib()
        raise EriError(f"{L.eri_strerror(code).decode()} ({code}): {L.eri_last_error().decode()}")


def _basis_args(basis):
    sh = np.ascontiguousarray(basis.shells)
    pr = np.ascontiguousarray(basis.prims)
    xyz = np.ascontiguousarray(basis.coords, dtype=np.float64)
    args = (_vp(sh.ctypes.data), ctypes.c_int(sh.shape[0]), _vp(pr.ctypes.data), ctypes.c_int(pr.shape[0]),
            _vp(xyz.ctypes.data), ctypes.c_int(xyz.shape[0]))
    return args, (sh, pr, xyz)


def _stream():
    import torch
    return _vp(torch.cuda.current_stream().cuda_stream)


def _dev_f64(t, shape=None):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise EriError("expected a contiguous float64 CUDA tensor")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise EriError(f"expected shape {shape}, got {tuple(t.shape)}")
    return _vp(t.data_ptr())


class Plan:
    """eri_plan_t*: geometry + basis + threshold dependent, density independent."""

    def __init__(self, handle, basis, is_list=False):
        self._h, self.basis, self.is_list = handle, basis, is_list

    def __del__(self):
        try:
            self.destroy()
        except Exception:   # interpreter shutdown: the module globals may already be gone; the process is ending anyway
            pass

    def destroy(self):
        if getattr(self, "_h", None):
            lib().eri_plan_destroy(self._h)
            self._h = None

    def build_jk(self, D, J=None, K=None):
        import torch
        n = self.basis.nao
        J = torch.empty((n, n), dtype=torch.float64, device=D.device) if J is None else J
        K = torch.empty((n, n), dtype=torch.float64, device=D.device) if K is None else K
        fn = lib().eri_list_plan_digest if self.is_list else lib().eri_plan_build_jk
        _check(fn(self._h, _dev_f64(D, (n, n)), _dev_f64(J, (n, n)), _dev_f64(K, (n, n)), _stream()))
        return J, K

    def build_jk_dens(self, D, J=None, K=None):
        """eri_plan_build_jk_dscreen: the build with the density factor of Eq. 8-9 in the screening test"""
        import torch
        n = self.basis.nao
        J = torch.empty((n, n), dtype=torch.float64, device=D.device) if J is None else J
        K = torch.empty((n, n), dtype=torch.float64, device=D.device) if K is None else K
        _check(lib().eri_plan_build_jk_dscreen(self._h, _dev_f64(D, (n, n)), _dev_f64(J, (n, n)), _dev_f64(K, (n, n)), _stream()))
        return J, K

    def dens_quartets(self) -> int:
        v = _i64(0)
        _check(lib().eri_plan_dscreen_quartets(self._h, ctypes.byref(v)))
        return int(v.value)

    def dens_group_max(self) -> tuple[np.ndarray, np.ndarray]:
        """eri_plan_dscreen_group_max: (ao_group[nao], P[ng, ng]) of the last density-weighted build"""
        ng = self.stats()["n_shell_groups"]
        ag = np.zeros(self.basis.nao, dtype=np.int32)
        P = np.zeros((ng, ng))
        _check(lib().eri_plan_dscreen_group_max(self._h, _vp(ag.ctypes.data), _vp(P.ctypes.data)))
        return ag, P

    def jk_grad(self, D, gJ=None, gK=None):
        import torch
        n, na = self.basis.nao, self.basis.natm
        gJ = torch.empty((na, 3), dtype=torch.float64, device=D.device) if gJ is None else gJ
        gK = torch.empty((na, 3), dtype=torch.float64, device=D.device) if gK is None else gK
        _check(lib().eri_plan_jk_grad(self._h, _dev_f64(D, (n, n)), _dev_f64(gJ, (na, 3)), _dev_f64(gK, (na, 3)), _stream()))
        return gJ, gK

    def build_jk_host(self, D, J, K):
        """D, J, K: C-contiguous float64 numpy arrays (ideally views of pinned memory)."""
        for a in (D, J, K):
            assert a.dtype == np.float64 and a.flags.c_contiguous and a.shape == (self.basis.nao, self.basis.nao)
        _check(lib().eri_plan_build_jk_host(self._h, _vp(D.ctypes.data), _vp(J.ctypes.data), _vp(K.ctypes.data), _stream()))
        return J, K

    def jk_grad_host(self, D, gJ, gK):
        assert D.dtype == np.float64 and D.flags.c_contiguous and D.shape == (self.basis.nao, self.basis.nao)
        for a in (gJ, gK):
            assert a.dtype == np.float64 and a.flags.c_contiguous and a.shape == (self.basis.natm, 3)
        _check(lib().eri_plan_jk_grad_host(self._h, _vp(D.ctypes.data), _vp(gJ.ctypes.data), _vp(gK.ctypes.data), _stream()))
        return gJ, gK

    def stats(self) -> dict:
        s = eri_stats_t()
        _check(lib().eri_plan_stats(self._h, ctypes.byref(s)))
        return {k: getattr(s, k) for k, _ in eri_stats_t._fields_}

    def class_stats(self) -> list[dict]:
        n = lib().eri_plan_num_classes(self._h)
        arr = (eri_class_stat_t * max(n, 1))()
        m = lib().eri_plan_class_stats(self._h, arr, n)
        if m < 0:
            _check(m)
        return [{k: getattr(arr[i], k) for k, _ in eri_class_stat_t._fields_} for i in range(m)]

    def set_timing(self, on: bool):
        _check(lib().eri_plan_set_timing(self._h, int(on)))

    def set_kernel_mode(self, mode: int):
        _check(lib().eri_plan_set_kernel_mode(self._h, int(mode)))

    def set_tuning(self, key: int, value: float):
        _check(lib().eri_plan_set_tuning(self._h, int(key), float(value)))

    def set_shard(self, rank: int, nranks: int):
        _check(lib().eri_plan_set_shard(self._h, int(rank), int(nranks)))


def eri_plan_create(basis, schwarz_thr: float, want_grad: bool = False) -> Plan:
    args, keep = _basis_args(basis)
    h = _vp()
    _check(lib().eri_plan_create(*args, _f64(schwarz_thr), ctypes.c_int(int(want_grad)), _stream(), ctypes.byref(h)))
    return Plan(h, basis)


def eri_list_plan_create(basis, quartets) -> Plan:
    args, keep = _basis_args(basis)
    q = np.ascontiguousarray(quartets, dtype=np.int32).reshape(-1, 4)
    h = _vp()
    _check(lib().eri_list_plan_create(*args, _vp(q.ctypes.data), ctypes.c_int(q.shape[0]), _stream(), ctypes.byref(h)))
    return Plan(h, basis, is_list=True)


def eri_build_jk(basis, D, schwarz_thr: float):
    """One-shot J/K build; D a (nao, nao) float64 CUDA tensor.  Returns (J, K) CUDA tensors."""
    import torch
    args, keep = _basis_args(basis)
    n = basis.nao
    J = torch.empty((n, n), dtype=torch.float64, device=D.device)
    K = torch.empty((n, n), dtype=torch.float64, device=D.device)
    _check(lib().eri_build_jk(*args, _dev_f64(D, (n, n)), _f64(schwarz_thr), _dev_f64(J), _dev_f64(K), _stream()))
    return J, K


def eri_jk_grad(basis, D, schwarz_thr: float):
    import torch
    args, keep = _basis_args(basis)
    n, na = basis.nao, basis.natm
    gJ = torch.empty((na, 3), dtype=torch.float64, device=D.device)
    gK = torch.empty((na, 3), dtype=torch.float64, device=D.device)
    _check(lib().eri_jk_grad(*args, _dev_f64(D, (n, n)), _f64(schwarz_thr), _dev_f64(gJ), _dev_f64(gK), _stream()))
    return gJ, gK


def eri_digest_quartet_list(basis, quartets, D):
    import torch
    args, keep = _basis_args(basis)
    q = np.ascontiguousarray(quartets, dtype=np.int32).reshape(-1, 4)
    n = basis.nao
    Jt = torch.empty((n, n), dtype=torch.float64, device=D.device)
    Kt = torch.empty((n, n), dtype=torch.float64, device=D.device)
    _check(lib().eri_digest_quartet_list(*args, _vp(q.ctypes.data), ctypes.c_int(q.shape[0]), _dev_f64(D, (n, n)),
                                         _dev_f64(Jt), _dev_f64(Kt), _stream()))
    return Jt, Kt


ERI_NOALLOC_MAX_GROUPS = 64


def eri_density_group_max_noalloc(D, ao_group, ngroups: int, P):
    """Allocation-free shell-group maxima of |D| (Eq. 9): D (nao, nao) float64, ao_group (nao,) int32, P (ngroups, ngroups)
    float64, all CUDA tensors supplied by the caller; the library allocates nothing (static device scratch)."""
    import torch
    nao = int(D.shape[0])
    if not (isinstance(ao_group, torch.Tensor) and ao_group.is_cuda and ao_group.dtype == torch.int32 and ao_group.is_contiguous()
            and ao_group.numel() == nao):
        raise EriError("ao_group: expected a contiguous int32 CUDA tensor of nao entries")
    _check(lib().eri_density_group_max_noalloc(_dev_f64(D, (nao, nao)), ctypes.c_int(nao), _vp(ao_group.data_ptr()), ctypes.c_int(int(ngroups)),
                                               _dev_f64(P, (ngroups, ngroups)), _stream()))
    return P


def eri_compute_quartets(basis, quartets) -> list[np.ndarray]:
    """Spherical blocks (ij|kl), one numpy array [ns_i, ns_j, ns_k, ns_l] per listed quartet."""
    import torch
    args, keep = _basis_args(basis)
    q = np.ascontiguousarray(quartets, dtype=np.int32).reshape(-1, 4)
    ls = basis.shells["l"]
    shapes = [tuple(2 * int(ls[s]) + 1 for s in row) for row in q]
    sizes = np.array([int(np.prod(s)) for s in shapes], dtype=np.int64)
    off = np.zeros(len(sizes), dtype=np.int64)
    if len(sizes):
        off[1:] = np.cumsum(sizes)[:-1]
    out = torch.zeros(int(sizes.sum()) if len(sizes) else 0, dtype=torch.float64, device="cuda")
    _check(lib().eri_compute_quartets(*args, _vp(q.ctypes.data), ctypes.c_int(q.shape[0]), _vp(out.data_ptr()),
                                      _vp(off.ctypes.data), _stream()))
    h = out.cpu().numpy()
    return [h[o:o + n].reshape(s).copy() for o, n, s in zip(off, sizes, shapes)]


def eri_schwarz(basis) -> np.ndarray:
    args, keep = _basis_args(basis)
    Q = np.zeros((basis.nshell, basis.nshell))
    _check(lib().eri_schwarz(*args, _vp(Q.ctypes.data), _stream()))
    return Q


def eri_rys_roots(nroots: int, x) -> tuple[np.ndarray, np.ndarray]:
    x = np.ascontiguousarray(x, dtype=np.float64).ravel()
    u = np.zeros((x.size, nroots))
    w = np.zeros((x.size, nroots))
    _check(lib().eri_rys_roots(ctypes.c_int(nroots), _vp(x.ctypes.data), ctypes.c_int(x.size), _vp(u.ctypes.data), _vp(w.ctypes.data)))
    return u, w


def eri_c2s_matrix(l: int) -> np.ndarray:
    T = np.zeros((2 * l + 1, (l + 1) * (l + 2) // 2))
    _check(lib().eri_c2s_matrix(ctypes.c_int(l), _vp(T.ctypes.data)))
    return T


def eri_measure_fp64_peak() -> float:
    v = _f64(0.0)
    _check(lib().eri_measure_fp64_peak(ctypes.byref(v), _stream()))
    return float(v.value)


def eri_canonical_flops(la, lb, lc, ld, ka, kb, kc, kd, deriv=False) -> float:
    return float(lib().eri_canonical_flops(la, lb, lc, ld, ka, kb, kc, kd, int(bool(deriv))))


ERI_TUNE_TILE_FILL_SCALE, ERI_TUNE_GRAD_MIN_TASKS, ERI_TUNE_PGRAD_MIN_NPP = 0, 1, 2


def _string_list(fn) -> list[str]:
    n = fn(None, 0)
    buf = ctypes.create_string_buffer(n)
    fn(buf, n)
    return [x for x in buf.value.decode().split("\n") if x]


def eri_kernel_catalog() -> list[str]:
    """every tuned kernel instantiation of the library, 'family la lb lc ld'"""
    return _string_list(lib().eri_kernel_catalog)


def eri_kernel_launched() -> list[str]:
    """the instantiations this process has launched so far"""
    return _string_list(lib().eri_kernel_launched)


def eri_version() -> str:
    return lib().eri_version().decode()

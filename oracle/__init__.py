"""ORACLE -- test infrastructure only (see md_oracle.cpp header).

ctypes wrapper over oracle/md_oracle.cpp.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` legs may import this package.  It imports nothing from the CUDA path; inputs are plain
numpy arrays in the layout of paper_2407_09700_b200.workloads (shells: 5 x int32, prims: 2 x float64).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

from . import sph

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "md_oracle.cpp")
_SO = os.path.join(_HERE, "libmd_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC", "-o", _SO, _SRC])
    return _SO


_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int32)


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_prim_eri.restype = ctypes.c_double
        _lib.oracle_jk.restype = ctypes.c_longlong
        _lib.oracle_jk_dscreen.restype = ctypes.c_longlong
        for l in range(7):
            T = sph.c2s(l)
            _lib.oracle_set_c2s(l, _d(T))
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(int(n))


def _basis_args(basis):
    sh = np.ascontiguousarray(basis.shells)
    pr = np.ascontiguousarray(basis.prims)
    xyz = np.ascontiguousarray(basis.coords, dtype=np.float64)
    keep = (sh, pr, xyz)
    args = (sh.ctypes.data_as(_ip), ctypes.c_int(sh.shape[0]), pr.ctypes.data_as(_dp), ctypes.c_int(pr.shape[0]),
            _d(xyz), ctypes.c_int(xyz.shape[0]))
    return args, keep


def boys(mmax: int, x: float) -> np.ndarray:
    F = np.zeros(mmax + 1)
    lib().oracle_boys(ctypes.c_int(mmax), ctypes.c_double(x), _d(F))
    return F


def prim_eri(powers, exps, centres) -> float:
    """[ab|cd] over raw primitive Cartesian Gaussians (Eq. 2).  powers[4][3], exps[4], centres[4][3]."""
    pw = np.ascontiguousarray(powers, dtype=np.int32).reshape(12)
    ex = np.ascontiguousarray(exps, dtype=np.float64).reshape(4)
    ct = np.ascontiguousarray(centres, dtype=np.float64).reshape(12)
    return float(lib().oracle_prim_eri(_i(pw), _d(ex), _d(ct)))


def eri_block(basis, i, j, k, l, deriv: bool = False) -> np.ndarray:
    n = [2 * int(basis.shells["l"][s]) + 1 for s in (i, j, k, l)]
    out = np.zeros(((3,) if deriv else ()) + tuple(n))
    args, keep = _basis_args(basis)
    lib().oracle_eri_block(*args, int(i), int(j), int(k), int(l), int(bool(deriv)), _d(out))
    return out


def overlap_block(basis, i, j) -> np.ndarray:
    """<i|j> of two contracted spherical shells from the E_0 Hermite coefficients (a pin helper, see md_oracle.cpp)."""
    out = np.zeros((2 * int(basis.shells["l"][i]) + 1, 2 * int(basis.shells["l"][j]) + 1))
    args, keep = _basis_args(basis)
    lib().oracle_overlap_block(*args, int(i), int(j), _d(out))
    return out


def schwarz(basis) -> np.ndarray:
    Q = np.zeros((basis.nshell, basis.nshell))
    args, keep = _basis_args(basis)
    lib().oracle_schwarz(*args, _d(Q))
    return Q


def jk(basis, D, thr: float = 0.0):
    D = np.ascontiguousarray(D, dtype=np.float64)
    J = np.zeros_like(D)
    K = np.zeros_like(D)
    args, keep = _basis_args(basis)
    n = lib().oracle_jk(*args, _d(D), ctypes.c_double(thr), _d(J), _d(K))
    return J, K, int(n)


def shell_groups(basis) -> np.ndarray:
    """Group id of every shell: shells of equal (l, nprim) form a set |a, K_a}; ids in sorted (l, K) order."""
    keys = sorted({(int(s["l"]), int(s["nprim"])) for s in basis.shells})
    return np.array([keys.index((int(s["l"]), int(s["nprim"]))) for s in basis.shells], dtype=np.int32)


def jk_dscreen(basis, D, thr: float):
    """J, K with the density-weighted batch screening of Eq. 8-9 at the level of shell groups; see md_oracle.cpp."""
    D = np.ascontiguousarray(D, dtype=np.float64)
    J = np.zeros_like(D)
    K = np.zeros_like(D)
    g = shell_groups(basis)
    args, keep = _basis_args(basis)
    n = lib().oracle_jk_dscreen(*args, _d(D), ctypes.c_double(thr), _i(g), ctypes.c_int(int(g.max()) + 1), _d(J), _d(K))
    return J, K, int(n)


def _block_sizes(basis, pairs):
    ls = basis.shells["l"]
    return [(2 * int(ls[a]) + 1, 2 * int(ls[b]) + 1) for a, b in pairs]


def _blocks(fn, basis, D, pairs):
    D = np.ascontiguousarray(D, dtype=np.float64)
    pairs = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
    sizes = _block_sizes(basis, pairs)
    out = np.zeros(sum(a * b for a, b in sizes))
    args, keep = _basis_args(basis)
    fn(*args, _d(D), _i(pairs), ctypes.c_int(pairs.shape[0]), _d(out))
    res, off = [], 0
    for a, b in sizes:
        res.append(out[off:off + a * b].reshape(a, b).copy())
        off += a * b
    return res


def j_blocks(basis, D, pairs):
    """J[i-shell, j-shell] blocks, each summed over all (k,l)."""
    return _blocks(lib().oracle_j_blocks, basis, D, pairs)


def k_blocks(basis, D, pairs):
    """K[i-shell, k-shell] blocks, each summed over all (j,l)."""
    return _blocks(lib().oracle_k_blocks, basis, D, pairs)


def digest_list(basis, D, quartets):
    D = np.ascontiguousarray(D, dtype=np.float64)
    q = np.ascontiguousarray(quartets, dtype=np.int32).reshape(-1, 4)
    Jt = np.zeros_like(D)
    Kt = np.zeros_like(D)
    args, keep = _basis_args(basis)
    lib().oracle_digest_list(*args, _d(D), _i(q), ctypes.c_int(q.shape[0]), _d(Jt), _d(Kt))
    return Jt, Kt


def jk_grad(basis, D, atoms=None, thr: float = 0.0):
    D = np.ascontiguousarray(D, dtype=np.float64)
    gJ = np.zeros((basis.natm, 3))
    gK = np.zeros((basis.natm, 3))
    at = np.ascontiguousarray([] if atoms is None else atoms, dtype=np.int32)
    args, keep = _basis_args(basis)
    lib().oracle_jk_grad(*args, _d(D), _i(at), ctypes.c_int(at.shape[0]), ctypes.c_double(thr), _d(gJ), _d(gK))
    return gJ, gK


def energy(basis, D, thr: float = 0.0):
    """E_J = 1/2 sum D_ij D_kl (ij|kl), E_K = 1/2 sum D_ik D_jl (ij|kl) (reading R13)."""
    J, K, _ = jk(basis, D, thr)
    return 0.5 * float(np.sum(D * J)), 0.5 * float(np.sum(D * K))

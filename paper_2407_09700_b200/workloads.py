"""Seeded synthetic inputs for cfg0..cfg4 (BASELINE.json `configs`; recipe in DESIGN.md "Input recipe").

This module serves BOTH the oracle tests and the CUDA path.  It holds none of the
method's arithmetic: it only draws geometries, basis-set parameters and densities,
and rescales contraction coefficients to unit self-overlap with the closed-form
radial integral of reading R2:

    <chi|chi> = sum_kk' c_k c_k' Gamma(l+3/2) / (2 (a_k+a_k')^(l+3/2)) = 1.

The paper measured on 32 H2O / cc-pVTZ -- neither that geometry nor the
basis data exist in this container, so these inputs stand in for them: same
shapes, sizes and contraction structure, synthetic numbers.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

ANGSTROM = 1.8897261246  # Bohr per Angstrom
SEED0 = 240709700

SHELL_DTYPE = np.dtype(
    [("atom", "<i4"), ("l", "<i4"), ("nprim", "<i4"), ("prim_off", "<i4"), ("ao_off", "<i4")]
)
PRIM_DTYPE = np.dtype([("exp", "<f8"), ("coef", "<f8")])


@dataclass
class Basis:
    """Plain container mirroring the C structs of include/eri.h."""

    shells: np.ndarray  # SHELL_DTYPE [nshell]
    prims: np.ndarray  # PRIM_DTYPE  [nprim]
    coords: np.ndarray  # float64 [natm,3], Bohr
    nao: int  # spherical functions, sum(2l+1)
    meta: dict = field(default_factory=dict)

    @property
    def nshell(self) -> int:
        return int(self.shells.shape[0])

    @property
    def natm(self) -> int:
        return int(self.coords.shape[0])

    def with_coords(self, coords: np.ndarray) -> "Basis":
        return Basis(self.shells.copy(), self.prims.copy(), np.ascontiguousarray(coords, dtype=np.float64),
                     self.nao, dict(self.meta))


def normalise(l: int, exps: np.ndarray, coefs: np.ndarray) -> np.ndarray:
    """Rescale raw coefficients to unit self-overlap (reading R2)."""
    e = np.asarray(exps, dtype=np.float64)
    c = np.asarray(coefs, dtype=np.float64)
    s = 0.0
    g = math.gamma(l + 1.5)
    for k in range(len(e)):
        for kk in range(len(e)):
            s += c[k] * c[kk] * g / (2.0 * (e[k] + e[kk]) ** (l + 1.5))
    return c / math.sqrt(s)


def _assemble(atom_shells: list[list[tuple[int, np.ndarray, np.ndarray]]], coords: np.ndarray, meta: dict) -> Basis:
    """atom_shells[atom] = list of (l, exps, coefs)."""
    sh, pr = [], []
    ao = 0
    for ia, lst in enumerate(atom_shells):
        for (l, e, c) in lst:
            sh.append((ia, l, len(e), len(pr), ao))
            for k in range(len(e)):
                pr.append((float(e[k]), float(c[k])))
            ao += 2 * l + 1
    return Basis(np.array(sh, dtype=SHELL_DTYPE), np.array(pr, dtype=PRIM_DTYPE),
                 np.ascontiguousarray(coords, dtype=np.float64), ao, meta)


# ----------------------------------------------------------------------------- geometry
def _water_monomer() -> np.ndarray:
    r = 0.96
    th = math.radians(104.5)
    return np.array([[0.0, 0.0, 0.0],
                     [r * math.sin(th / 2), 0.0, r * math.cos(th / 2)],
                     [-r * math.sin(th / 2), 0.0, r * math.cos(th / 2)]])  # Angstrom; O,H,H


def _rotation(rng: np.random.Generator) -> np.ndarray:
    q = rng.standard_normal(4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def water_lattice(rng: np.random.Generator, dims: tuple[int, int, int]) -> np.ndarray:
    """Molecules on a 3.0 A cubic lattice, last index fastest; per molecule: orientation, then shift."""
    mono = _water_monomer()
    out = []
    for ix in range(dims[0]):
        for iy in range(dims[1]):
            for iz in range(dims[2]):
                R = _rotation(rng)
                shift = rng.uniform(-0.15, 0.15, 3)
                origin = 3.0 * np.array([ix, iy, iz], dtype=np.float64) + shift
                out.append(mono @ R.T + origin)
    return np.concatenate(out, axis=0) * ANGSTROM


def water_dimer(rng: np.random.Generator) -> np.ndarray:
    mono = _water_monomer()
    m1 = mono @ _rotation(rng).T
    m2 = mono @ _rotation(rng).T + np.array([2.9, 0.0, 0.0])
    xyz = np.concatenate([m1, m2], axis=0)
    xyz = xyz + rng.normal(0.0, 0.02, xyz.shape)
    return xyz * ANGSTROM


# ----------------------------------------------------------------------------- basis recipes
def _even_tempered(rng, l, K, a0, r, jitter=True, coefs=None):
    if jitter:
        a0 = a0 * math.exp(rng.uniform(-0.1, 0.1))
    e = a0 * r ** np.arange(K, dtype=np.float64)
    c = rng.uniform(0.2, 1.0, K) if coefs is None else coefs
    return (l, e, normalise(l, e, c))


def _basis_minimal(rng):
    """cfg0: O 1s,2s,2p ; H 1s, all K=3, seeded a0 in [0.1,130], r in [3,6]."""
    def draw(l):
        a0 = math.exp(rng.uniform(math.log(0.1), math.log(130.0)))
        r = rng.uniform(3.0, 6.0)
        e = a0 * r ** np.arange(3, dtype=np.float64)
        c = rng.uniform(0.2, 1.0, 3)
        return (l, e, normalise(l, e, c))
    o = [draw(0), draw(0), draw(1)]
    h = [draw(0)]
    return o, h


def _basis_dzp(rng):
    """cfg2: O 3s2p1d (core s K=6), H 2s1p."""
    o = [_even_tempered(rng, 0, 6, 7.0, 3.2), _even_tempered(rng, 0, 3, 0.9, 3.4), _even_tempered(rng, 0, 1, 0.28, 1.0),
         _even_tempered(rng, 1, 3, 0.9, 3.6), _even_tempered(rng, 1, 1, 0.25, 1.0),
         _even_tempered(rng, 2, 1, 0.9, 1.0)]
    h = [_even_tempered(rng, 0, 3, 0.6, 4.0), _even_tempered(rng, 0, 1, 0.16, 1.0),
         _even_tempered(rng, 1, 1, 1.0, 1.0)]
    return o, h


def _basis_tz(rng):
    """cfg3/cfg4: O 4s3p2d1f (two K=8 general-contraction-like s shells on the same exponents), H 3s2p1d."""
    s1 = _even_tempered(rng, 0, 8, 6.0, 2.9)
    c2 = rng.uniform(0.2, 1.0, 8)
    c2[4:] *= -1.0  # negative on the four tightest (largest exponents are the last four: a0*r^i ascending)
    s2 = (0, s1[1].copy(), normalise(0, s1[1], c2))
    o = [s1, s2, _even_tempered(rng, 0, 1, 0.9, 1.0), _even_tempered(rng, 0, 1, 0.25, 1.0),
         _even_tempered(rng, 1, 3, 2.0, 3.5), _even_tempered(rng, 1, 1, 0.6, 1.0), _even_tempered(rng, 1, 1, 0.2, 1.0),
         _even_tempered(rng, 2, 1, 1.8, 1.0), _even_tempered(rng, 2, 1, 0.55, 1.0),
         _even_tempered(rng, 3, 1, 1.2, 1.0)]
    h = [_even_tempered(rng, 0, 3, 1.1, 4.6), _even_tempered(rng, 0, 1, 0.32, 1.0), _even_tempered(rng, 0, 1, 0.10, 1.0),
         _even_tempered(rng, 1, 1, 1.3, 1.0), _even_tempered(rng, 1, 1, 0.38, 1.0),
         _even_tempered(rng, 2, 1, 1.0, 1.0)]
    return o, h


def _density_cct(rng, nao, ncol):
    C = rng.standard_normal((nao, ncol)) / math.sqrt(nao)
    return np.ascontiguousarray(C @ C.T)


def water_cluster(dims, basis_kind: str, seed: int, name: str):
    """Generic builder used by cfg2/3/4 and by reduced-size test variants (same recipe, other lattice)."""
    rng = np.random.default_rng(seed)
    xyz = water_lattice(rng, dims)
    o, h = {"dzp": _basis_dzp, "tz": _basis_tz, "min": _basis_minimal}[basis_kind](rng)
    nw = dims[0] * dims[1] * dims[2]
    basis = _assemble([o, h, h] * nw, xyz, {"name": name, "n_water": nw, "basis": basis_kind, "seed": seed})
    D = _density_cct(rng, basis.nao, 5 * nw)
    return basis, D


def cfg0():
    """Water dimer, minimal-like K=3 basis, 14 functions, D = C C^T with C 14x10, tau = 0."""
    rng = np.random.default_rng(SEED0 + 0)
    xyz = water_dimer(rng)
    o, h = _basis_minimal(rng)
    basis = _assemble([o, h, h] * 2, xyz, {"name": "cfg0", "n_water": 2, "basis": "min", "seed": SEED0})
    D = _density_cct(rng, basis.nao, 10)
    return basis, D, 0.0


def cfg2():
    b, D = water_cluster((2, 2, 2), "dzp", SEED0 + 2, "cfg2")
    return b, D, 1e-13


def cfg3():
    b, D = water_cluster((4, 4, 2), "tz", SEED0 + 3, "cfg3")
    return b, D, 1e-13


def cfg4():
    b, D = water_cluster((4, 2, 2), "tz", SEED0 + 4, "cfg4")
    return b, D, 1e-13


# ----------------------------------------------------------------------------- chain workload
def _basis_spd(rng, scale):
    """Polarised split-valence-like heavy atom: s(K=6) core, s(3)+s(1) and p(3)+p(1) valence, one d; seeded synthetic
    even-tempered exponents, `scale` separates the element kinds (no real basis-set data)."""
    return [_even_tempered(rng, 0, 6, 9.0 * scale, 3.1), _even_tempered(rng, 0, 3, 0.9 * scale, 3.3), _even_tempered(rng, 0, 1, 0.22 * scale, 1.0),
            _even_tempered(rng, 1, 3, 0.9 * scale, 3.4), _even_tempered(rng, 1, 1, 0.2 * scale, 1.0),
            _even_tempered(rng, 2, 1, 0.8, 1.0)]


def chain(n_res: int = 30, seed: int = SEED0 + 5, thr: float = 1e-10):
    """Long, spatially extended system with the shapes of the paper's polyglycine set (Table I: Gly_30 with
    a polarised double-zeta basis has 213 atoms and 1878 functions): a zigzag chain of n_res residues of 4 heavy atoms
    (N, C, C, O kinds) and 3 hydrogens, 3.63 A per residue, terminated by H and OH; heavy atoms 3s2p1d (core s contracted
    over 6 primitives), hydrogen 2s; spherical functions.  Here screening decides the time (tau = 1e-10 as in the paper).
    The geometry and all basis-set numbers are synthetic stand-ins: the paper's test set is not in this container."""
    rng = np.random.default_rng(seed)
    tmpl = [("N", (0.00, 0.30, 0.0)), ("H", (0.00, 1.30, 0.0)), ("C", (1.21, -0.45, 0.0)), ("H", (1.21, -1.10, 0.88)),
            ("H", (1.21, -1.10, -0.88)), ("C", (2.42, 0.35, 0.0)), ("O", (2.42, 1.58, 0.0))]
    kinds, xyz = [], []
    for i in range(n_res):
        sgn = 1.0 if i % 2 == 0 else -1.0
        for k, (x, y, z) in tmpl:
            kinds.append(k); xyz.append((3.63 * i + x, sgn * y, z))
    sgn = 1.0 if (n_res - 1) % 2 == 0 else -1.0
    kinds += ["H", "O", "H"]
    xyz += [(-0.90, -0.15, 0.0), (3.63 * (n_res - 1) + 3.60, -sgn * 0.35, 0.0), (3.63 * (n_res - 1) + 4.15, sgn * 0.45, 0.0)]
    xyz = (np.array(xyz) + rng.normal(0.0, 0.03, (len(xyz), 3))) * ANGSTROM
    shells = {"C": _basis_spd(rng, 1.0), "N": _basis_spd(rng, 1.35), "O": _basis_spd(rng, 1.75),
              "H": [_even_tempered(rng, 0, 3, 0.45, 4.2), _even_tempered(rng, 0, 1, 0.16, 1.0)]}
    basis = _assemble([shells[k] for k in kinds], xyz, {"name": f"chain{n_res}", "n_res": n_res, "basis": "spd", "seed": seed})
    D = _density_cct(rng, basis.nao, 15 * n_res + 5)
    return basis, D, thr


# ----------------------------------------------------------------------------- cfg1: ERI class microbenchmark
def canonical_classes(lmax: int = 4) -> list[tuple[int, int, int, int]]:
    """(la,lb,lc,ld) with la>=lb, lc>=ld, (la,lb)>=(lc,ld); 120 classes for lmax=4."""
    out = []
    for la in range(lmax + 1):
        for lb in range(la + 1):
            for lc in range(la + 1):
                for ld in range(lc + 1):
                    if (lc, ld) <= (la, lb):
                        out.append((la, lb, lc, ld))
    return out


def cfg1_class(cls: tuple[int, int, int, int], K: int, nquartets: int = 100_000, pool: int = 32):
    """Pools of `pool` shells per distinct l (own centres in a 10 Bohr box), explicit quartet list.

    Returns (basis, D, quartets[n,4] int32 shell ids).  Quartets are digested as an explicit list:
    six updates each, no symmetry factor, no final symmetrisation."""
    classes = canonical_classes()
    cid = classes.index(tuple(cls))
    rng = np.random.default_rng(SEED0 + 1 + 1000 * cid + K)
    ls = sorted(set(cls))
    atom_shells, coords, pools = [], [], {}
    for l in ls:
        ids = []
        for _ in range(pool):
            centre = rng.uniform(0.0, 10.0, 3)
            e = np.sort(np.exp(rng.uniform(math.log(0.05), math.log(50.0), K)))[::-1].copy()
            c = rng.uniform(0.2, 1.0, K)
            ids.append(len(atom_shells))
            atom_shells.append([(l, e, normalise(l, e, c))])
            coords.append(centre)
        pools[l] = np.array(ids, dtype=np.int32)
    basis = _assemble(atom_shells, np.array(coords), {"name": f"cfg1_{cls}_K{K}", "class": tuple(cls), "K": K})
    q = np.empty((nquartets, 4), dtype=np.int32)
    for pos, l in enumerate(cls):
        q[:, pos] = pools[l][rng.integers(0, pool, nquartets)]
    G = rng.standard_normal((basis.nao, basis.nao)) / math.sqrt(basis.nao)
    D = np.ascontiguousarray(0.5 * (G + G.T))
    return basis, D, np.ascontiguousarray(q)


def subcluster(basis: Basis, n_water: int) -> Basis:
    """First n_water molecules of a water cluster (same basis, same geometry) -- used for the cfg4 oracle parity."""
    natm = 3 * n_water
    keep = basis.shells["atom"] < natm
    sh = basis.shells[keep].copy()
    nprim = int(sh["prim_off"][-1] + sh["nprim"][-1])
    nao = int(sh["ao_off"][-1] + 2 * sh["l"][-1] + 1)
    meta = dict(basis.meta)
    meta["n_water"] = n_water
    return Basis(sh, basis.prims[:nprim].copy(), basis.coords[:natm].copy(), nao, meta)

"""ORACLE (test infrastructure): Cartesian -> real-solid-harmonic matrices, reading R3 of SURVEY.md 8(c).

Definition used: Y_lm(r) = r^l * y_lm(theta, phi), y_lm the REAL spherical harmonic, unit-normalised on the
sphere, m = -l..+l for every l (so l=1 is y,z,x):
    m > 0 : sqrt(2) (-1)^m Re Y_l^m      m < 0 : sqrt(2) (-1)^m Im Y_l^|m|      m = 0 : Y_l^0
with Y_l^m the complex spherical harmonic of scipy (`scipy.special.sph_harm_y`, Condon-Shortley phase).

Route (deliberately different from the library's closed formula): Y_lm is a homogeneous polynomial of degree l,
so its expansion coefficients in the nc(l) monomials x^lx y^ly z^lz are found by solving an (over-determined,
consistent) linear system on sample points, evaluating the left side from the definition above.  Small
coefficients (< 1e-13) are exact zeros and are snapped to 0.

Cartesian component order inside a shell: lx descending, then ly descending (xx,xy,xz,yy,yz,zz).
"""
from __future__ import annotations

import functools

import numpy as np
from scipy.special import sph_harm_y


def cart_powers(l: int) -> list[tuple[int, int, int]]:
    return [(lx, ly, l - lx - ly) for lx in range(l, -1, -1) for ly in range(l - lx, -1, -1)]


def real_solid_harmonic(l: int, m: int, xyz: np.ndarray) -> np.ndarray:
    x, y, z = xyz[:, 0], xyz[:, 1], xyz[:, 2]
    r = np.sqrt(x * x + y * y + z * z)
    theta = np.arccos(z / r)
    phi = np.arctan2(y, x)
    Y = sph_harm_y(l, abs(m), theta, phi)
    if m > 0:
        ang = np.sqrt(2.0) * (-1) ** m * Y.real
    elif m < 0:
        ang = np.sqrt(2.0) * (-1) ** m * Y.imag
    else:
        ang = Y.real
    return r ** l * ang


@functools.lru_cache(maxsize=None)
def c2s(l: int) -> np.ndarray:
    """ns(l) x nc(l) matrix T with Y_lm = sum_c T[m+l, c] x^lx y^ly z^lz."""
    rng = np.random.default_rng(12345 + l)
    pts = rng.standard_normal((40 * (l + 1) * (l + 2), 3))
    pts /= np.linalg.norm(pts, axis=1)[:, None]
    pts *= rng.uniform(0.7, 1.3, pts.shape[0])[:, None]
    pw = cart_powers(l)
    M = np.stack([pts[:, 0] ** a * pts[:, 1] ** b * pts[:, 2] ** c for (a, b, c) in pw], axis=1)
    T = np.empty((2 * l + 1, len(pw)))
    for m in range(-l, l + 1):
        sol, *_ = np.linalg.lstsq(M, real_solid_harmonic(l, m, pts), rcond=None)
        T[m + l] = sol
    T[np.abs(T) < 1e-13] = 0.0
    return np.ascontiguousarray(T)

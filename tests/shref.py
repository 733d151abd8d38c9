"""Test-side numpy helpers, independent of BOTH the oracle and the CUDA path.

They evaluate real spherical harmonics through scipy's associated Legendre functions, integrate on
fine Gauss-Legendre x uniform-phi grids, and build real-basis Wigner-D matrices by projection.
They are the "something other than itself" the oracle is pinned to (brute-force quadrature,
equivariance), and are slow on purpose.

Convention (readings R1/R2; PAPER.md:663 Eq.(C1)): orthonormal on S^2, no
Condon-Shortley phase, order m=-l..l, flat index l*l+l+m.
"""
from __future__ import annotations

import math

import numpy as np
from scipy.special import lpmv


def lm_index(l: int, m: int) -> int:
    return l * l + l + m


def norm_legendre(l: int, m: int, x: np.ndarray) -> np.ndarray:
    """Pt_l^m(x) = sqrt((2l+1)/(4pi) (l-m)!/(l+m)!) P_l^m(x), P_l^m without Condon-Shortley phase."""
    n = math.sqrt((2 * l + 1) / (4 * math.pi) * math.factorial(l - m) / math.factorial(l + m))
    return n * ((-1) ** m) * lpmv(m, l, x)  # scipy's lpmv carries the CS phase; remove it


def real_sh(lmax: int, theta: np.ndarray, phi: np.ndarray) -> np.ndarray:
    """Y[..., (lmax+1)^2] at polar angle theta and azimuth phi (broadcast together)."""
    theta, phi = np.broadcast_arrays(np.asarray(theta, float), np.asarray(phi, float))
    x = np.cos(theta)
    out = np.zeros(theta.shape + ((lmax + 1) ** 2,))
    s2 = math.sqrt(2.0)
    for l in range(lmax + 1):
        out[..., lm_index(l, 0)] = norm_legendre(l, 0, x)
        for m in range(1, l + 1):
            p = norm_legendre(l, m, x)
            out[..., lm_index(l, m)] = s2 * p * np.cos(m * phi)
            out[..., lm_index(l, -m)] = s2 * p * np.sin(m * phi)
    return out


def real_sh_xyz(lmax: int, xyz: np.ndarray) -> np.ndarray:
    xyz = np.asarray(xyz, float)
    r = np.linalg.norm(xyz, axis=-1)
    theta = np.arccos(np.clip(xyz[..., 2] / r, -1.0, 1.0))
    phi = np.arctan2(xyz[..., 1], xyz[..., 0])
    return real_sh(lmax, theta, phi)


def real_sh_surface_grad(lmax: int, theta: np.ndarray, phi: np.ndarray, h: float = 1e-3):
    """(dY/dtheta, (1/sin theta) dY/dphi) by 6th-order central differences (brute force on purpose)."""
    theta, phi = np.broadcast_arrays(np.asarray(theta, float), np.asarray(phi, float))
    c = np.array([-1 / 60, 3 / 20, -3 / 4, 0.0, 3 / 4, -3 / 20, 1 / 60])
    dth = sum(ck * real_sh(lmax, theta + k * h, phi) for ck, k in zip(c, range(-3, 4))) / h
    dph = sum(ck * real_sh(lmax, theta, phi + k * h) for ck, k in zip(c, range(-3, 4))) / h
    return dth, dph / np.sin(theta)[..., None]


def sphere_grid(n_theta: int, n_phi: int):
    """Gauss-Legendre in cos(theta) x uniform phi; returns theta[U,1], phi[1,V], weights[U,V] (sum 4pi)."""
    x, w = np.polynomial.legendre.leggauss(n_theta)
    theta = np.arccos(x)[:, None]
    phi = (2 * np.pi * np.arange(n_phi) / n_phi)[None, :]
    wt = w[:, None] * np.full((1, n_phi), 2 * np.pi / n_phi)
    return theta, phi, wt


def real_gaunt_bruteforce(lmax: int, lmax_out: int, n_theta: int = 40, n_phi: int = 81) -> np.ndarray:
    th, ph, w = sphere_grid(n_theta, n_phi)
    Y = real_sh(max(lmax, lmax_out), th, ph)
    Yi = Y[..., : (lmax + 1) ** 2]
    Yo = Y[..., : (lmax_out + 1) ** 2]
    return np.einsum("uv,uva,uvb,uvc->abc", w, Yi, Yi, Yo, optimize=True)


def real_curl_bruteforce(lmax: int, lmax_out: int, n_theta: int = 40, n_phi: int = 81) -> np.ndarray:
    """Q(a,b;c) = int r.[grad Y_a x grad Y_b] Y_c dOmega
              = int (dth Y_a * (1/sin) dph Y_b - (1/sin) dph Y_a * dth Y_b) Y_c dOmega   (Eq.(11))."""
    th, ph, w = sphere_grid(n_theta, n_phi)
    Yo = real_sh(lmax_out, th, ph)
    dth, dph = real_sh_surface_grad(lmax, th, ph)
    t1 = np.einsum("uv,uva,uvb,uvc->abc", w, dth, dph, Yo, optimize=True)
    return t1 - t1.transpose(1, 0, 2)


def random_rotation(rng: np.random.Generator) -> np.ndarray:
    q = rng.standard_normal(4)
    q /= np.linalg.norm(q)
    a, b, c, d = q
    return np.array([
        [a * a + b * b - c * c - d * d, 2 * (b * c - a * d), 2 * (b * d + a * c)],
        [2 * (b * c + a * d), a * a - b * b + c * c - d * d, 2 * (c * d - a * b)],
        [2 * (b * d - a * c), 2 * (c * d + a * b), a * a - b * b - c * c + d * d],
    ])


def wigner_D_real(lmax: int, R: np.ndarray) -> np.ndarray:
    """D[a,b] = int Y_a(R r) Y_b(r) dOmega on an exact grid: coefficients transform as h' = D h when the
    field is rotated actively by R, and Y(R r) = D Y(r).  Block diagonal in l (checked by the tests)."""
    th, ph, w = sphere_grid(lmax + 2, 2 * lmax + 3)
    Y = real_sh(lmax, th, ph)
    xyz = np.stack([np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph), np.cos(th) * np.ones_like(ph)], -1)
    YR = real_sh_xyz(lmax, xyz @ R.T)
    return np.einsum("uv,uva,uvb->ab", w, YR, Y, optimize=True)


def grid_pipeline_onsite(Ha: np.ndarray, Hb: np.ndarray, lmax: int, lmax_out: int, odd: bool,
                         n_theta: int = 48, n_phi: int = 97) -> np.ndarray:
    """Brute-force fine-grid evaluation of T[lm] for one channel: even = int (A B) Y_lm, odd = int {A,B} Y_lm.
    Ha, Hb: [..., (lmax+1)^2].  Returns [..., (lmax_out+1)^2]."""
    th, ph, w = sphere_grid(n_theta, n_phi)
    Yo = real_sh(lmax_out, th, ph)
    if not odd:
        Y = real_sh(lmax, th, ph)
        fa = np.einsum("uva,...a->...uv", Y, Ha)
        fb = np.einsum("uva,...a->...uv", Y, Hb)
        S = fa * fb
    else:
        dth, dph = real_sh_surface_grad(lmax, th, ph)
        a_t = np.einsum("uva,...a->...uv", dth, Ha)
        a_p = np.einsum("uva,...a->...uv", dph, Ha)
        b_t = np.einsum("uva,...a->...uv", dth, Hb)
        b_p = np.einsum("uva,...a->...uv", dph, Hb)
        S = a_t * b_p - a_p * b_t
    return np.einsum("uv,...uv,uvc->...c", w, S, Yo, optimize=True)

"""Pins of the nu-body oracle (oracle_onsite_nbody, end of Sec. VI), CPU only.

Pinned to: brute-force fine-grid quadrature of the pointwise product of nu fields (tests/shref.py, independent
code), the closed form Y_10^3 = (3/4pi)^(3/2) (3/5 z + 2/5 P_3(z)) (z^3 in Legendre polynomials), the constant
field, the reduction to oracle_onsite at nu = 2, symmetry under permutation of the factors, and SO(3) equivariance
with Wigner-D matrices built by projection.
"""
import math

import numpy as np
import pytest

from oracle import cgtp_oracle as orc
from paper_2605_15073_b200 import synthetic
from tests import shref


def _fine_grid_reference(inp, n_theta=40, n_phi=81):
    """Project -> evaluate every field on a fine grid -> multiply -> integrate against Y_lm -> project."""
    th, ph, w = shref.sphere_grid(n_theta, n_phi)
    Y = shref.real_sh(inp.lmax, th, ph)
    Yo = shref.real_sh(inp.lmax_out, th, ph)
    S = None
    for s in range(inp.nu):
        H = np.einsum("cn,bnl->bcl", inp.W_in[s].astype(float), inp.X[s].astype(float))
        f = np.einsum("uva,bca->bcuv", Y, H)
        S = f if S is None else S * f
    T = np.einsum("uv,bcuv,uvo->bco", w, S, Yo, optimize=True)
    return np.einsum("nc,bco->bno", inp.W_out.astype(float), T)


@pytest.mark.parametrize("nu,lmax,lmax_out", [(3, 2, 3), (3, 2, 6), (4, 1, 4), (4, 2, 2), (2, 3, 4), (3, 3, 0), (1, 3, 2)])
def test_nbody_vs_fine_grid_quadrature(nu, lmax, lmax_out):
    inp = synthetic.make_nbody(nu, lmax, lmax_out, N=3, C=4, batch=4, seed=100 * nu + 10 * lmax + lmax_out)
    got = orc.onsite_nbody(inp.X, inp.W_in, inp.W_out, lmax, lmax_out)
    ref = _fine_grid_reference(inp)
    assert np.abs(ref).max() > 1e-2
    assert np.abs(got - ref).max() / np.abs(ref).max() < 1e-12


def test_nbody_closed_form_cube_of_Y10_and_constant():
    # Y_10 = sqrt(3/4pi) z and z^3 = 3/5 P_1(z) + 2/5 P_3(z), Y_l0 = sqrt((2l+1)/4pi) P_l:
    #   Y_10^3 = (3/4pi)^(3/2) [ 3/5 sqrt(4pi/3) Y_10 + 2/5 sqrt(4pi/7) Y_30 ]
    lmax, lmax_out, nu = 1, 3, 3
    X = np.zeros((nu, 1, 1, 4))
    X[:, 0, 0, shref.lm_index(1, 0)] = 1.0
    W_in = np.ones((nu, 1, 1))
    W_out = np.ones((1, 1))
    got = orc.onsite_nbody(X, W_in, W_out, lmax, lmax_out)[0, 0]
    want = np.zeros(16)
    k = (3 / (4 * math.pi)) ** 1.5
    want[shref.lm_index(1, 0)] = k * 0.6 * math.sqrt(4 * math.pi / 3)
    want[shref.lm_index(3, 0)] = k * 0.4 * math.sqrt(4 * math.pi / 7)
    assert np.abs(got - want).max() < 1e-14
    # constant fields a_s Y_00: product = prod(a_s) (4pi)^(-(nu-1)/2) Y_00
    for nu in (1, 2, 3, 4, 5):
        a = np.arange(2, 2 + nu, dtype=float)
        X = np.zeros((nu, 1, 1, 9))
        X[:, 0, 0, 0] = a
        got = orc.onsite_nbody(X, np.ones((nu, 1, 1)), np.ones((1, 1)), 2, 2)[0, 0]
        want = np.zeros(9)
        want[0] = a.prod() * (4 * math.pi) ** (-(nu - 1) / 2)
        assert np.abs(got - want).max() < 1e-13 * want[0]


def test_nbody_nu2_reduces_to_onsite_even_sector():
    lmax, lmax_out = 3, 4
    inp = synthetic.make_onsite(lmax, lmax_out, N=4, C=5, batch=6, seed=3, parity_mask=np.zeros(5, np.uint8))
    ref = orc.onsite(inp.A, inp.B, inp.W_a, inp.W_b, inp.W_out, lmax, lmax_out, inp.parity_mask)[:, 0]
    got = orc.onsite_nbody(np.stack([inp.A, inp.B]), np.stack([inp.W_a, inp.W_b]), inp.W_out, lmax, lmax_out)
    assert np.abs(got - ref).max() <= 1e-14 * np.abs(ref).max()


def test_nbody_factor_permutation_and_multilinearity():
    nu, lmax, lmax_out = 4, 2, 3
    inp = synthetic.make_nbody(nu, lmax, lmax_out, N=3, C=4, batch=3, seed=9)
    base = orc.onsite_nbody(inp.X, inp.W_in, inp.W_out, lmax, lmax_out)
    perm = [2, 0, 3, 1]
    got = orc.onsite_nbody(inp.X[perm], inp.W_in[perm], inp.W_out, lmax, lmax_out)
    assert np.abs(got - base).max() < 1e-13 * np.abs(base).max()
    X2 = inp.X.astype(float).copy()
    X2[1] *= -2.5
    got = orc.onsite_nbody(X2, inp.W_in, inp.W_out, lmax, lmax_out)
    assert np.abs(got + 2.5 * base).max() < 1e-13 * np.abs(base).max()


def test_nbody_equivariance_and_inversion():
    nu, lmax, lmax_out = 3, 2, 4
    inp = synthetic.make_nbody(nu, lmax, lmax_out, N=3, C=4, batch=3, seed=11)
    base = orc.onsite_nbody(inp.X, inp.W_in, inp.W_out, lmax, lmax_out)
    rng = np.random.default_rng(5)
    R = shref.random_rotation(rng)
    D = shref.wigner_D_real(lmax_out, R)
    L2 = (lmax + 1) ** 2
    Xr = np.einsum("ab,...b->...a", D[:L2, :L2], inp.X.astype(float))
    got = orc.onsite_nbody(Xr, inp.W_in, inp.W_out, lmax, lmax_out)
    want = np.einsum("ab,...b->...a", D, base)
    assert np.abs(got - want).max() < 1e-12 * np.abs(base).max()
    # inversion: natural-parity inputs (-1)^l; a product of natural-parity fields has natural parity
    sgn_in = np.array([(-1.0) ** l for l in range(lmax + 1) for _ in range(2 * l + 1)])
    sgn_out = np.array([(-1.0) ** l for l in range(lmax_out + 1) for _ in range(2 * l + 1)])
    got = orc.onsite_nbody(inp.X * sgn_in, inp.W_in, inp.W_out, lmax, lmax_out)
    assert np.abs(got - base * sgn_out).max() < 1e-13 * np.abs(base).max()

"""Pins of the FP64 oracle against things other than itself (all CPU, -m "not gpu").

Each test names the passage of PAPER.md (= /root/reference/PAPER.md) or the mathematical fact it
rests on.  A plausible mistake in the oracle (dropped term, wrong sign/index, transposed operand)
must fail at least one of them.
"""
import math
import os

import numpy as np
import pytest
import sympy
from sympy.physics.wigner import clebsch_gordan as sy_cg
from sympy.physics.wigner import gaunt as sy_gaunt
from sympy.physics.wigner import wigner_3j as sy_3j

from oracle import cgtp_oracle as orc
from tests import shref

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------------------------------------
# Wigner 3j / CG against sympy's exact rational arithmetic
# ---------------------------------------------------------------------------------------------
def _random_3j_args(rng, lo, hi, n):
    out = []
    while len(out) < n:
        j1, j2 = rng.integers(lo, hi + 1, 2)
        j3 = rng.integers(abs(j1 - j2), j1 + j2 + 1)
        m1 = rng.integers(-j1, j1 + 1)
        m2 = rng.integers(-j2, j2 + 1)
        m3 = -(m1 + m2)
        if abs(m3) <= j3:
            out.append(tuple(int(v) for v in (j1, j2, j3, m1, m2, m3)))
    return out


def test_wigner3j_all_small_vs_sympy():
    worst = 0.0
    for j1 in range(0, 4):
        for j2 in range(0, 4):
            for j3 in range(abs(j1 - j2), j1 + j2 + 1):
                for m1 in range(-j1, j1 + 1):
                    for m2 in range(-j2, j2 + 1):
                        m3 = -(m1 + m2)
                        if abs(m3) > j3:
                            continue
                        ref = float(sy_3j(j1, j2, j3, m1, m2, m3))
                        worst = max(worst, abs(orc.wigner3j(j1, j2, j3, m1, m2, m3) - ref))
    assert worst < 1e-14


def test_wigner3j_large_l_vs_sympy():
    rng = np.random.default_rng(7)
    cases = _random_3j_args(rng, 10, 20, 60)
    cases += [(20, 20, 20, 0, 0, 0), (20, 20, 20, 5, -12, 7), (20, 20, 19, -1, 1, 0), (20, 19, 2, -1, 1, 0),
              (20, 20, 40, 20, 20, -40), (20, 20, 0, 7, -7, 0)]
    worst = 0.0
    for c in cases:
        ref = float(sy_3j(*c).evalf(30))
        worst = max(worst, abs(orc.wigner3j(*c) - ref))
    assert worst < 1e-12, worst


def test_cg_vs_sympy_and_orthogonality():
    rng = np.random.default_rng(3)
    for (j1, j2, j3, m1, m2, m3) in _random_3j_args(rng, 0, 8, 60):
        ref = float(sy_cg(j1, j2, j3, m1, m2, -m3).evalf(30))
        assert abs(orc.cg(j1, m1, j2, m2, j3, -m3) - ref) < 1e-13
    # sum_{m1 m2} <l1m1 l2m2|lm> <l1m1 l2m2|l'm'> = delta
    l1, l2 = 3, 2
    for l in range(abs(l1 - l2), l1 + l2 + 1):
        for lp in range(abs(l1 - l2), l1 + l2 + 1):
            for m in range(-min(l, lp), min(l, lp) + 1):
                s = sum(orc.cg(l1, m1, l2, m - m1, l, m) * orc.cg(l1, m1, l2, m - m1, lp, m)
                        for m1 in range(-l1, l1 + 1) if abs(m - m1) <= l2)
                assert abs(s - (1.0 if l == lp else 0.0)) < 1e-13


def test_eq6_closed_form_vs_racah_and_sympy():
    """PAPER.md:59 Eq.(6)-(7), :70 Eq.(8)."""
    for l1 in range(0, 7):
        for l2 in range(0, 7):
            for l in range(abs(l1 - l2), l1 + l2 + 1):
                closed = orc.cg000_closed(l1, l2, l)
                assert abs(closed - orc.cg(l1, 0, l2, 0, l, 0)) < 1e-13
                if (l1 + l2 + l) % 2:
                    assert closed == 0.0
    for (l1, l2, l) in [(1, 1, 2), (2, 2, 2), (3, 2, 5), (4, 4, 0), (5, 3, 4)]:
        assert abs(orc.cg000_closed(l1, l2, l) - float(sy_cg(l1, l2, l, 0, 0, 0))) < 1e-14


# ---------------------------------------------------------------------------------------------
# Complex Gaunt Eq.(4)-(5)
# ---------------------------------------------------------------------------------------------
def test_complex_gaunt_vs_sympy_and_special_case():
    """int Y1 Y2 Y3* = (-1)^m3 * sympy.gaunt(l1,l2,l3,m1,m2,-m3)  (PAPER.md:49-:55)."""
    rng = np.random.default_rng(11)
    n = 0
    for (l1, l2, l, m1, m2, m3) in _random_3j_args(rng, 0, 6, 200):
        m = -m3
        ref = float(sy_gaunt(l1, l2, l, m1, m2, -m)) * (-1) ** m
        got = orc.gaunt_complex(l1, m1, l2, m2, l, m)
        assert abs(got - ref) < 1e-13
        n += ref != 0.0
    assert n > 20
    # l1 = 0: Gaunt = delta / sqrt(4 pi)
    for l in range(0, 5):
        for m in range(-l, l + 1):
            assert abs(orc.gaunt_complex(0, 0, l, m, l, m) - 1 / math.sqrt(4 * math.pi)) < 1e-14


# ---------------------------------------------------------------------------------------------
# kappa^-1: printed values and worked example
# ---------------------------------------------------------------------------------------------
def test_kappa_inv_printed_values():
    rows = [ln.split() for ln in open(os.path.join(GOLD, "kappa_inv_printed.txt")) if ln.strip() and ln[0] != "#"]
    assert len(rows) == 6
    for r in rows:
        l1, l2, l, val, digits = int(r[0]), int(r[1]), int(r[2]), float(r[3]), int(r[4])
        got = abs(orc.kappa_inv_imag(l1, l2, l))
        assert abs(got - val) <= 0.5 * 10 ** (-digits) + 1e-12, (l1, l2, l, got, val)
    # the sign of the one printed signed value: +0.690988 i
    assert orc.kappa_inv_imag(1, 1, 1) > 0


def test_worked_example_A11_A13():
    gold = {ln.split()[0]: float(ln.split()[1])
            for ln in open(os.path.join(GOLD, "worked_example_A11_A13.txt")) if ln.strip() and ln[0] != "#"}
    assert abs(gold["Q_imag"] - math.sqrt(3 / (4 * math.pi))) < 1e-15  # fixture typed correctly
    assert abs(orc.q_complex_imag(1, 1, 1, -1, 1, 0) - gold["Q_imag"]) < 1e-14
    assert abs(orc.cg(1, 1, 1, -1, 1, 0) - gold["G"]) < 1e-14
    assert abs(orc.kappa_inv_imag(1, 1, 1) - gold["kappa_inv_imag"]) < 1e-14


def test_kappa_support_and_exchange():
    """Support :583-:585; Q antisymmetric under (l1m1)<->(l2m2), Eq.(10) :101."""
    for l1 in range(0, 5):
        for l2 in range(0, 5):
            for l in range(0, 9):
                k = orc.kappa_inv_imag(l1, l2, l)
                on = l1 >= 1 and l2 >= 1 and abs(l1 - l2) <= l <= l1 + l2 and (l1 + l2 + l) % 2 == 1
                assert (k != 0.0) == on
                if on:
                    for m1 in range(-l1, l1 + 1):
                        for m2 in range(-l2, l2 + 1):
                            if abs(m1 + m2) <= l:
                                q12 = orc.q_complex_imag(l1, m1, l2, m2, l, m1 + m2)
                                q21 = orc.q_complex_imag(l2, m2, l1, m1, l, m1 + m2)
                                assert abs(q12 + q21) < 1e-13


# ---------------------------------------------------------------------------------------------
# Real-basis tables against brute-force quadrature and textbook special cases
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("lmax,lmax_out", [(3, 3), (2, 4)])
def test_real_gaunt_vs_bruteforce_quadrature(lmax, lmax_out):
    G = orc.real_coupling_dense(lmax, lmax_out, False)
    ref = shref.real_gaunt_bruteforce(lmax, lmax_out)
    assert np.abs(G - ref).max() < 1e-12
    assert orc.real_coupling(lmax, lmax_out, False)[4] < 1e-14  # imaginary parts vanish
    if lmax == lmax_out:
        assert np.abs(G - G.transpose(1, 0, 2)).max() < 1e-14
        assert np.abs(G - G.transpose(2, 1, 0)).max() < 1e-13  # totally symmetric


@pytest.mark.parametrize("lmax,lmax_out", [(3, 3), (2, 4)])
def test_real_curl_vs_bruteforce_quadrature(lmax, lmax_out):
    Q = orc.real_coupling_dense(lmax, lmax_out, True)
    ref = shref.real_curl_bruteforce(lmax, lmax_out)
    assert np.abs(Q - ref).max() < 1e-9  # finite-difference gradient in the brute force
    assert np.abs(Q + Q.transpose(1, 0, 2)).max() < 1e-14  # antisymmetric in the two inputs
    assert orc.real_coupling(lmax, lmax_out, True)[4] < 1e-14
    # odd sector has no l=0 output and no l1=0 / l2=0 input (support rule :585)
    assert np.abs(Q[:, :, 0]).max() == 0.0 and np.abs(Q[0]).max() == 0.0 and np.abs(Q[:, 0]).max() == 0.0


def test_parity_selection_rules():
    """Eq.(8) :70 and Eq.(A7) :560: even table lives on l1+l2+l even, odd table on l1+l2+l odd."""
    deg = lambda idx: np.floor(np.sqrt(idx)).astype(int)
    for odd in (False, True):
        i1, i2, io, val, _ = orc.real_coupling(4, 4, odd)
        s = deg(i1) + deg(i2) + deg(io)
        assert np.all(s % 2 == int(odd))
        assert np.all(np.abs(val) > 1e-12)


def test_cross_and_dot_product_blocks():
    """(1,1,1) block of Qr = sqrt(3/4pi) eps_abc in (y,z,x) order; (1,1,0) block of Gr = delta/sqrt(4pi)."""
    Q = orc.real_coupling_dense(1, 1, True)
    G = orc.real_coupling_dense(1, 1, False)
    rng = np.random.default_rng(5)
    a, b = rng.standard_normal(3), rng.standard_normal(3)  # Cartesian (x,y,z)
    to_sh = lambda v: np.array([v[1], v[2], v[0]])  # (y,z,x) = m=-1,0,+1
    ha, hb = np.zeros(4), np.zeros(4)
    ha[1:], hb[1:] = to_sh(a), to_sh(b)
    cross = np.einsum("abc,a,b->c", Q, ha, hb)
    assert np.abs(cross[1:] - math.sqrt(3 / (4 * math.pi)) * to_sh(np.cross(a, b))).max() < 1e-14
    assert cross[0] == 0.0
    dot = np.einsum("abc,a,b->c", G, ha, hb)
    assert abs(dot[0] - a.dot(b) / math.sqrt(4 * math.pi)) < 1e-14


def test_real_sh_vs_scipy_and_cartesian():
    rng = np.random.default_rng(9)
    for _ in range(20):
        v = rng.standard_normal(3) * rng.uniform(0.5, 4.0)
        got = orc.real_sh(8, v)
        ref = shref.real_sh_xyz(8, v)
        assert np.abs(got - ref).max() < 1e-13
        n = v / np.linalg.norm(v)
        assert abs(got[0] - 1 / math.sqrt(4 * math.pi)) < 1e-15
        assert np.abs(got[1:4] - math.sqrt(3 / (4 * math.pi)) * np.array([n[1], n[2], n[0]])).max() < 1e-14
        # Y(-r) = (-1)^l Y(r)
        neg = orc.real_sh(8, -v)
        sign = np.concatenate([np.full(2 * l + 1, (-1.0) ** l) for l in range(9)])
        assert np.abs(neg - sign * got).max() < 1e-13
    # poles
    assert np.abs(orc.real_sh(4, (0, 0, 2.0)) - shref.real_sh_xyz(4, np.array([0, 0, 2.0]))).max() < 1e-14


def test_real_sh_orthonormal_and_addition_theorem():
    th, ph, w = shref.sphere_grid(12, 25)
    xyz = np.stack([np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph), np.cos(th) * np.ones_like(ph)], -1)
    Y = np.array([[orc.real_sh(6, xyz[u, v]) for v in range(xyz.shape[1])] for u in range(xyz.shape[0])])
    gram = np.einsum("uv,uva,uvb->ab", w, Y, Y)
    assert np.abs(gram - np.eye(49)).max() < 1e-13
    rng = np.random.default_rng(2)
    a, b = rng.standard_normal(3), rng.standard_normal(3)
    a /= np.linalg.norm(a)
    b /= np.linalg.norm(b)
    Ya, Yb = orc.real_sh(6, a), orc.real_sh(6, b)
    for l in range(7):
        s = Ya[l * l:(l + 1) ** 2].dot(Yb[l * l:(l + 1) ** 2])
        ref = (2 * l + 1) / (4 * math.pi) * float(sympy.legendre(l, a.dot(b)))
        assert abs(s - ref) < 1e-13


def test_nnz_counts_match_selection_rule_count():
    """Every (a,b;c) allowed by triangle + parity + the real-basis azimuthal rule is counted once."""
    for odd in (False, True):
        dense = orc.real_coupling_dense(3, 3, odd)
        ref = shref.real_curl_bruteforce(3, 3) if odd else shref.real_gaunt_bruteforce(3, 3)
        assert (np.abs(dense) > 1e-12).sum() == (np.abs(ref) > 1e-8).sum()
        assert (np.abs(dense) > 1e-12).sum() == orc.real_coupling(3, 3, odd)[0].shape[0]

"""Whole-pipeline pins of the oracle (oracle_onsite / oracle_message / oracle_segments), CPU only.

Pinned to: brute-force fine-grid quadrature of the fields (tests/shref.py, independent code),
SO(3) equivariance with Wigner-D matrices built by projection (PAPER.md:633 App. B test 5, :651),
inversion parity (Table I :86-:93), self-coupled vanishing (Eq.(27) :221, App. B test 6 :637),
single-edge reduction of Eq.(2) to Eq.(1), Parseval, bilinearity, numpy segmentation.
"""
import numpy as np
import pytest

from oracle import cgtp_oracle as orc
from paper_2605_15073_b200 import synthetic
from tests import shref


def _sector_err(got, ref):
    """R14 norm: max|got-ref| / max|ref| per parity sector (axis 1)."""
    return [np.abs(got[:, s] - ref[:, s]).max() / max(np.abs(ref[:, s]).max(), 1e-300) for s in (0, 1)]


def _numpy_reference_onsite(inp, n_theta=40, n_phi=81):
    """Project -> evaluate fields on a fine grid -> product / bracket -> integrate -> project (float64)."""
    Ha = np.einsum("cn,bnl->bcl", inp.W_a.astype(float), inp.A.astype(float))
    Hb = np.einsum("cn,bnl->bcl", inp.W_b.astype(float), inp.B.astype(float))
    Te = shref.grid_pipeline_onsite(Ha, Hb, inp.lmax, inp.lmax_out, False, n_theta, n_phi)
    To = shref.grid_pipeline_onsite(Ha, Hb, inp.lmax, inp.lmax_out, True, n_theta, n_phi)
    m = inp.parity_mask.astype(bool)
    out = np.zeros((inp.batch, 2, inp.N, (inp.lmax_out + 1) ** 2))
    out[:, 0] = np.einsum("nc,bcl->bnl", inp.W_out[:, ~m].astype(float), Te[:, ~m])
    out[:, 1] = np.einsum("nc,bcl->bnl", inp.W_out[:, m].astype(float), To[:, m])
    return out


@pytest.mark.parametrize("lmax,lmax_out", [(2, 2), (3, 3), (2, 4), (3, 1)])
def test_onsite_vs_fine_grid_quadrature(lmax, lmax_out):
    inp = synthetic.make_onsite(lmax, lmax_out, N=3, C=4, batch=5, seed=lmax * 10 + lmax_out,
                                parity_mask=[0, 1, 1, 0])
    got = orc.onsite(inp.A, inp.B, inp.W_a, inp.W_b, inp.W_out, lmax, lmax_out, inp.parity_mask)
    ref = _numpy_reference_onsite(inp)
    e0, e1 = _sector_err(got, ref)
    assert e0 < 1e-12 and e1 < 1e-8, (e0, e1)  # odd sector: finite-difference gradients in the brute force
    assert np.abs(ref[:, 1]).max() > 1e-2 and np.abs(ref[:, 0]).max() > 1e-2


def _rotate_feats(X, D):
    return np.einsum("ab,...b->...a", D, X)


def test_onsite_equivariance_and_inversion():
    lmax = 4
    inp = synthetic.make_onsite(lmax, lmax, N=4, C=6, batch=3, seed=21)
    base = orc.onsite(inp.A, inp.B, inp.W_a, inp.W_b, inp.W_out, lmax, lmax, inp.parity_mask)
    rng = np.random.default_rng(4)
    for _ in range(2):
        R = shref.random_rotation(rng)
        D = shref.wigner_D_real(lmax, R)
        assert np.abs(D @ D.T - np.eye(D.shape[0])).max() < 1e-12
        # block diagonal in l, and D^1 = R in (y,z,x) order
        P = np.array([[0, 1, 0], [0, 0, 1], [1, 0, 0]], float)  # (x,y,z) -> (y,z,x)
        assert np.abs(D[1:4, 1:4] - P @ R @ P.T).max() < 1e-12
        assert np.abs(D[0, 1:]).max() < 1e-12 and np.abs(D[4:9, 1:4]).max() < 1e-12
        rot = orc.onsite(_rotate_feats(inp.A, D), _rotate_feats(inp.B, D), inp.W_a, inp.W_b, inp.W_out,
                         lmax, lmax, inp.parity_mask)
        e0, e1 = _sector_err(rot, _rotate_feats(base, D))
        assert e0 < 1e-12 and e1 < 1e-12
    # inversion: h_lm -> (-1)^l h_lm; sector 0 picks (-1)^l, sector 1 picks -(-1)^l  (Table I :86-:93)
    sign = np.concatenate([np.full(2 * l + 1, (-1.0) ** l) for l in range(lmax + 1)])
    inv = orc.onsite(inp.A * sign, inp.B * sign, inp.W_a, inp.W_b, inp.W_out, lmax, lmax, inp.parity_mask)
    assert np.abs(inv[:, 0] - base[:, 0] * sign).max() < 1e-12
    assert np.abs(inv[:, 1] + base[:, 1] * sign).max() < 1e-12


def test_onsite_exchange_bilinearity_selfcoupling():
    lmax = 3
    inp = synthetic.make_onsite(lmax, lmax, N=4, C=6, batch=4, seed=33)
    f = lambda A, B, Wa, Wb: orc.onsite(A, B, Wa, Wb, inp.W_out, lmax, lmax, inp.parity_mask)
    base = f(inp.A, inp.B, inp.W_a, inp.W_b)
    # exchanging the factors keeps sector 0 and negates sector 1 (Eq.(10) :101)
    sw = f(inp.B, inp.A, inp.W_b, inp.W_a)
    assert np.abs(sw[:, 0] - base[:, 0]).max() < 1e-13 and np.abs(sw[:, 1] + base[:, 1]).max() < 1e-13
    # bilinear in A
    A2 = np.random.default_rng(1).standard_normal(inp.A.shape)
    lin = f(2.0 * inp.A + A2, inp.B, inp.W_a, inp.W_b)
    assert np.abs(lin - (2.0 * base + f(A2, inp.B, inp.W_a, inp.W_b))).max() < 1e-11
    # A = B with symmetric channel mixing (W_a = W_b): odd sector vanishes (Eq.(27) :221, App. B test 6)
    selfc = f(inp.A, inp.A, inp.W_a, inp.W_a)
    assert np.abs(selfc[:, 1]).max() < 1e-13 and np.abs(selfc[:, 0]).max() > 1e-2
    # antisymmetric mixing keeps it alive (:641)
    anti = f(inp.A, inp.A, inp.W_a, inp.W_b)
    assert np.abs(anti[:, 1]).max() > 1e-2
    # odd sector has no l=0 output (support rule :585)
    assert np.abs(base[:, 1, :, 0]).max() == 0.0


def test_onsite_parseval_full_band():
    """lmax_out = 2 lmax: sum_lm T_lm^2 = int (A B)^2 dOmega for one even channel with unit weights."""
    lmax = 2
    rng = np.random.default_rng(8)
    A = rng.standard_normal((1, 1, 9))
    B = rng.standard_normal((1, 1, 9))
    one = np.ones((1, 1))
    out = orc.onsite(A, B, one, one, one, lmax, 2 * lmax, np.zeros(1, np.uint8))
    th, ph, w = shref.sphere_grid(12, 25)
    Y = shref.real_sh(lmax, th, ph)
    fa, fb = Y @ A[0, 0], Y @ B[0, 0]
    assert abs((out[0, 0, 0] ** 2).sum() - (w * (fa * fb) ** 2).sum()) < 1e-12


def test_segments_vs_numpy():
    rng = np.random.default_rng(0)
    nodes = 37
    deg = rng.integers(0, 6, nodes)
    deg[[0, 5, 36]] = 0
    recv = np.repeat(np.arange(nodes), deg)
    snd = rng.integers(0, nodes, recv.shape[0])
    rc, rp = orc.segments(np.stack([snd, recv]), nodes)
    assert rc == 0
    assert np.array_equal(rp, np.searchsorted(recv, np.arange(nodes + 1), side="left"))
    assert np.array_equal(np.diff(rp), deg)
    bad = np.stack([snd, recv[::-1]])
    assert orc.segments(bad, nodes)[0] == 4
    oob = np.stack([snd, recv]).copy()
    oob[0, 0] = nodes
    assert orc.segments(oob, nodes)[0] == 4
    rc, rp = orc.segments(np.zeros((2, 0), np.int64), 3)
    assert rc == 0 and np.array_equal(rp, np.zeros(4, np.int64))


def test_message_single_edge_reduces_to_onsite():
    """One edge j->i: Eq.(2) = Eq.(1) with A^(1) = R~ Y(r_hat) (factor 1) and A^(2) = node feature of j."""
    lmax, N, C = 3, 3, 4
    m = synthetic.make_message(lmax, lmax, N, C, nodes=2, degree=np.array([1, 0]), seed=2, parity_mask=[0, 1, 0, 1])
    assert m.E == 1 and m.edge_index[0, 0] == 1 and m.edge_index[1, 0] == 0
    got = orc.message(m.node_feats, m.edge_index, m.edge_vec, m.edge_radial, m.W_node, m.W_out, lmax, lmax,
                      m.parity_mask)
    Y = shref.real_sh_xyz(lmax, m.edge_vec[0].astype(float))
    # factor 1 enters through an identity "projection": N=C channels carrying R~[c] Y
    A1 = (m.edge_radial[0].astype(float)[:, None] * Y[None, :])[None]  # [1, C, L2]
    Wn = m.W_node.astype(float)
    H2 = np.einsum("cn,nl->cl", Wn, m.node_feats[1].astype(float))[None]  # [1, C, L2]
    eye = np.eye(C)
    ref = orc.onsite(A1, H2, eye, eye, np.pad(m.W_out.astype(float), ((0, C - N), (0, 0))), lmax, lmax, m.parity_mask)
    assert np.abs(got[0] - ref[0][:, :N]).max() < 1e-13
    assert np.abs(got[1]).max() == 0.0  # receiver without edges -> zeros


def test_message_vs_fine_grid_quadrature():
    lmax, N, C = 2, 3, 4
    m = synthetic.make_message(lmax, lmax, N, C, nodes=5, degree=np.array([2, 0, 3, 1, 2]), seed=6,
                               parity_mask=[1, 0, 0, 1])
    got = orc.message(m.node_feats, m.edge_index, m.edge_vec, m.edge_radial, m.W_node, m.W_out, lmax, lmax,
                      m.parity_mask)
    H = np.einsum("cn,jnl->jcl", m.W_node.astype(float), m.node_feats.astype(float))
    T = np.zeros((m.nodes, 2, C, (lmax + 1) ** 2))
    for e in range(m.E):
        j, i = m.edge_index[:, e]
        a = m.edge_radial[e].astype(float)[:, None] * shref.real_sh_xyz(lmax, m.edge_vec[e].astype(float))[None]
        T[i, 0] += shref.grid_pipeline_onsite(a, H[j], lmax, lmax, False, 24, 49)
        T[i, 1] += shref.grid_pipeline_onsite(a, H[j], lmax, lmax, True, 24, 49)
    mk = m.parity_mask.astype(bool)
    ref = np.zeros_like(got)
    ref[:, 0] = np.einsum("nc,icl->inl", m.W_out[:, ~mk].astype(float), T[:, 0][:, ~mk])
    ref[:, 1] = np.einsum("nc,icl->inl", m.W_out[:, mk].astype(float), T[:, 1][:, mk])
    e0, e1 = _sector_err(got, ref)
    assert e0 < 1e-12 and e1 < 1e-8


def test_message_equivariance_inversion_permutation_subset():
    lmax, N, C, nodes = 3, 4, 6, 7
    m = synthetic.make_message(lmax, lmax, N, C, nodes, degree=3, seed=12)
    f = lambda X, ei, ev, er, rl=None: orc.message(X, ei, ev, er, m.W_node, m.W_out, lmax, lmax, m.parity_mask, rl)
    base = f(m.node_feats, m.edge_index, m.edge_vec, m.edge_radial)
    R = shref.random_rotation(np.random.default_rng(3))
    D = shref.wigner_D_real(lmax, R)
    rot = f(_rotate_feats(m.node_feats.astype(float), D), m.edge_index, m.edge_vec.astype(float) @ R.T, m.edge_radial)
    e0, e1 = _sector_err(rot, _rotate_feats(base, D))
    assert e0 < 1e-12 and e1 < 1e-12
    sign = np.concatenate([np.full(2 * l + 1, (-1.0) ** l) for l in range(lmax + 1)])
    inv = f(m.node_feats * sign, m.edge_index, -m.edge_vec, m.edge_radial)
    assert np.abs(inv[:, 0] - base[:, 0] * sign).max() < 1e-12
    assert np.abs(inv[:, 1] + base[:, 1] * sign).max() < 1e-12
    # only the direction of edge_vec matters (R11); duplicate edges add (R16)
    scaled = f(m.node_feats, m.edge_index, m.edge_vec.astype(float) * 3.0, m.edge_radial)
    assert np.abs(scaled - base).max() < 1e-12
    # permuting edges inside a segment changes nothing beyond round-off
    perm = np.arange(m.E).reshape(nodes, 3)[:, ::-1].reshape(-1)
    pm = f(m.node_feats, m.edge_index[:, perm], m.edge_vec[perm], m.edge_radial[perm])
    assert np.abs(pm - base).max() < 1e-12
    # receiver subset = rows of the full result
    sub = f(m.node_feats, m.edge_index, m.edge_vec, m.edge_radial, [5, 0, 2])
    assert np.array_equal(sub, base[[5, 0, 2]])

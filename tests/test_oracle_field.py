"""Pins of the two-field oracle (oracle_message_field; Eq.(28) :236, Sec. VII C f :471), CPU only.

Pinned to: oracle_message (itself pinned to fine-grid quadrature) for edge fields of the form R[e,n] Y(r_e) -- the
special case Eq.(28) generalises; brute-force fine-grid quadrature of the pooled pointwise product / surface-curl
pairing (tests/shref.py, independent code); receivers with one in-edge = oracle_onsite of (edge field, sender
feature); edge order inside a segment; empty receivers; SO(3) equivariance and inversion.
"""
import numpy as np
import pytest

from oracle import cgtp_oracle as orc
from paper_2605_15073_b200 import synthetic
from tests import shref


def _case(lmax, lmax_out, N=3, Ne=2, C=4, nodes=5, degree=3, seed=0):
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, degree, seed=seed)
    XE, W_edge = synthetic.make_edge_field(m, Ne, seed=seed)
    return m, XE, W_edge


def _run(m, XE, W_edge, node_feats=None):
    X = m.node_feats if node_feats is None else node_feats
    return orc.message_field(X, m.edge_index, XE, W_edge, m.W_node, m.W_out, m.lmax, m.lmax_out, m.parity_mask)


@pytest.mark.parametrize("lmax,lmax_out", [(2, 2), (3, 4), (1, 2)])
def test_field_reduces_to_message_for_RY_edge_fields(lmax, lmax_out):
    # I^(E)[e,n,lm] = R[e,n] Y_lm(r_e)  =>  a[e,c,lm] = (W_edge R)[e,c] Y_lm(r_e): Eq.(2) with edge_radial = R W_edge^T
    m, _, W_edge = _case(lmax, lmax_out, seed=10 * lmax + lmax_out)
    rng = np.random.default_rng(1)
    Ne = W_edge.shape[1]
    R = rng.standard_normal((m.E, Ne))
    Y = shref.real_sh_xyz(lmax, m.edge_vec.astype(float) / np.linalg.norm(m.edge_vec.astype(float), axis=1, keepdims=True))
    XE = R[:, :, None] * Y[:, None, :]
    got = _run(m, XE, W_edge)
    ref = orc.message(m.node_feats, m.edge_index, m.edge_vec, R @ W_edge.astype(float).T, m.W_node, m.W_out, lmax,
                      lmax_out, m.parity_mask)
    assert np.abs(ref).max() > 1e-3
    assert np.abs(got - ref).max() < 1e-12 * np.abs(ref).max()


@pytest.mark.parametrize("lmax,lmax_out", [(2, 3), (3, 2)])
def test_field_vs_fine_grid_quadrature(lmax, lmax_out):
    m, XE, W_edge = _case(lmax, lmax_out, nodes=4, degree=np.array([2, 0, 3, 1]), seed=3)
    got = _run(m, XE, W_edge)
    a = np.einsum("cn,enl->ecl", W_edge.astype(float), XE.astype(float))
    H = np.einsum("cn,jnl->jcl", m.W_node.astype(float), m.node_feats.astype(float))[m.edge_index[0]]
    T = np.zeros((m.nodes, m.C, (lmax_out + 1) ** 2))
    for c in range(m.C):
        Te = shref.grid_pipeline_onsite(a[:, c], H[:, c], lmax, lmax_out, odd=bool(m.parity_mask[c]))
        np.add.at(T[:, c], m.edge_index[1], Te)
    ref = np.zeros_like(got)
    for s in range(2):
        sel = m.parity_mask == s
        ref[:, s] = np.einsum("nc,ico->ino", m.W_out.astype(float)[:, sel], T[:, sel])
    assert np.abs(ref[:, 0]).max() > 1e-3 and np.abs(ref[:, 1]).max() > 1e-3
    assert np.abs(got - ref).max() < 1e-6 * np.abs(ref).max()   # finite-difference gradients in shref (odd sector)
    assert np.abs(got[:, 0] - ref[:, 0]).max() < 1e-12 * np.abs(ref).max()
    assert np.abs(got[1]).max() == 0.0                           # receiver without in-edges


def test_field_one_edge_per_receiver_is_onsite_and_edge_order():
    lmax, lmax_out = 3, 3
    m, XE, W_edge = _case(lmax, lmax_out, N=3, Ne=3, nodes=6, degree=1, seed=5)
    got = _run(m, XE, W_edge)
    ref = orc.onsite(XE, m.node_feats[m.edge_index[0]], W_edge, m.W_node, m.W_out, lmax, lmax_out, m.parity_mask)
    assert np.abs(got - ref).max() < 1e-13 * np.abs(ref).max()
    # swapping the factors changes the sign of the odd sector only (R10: the edge field is factor 1)
    swp = orc.onsite(m.node_feats[m.edge_index[0]], XE, m.W_node, W_edge, m.W_out, lmax, lmax_out, m.parity_mask)
    assert np.abs(got[:, 0] - swp[:, 0]).max() < 1e-13 * np.abs(ref).max()
    assert np.abs(got[:, 1] + swp[:, 1]).max() < 1e-13 * np.abs(ref).max()
    # permuting the edges inside every segment leaves the sums unchanged
    m, XE, W_edge = _case(lmax, lmax_out, nodes=5, degree=4, seed=6)
    base = _run(m, XE, W_edge)
    perm = np.arange(m.E).reshape(5, 4)[:, ::-1].reshape(-1)
    m2 = synthetic.make_message(lmax, lmax_out, 3, 4, 5, 4, seed=6)
    m2.edge_index = m.edge_index[:, perm]
    got = _run(m2, XE[perm], W_edge)
    assert np.abs(got - base).max() < 1e-13 * np.abs(base).max()


def test_field_equivariance_and_inversion():
    lmax, lmax_out = 2, 3
    m, XE, W_edge = _case(lmax, lmax_out, seed=8)
    base = _run(m, XE, W_edge)
    R = shref.random_rotation(np.random.default_rng(2))
    D = shref.wigner_D_real(lmax_out, R)
    L2 = (lmax + 1) ** 2
    rot = lambda x: np.einsum("ab,...b->...a", D[:L2, :L2], x.astype(float))
    got = _run(m, rot(XE), W_edge, node_feats=rot(m.node_feats))
    want = np.einsum("ab,...b->...a", D, base)
    assert np.abs(got - want).max() < 1e-12 * np.abs(base).max()
    # inversion of natural-parity inputs: even sector (-1)^l, odd sector -(-1)^l (pseudo-tensor, :111)
    sgn_in = np.array([(-1.0) ** l for l in range(lmax + 1) for _ in range(2 * l + 1)])
    sgn_out = np.array([(-1.0) ** l for l in range(lmax_out + 1) for _ in range(2 * l + 1)])
    got = _run(m, XE * sgn_in, W_edge, node_feats=m.node_feats * sgn_in)
    assert np.abs(got[:, 0] - base[:, 0] * sgn_out).max() < 1e-13 * np.abs(base).max()
    assert np.abs(got[:, 1] + base[:, 1] * sgn_out).max() < 1e-13 * np.abs(base).max()


# ------------------------------------------------------------------ l-dependent weights on the two-field coupling
def _lof(lmax):
    return np.concatenate([np.full(2 * l + 1, l) for l in range(lmax + 1)])


def test_field_lw_reduces_and_selects_degrees():
    lmax, lo = 3, 4
    m, XE, W_edge = _case(lmax, lo, N=3, Ne=2, C=4, nodes=5, degree=3, seed=21)
    base = _run(m, XE, W_edge)
    rep = lambda W, n: np.repeat(W[None].astype(np.float64), n, axis=0)
    run_lw = lambda We, Wn, Wo, xe=XE, x=m.node_feats: orc.message_field_lw(x, m.edge_index, xe, We, Wn, Wo, lmax, lo, m.parity_mask)
    assert np.array_equal(run_lw(rep(W_edge, lmax + 1), rep(m.W_node, lmax + 1), rep(m.W_out, lo + 1)), base)
    lv, lvo = _lof(lmax), _lof(lo)
    for l0 in range(lmax + 1):
        We = np.zeros((lmax + 1,) + W_edge.shape)
        We[l0] = W_edge
        got = run_lw(We, rep(m.W_node, lmax + 1), rep(m.W_out, lo + 1))
        ref = _run(m, XE * (lv == l0), W_edge)
        assert np.abs(got - ref).max() < 1e-13 and np.abs(ref).max() > 1e-3
        Wn = np.zeros((lmax + 1,) + m.W_node.shape)
        Wn[l0] = m.W_node
        got = run_lw(rep(W_edge, lmax + 1), Wn, rep(m.W_out, lo + 1))
        ref = _run(m, XE, W_edge, node_feats=m.node_feats * (lv == l0))
        assert np.abs(got - ref).max() < 1e-13 and np.abs(ref).max() > 1e-3
    for l0 in range(lo + 1):
        Wo = np.zeros((lo + 1,) + m.W_out.shape)
        Wo[l0] = m.W_out
        got = run_lw(rep(W_edge, lmax + 1), rep(m.W_node, lmax + 1), Wo)
        assert np.abs(got - base * (lvo == l0)).max() < 1e-13


def test_field_lw_vs_numpy_projections_around_the_shared_oracle():
    lmax, N, Ne, C = 3, 3, 2, 4
    m, XE, _ = _case(lmax, lmax, N=N, Ne=Ne, C=C, nodes=6, degree=np.array([2, 0, 3, 1, 4, 2]), seed=23)
    (Wn,), Wo = synthetic.lw_weights(lmax, lmax, N, C, seed=23, n_in=1)
    (We,), _ = synthetic.lw_weights(lmax, lmax, Ne, C, seed=29, n_in=1)
    got = orc.message_field_lw(m.node_feats, m.edge_index, XE, We, Wn, Wo, lmax, lmax, m.parity_mask)
    lv = _lof(lmax)
    a = np.einsum("qcn,enq->ecq", We[lv].astype(float), XE.astype(float))
    H = np.einsum("qcn,jnq->jcq", Wn[lv].astype(float), m.node_feats.astype(float))
    eye = np.eye(C)
    T = orc.message_field(H, m.edge_index, a, eye, eye, eye, lmax, lmax, m.parity_mask)  # [i, s, c, lm]
    ref = np.einsum("qnc,iscq->isnq", Wo[lv].astype(float), T)
    assert np.abs(got - ref).max() < 1e-12 and np.abs(ref).max() > 1e-2
    R = shref.random_rotation(np.random.default_rng(6))
    D = shref.wigner_D_real(lmax, R)
    rot = lambda x: np.einsum("ab,...b->...a", D, x.astype(float))
    got_r = orc.message_field_lw(rot(m.node_feats), m.edge_index, rot(XE), We, Wn, Wo, lmax, lmax, m.parity_mask)
    assert np.abs(got_r - rot(got)).max() < 1e-11

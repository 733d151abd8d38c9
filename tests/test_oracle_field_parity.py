"""Pins of oracle_message_field_parity (two parity-bearing fields, Eq.(28) PAPER.md:236 with the parity labels of both
fields, Sec. VI E :232-:240, Sec. VII C f :471) against things other than itself: the natural-parity two-field oracle per
run, the parity-labelled on-site oracle on one-edge receivers, exact vanishing in the wrong sector (the dispatch check
B7, :647, carried over to two fields), inversion with the slots' parity labels (Table I :86-:93) and Wigner-D rotation."""
import numpy as np
import pytest

from oracle import cgtp_oracle as orc
from paper_2605_15073_b200 import synthetic
from tests import shref


def _case(lmax=2, lmax_out=2, N=3, Ne=2, C=2, nodes=9, seed=0):
    rng = np.random.default_rng(seed)
    deg = rng.integers(0, 5, nodes)
    deg[0] = 0
    deg[-1] = 4
    return synthetic.make_field_parity(lmax, lmax_out, N, Ne, C, nodes, deg, seed=seed)


def _run(q, **kw):
    d = dict(node_feats=q.node_feats, edge_feats=q.edge_feats, W_edge=q.W_edge, W_node=q.W_node, W_out=q.W_out)
    d.update(kw)
    return orc.message_field_parity(d["node_feats"], q.edge_index, d["edge_feats"], d["W_edge"], d["W_node"], d["W_out"],
                                    q.lmax, q.lmax_out)


def _degrees(lmax):
    return np.concatenate([np.full(2 * l + 1, l) for l in range(lmax + 1)])


@pytest.mark.parametrize("s1,s2", [(0, 0), (0, 1), (1, 0), (1, 1)])
def test_one_slot_pair_reduces_to_the_natural_parity_two_field_oracle(s1, s2):
    """Only slot s1 of the edge field and slot s2 of the node field populated: the runs (cat, s1, s2, tau) are the only
    ones that see data; each is oracle_message_field (which knows no slots) with that run's weights, restricted to the
    output degrees (-1)^l = sigma, landing in sector s1^s2 (alpha) / 1^s1^s2 (beta) because p = p1 p2 (:236)."""
    q = _case(lmax=3, lmax_out=3, seed=3)
    X = np.zeros_like(q.node_feats)
    XE = np.zeros_like(q.edge_feats)
    X[:, s2] = q.node_feats[:, s2]
    XE[:, s1] = q.edge_feats[:, s1]
    got = _run(q, node_feats=X, edge_feats=XE)
    lv = _degrees(q.lmax_out)
    want = np.zeros_like(got)
    for cat in (0, 1):
        for tau in (0, 1):
            r = 8 * cat + 4 * s1 + 2 * s2 + tau
            mask = np.full(q.C, cat, np.uint8)
            nat = orc.message_field(X[:, s2], q.edge_index, XE[:, s1], q.W_edge[r], q.W_node[r], q.W_out[r], q.lmax,
                                    q.lmax_out, mask)
            sector = (s1 ^ s2) if cat == 0 else (1 ^ s1 ^ s2)
            sel = (lv % 2) == tau
            want[:, sector][:, :, sel] += nat[:, cat][:, :, sel]
    assert np.abs(got - want).max() <= 1e-12 * max(np.abs(want).max(), 1.0)
    assert np.abs(want).max() > 0.1


def test_one_edge_receivers_equal_the_parity_labelled_onsite_oracle():
    """A receiver with a single in-edge: the pooled coupling is the on-site contraction (Eq.(1) is "the on-site
    specialization" of Eq.(28), :238) with A = edge field, B = sender's node field (N = Ne so the shapes agree)."""
    lmax, N, C, nodes = 2, 3, 2, 6
    q = synthetic.make_field_parity(lmax, lmax, N, N, C, nodes, np.ones(nodes, np.int64), seed=5)
    got = _run(q)
    snd = q.edge_index[0]
    ref = orc.onsite_parity(q.edge_feats, q.node_feats[snd], q.W_edge, q.W_node, q.W_out, lmax, lmax)
    recv = q.edge_index[1]
    assert np.array_equal(recv, np.arange(nodes))
    assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()


def test_wrong_sector_vanishes_exactly():
    """B7 (:647) for two fields: with the edge field restricted to l1 = 0, natural slot (p1 = +1) and the node field on its
    natural slot only (p2 = (-1)^l2), every term has p = (-1)^l2 = (-1)^l (l = l2 for l1 = 0; the curl coupling needs
    l1 >= 1 and vanishes), so the opposite-parity sector is exactly zero; moving the node field to slot 1 moves the whole
    result to sector 1."""
    q = _case(lmax=2, lmax_out=2, seed=7)
    XE = np.zeros_like(q.edge_feats)
    XE[:, 0, :, 0] = q.edge_feats[:, 0, :, 0]  # l1 = 0 only, natural slot
    X = np.zeros_like(q.node_feats)
    X[:, 0] = q.node_feats[:, 0]
    out = _run(q, node_feats=X, edge_feats=XE)
    assert np.abs(out[:, 1]).max() == 0.0 and np.abs(out[:, 0]).max() > 0.0
    X2 = np.zeros_like(q.node_feats)
    X2[:, 1] = q.node_feats[:, 0]
    out2 = _run(q, node_feats=X2, edge_feats=XE)
    assert np.abs(out2[:, 0]).max() == 0.0 and np.abs(out2[:, 1]).max() > 0.0
    # edge field on l1 = 1, natural slot (p1 = -1), node natural: alpha terms (l1+l2+l even) carry p = -(-1)^l2 = (-1)^l,
    # beta terms (l1+l2+l odd) carry p = -(-1)^l2 = -(-1)^l: both sectors are fed, each from one category only
    XE1 = np.zeros_like(q.edge_feats)
    XE1[:, 0, :, 1:4] = q.edge_feats[:, 0, :, 1:4]
    Wo_alpha = q.W_out.copy(); Wo_alpha[8:] = 0
    Wo_beta = q.W_out.copy(); Wo_beta[:8] = 0
    oa = _run(q, node_feats=X, edge_feats=XE1, W_out=Wo_alpha)
    ob = _run(q, node_feats=X, edge_feats=XE1, W_out=Wo_beta)
    assert np.abs(oa[:, 1]).max() == 0.0 and np.abs(oa[:, 0]).max() > 0.0
    assert np.abs(ob[:, 0]).max() == 0.0 and np.abs(ob[:, 1]).max() > 0.0


def test_inversion_with_slot_labels():
    """Under inversion slot s at degree l picks (-1)^(s+l) on both fields (Table I :86-:93); the output slots pick the same
    labels: out[:, 0] -> (-1)^l out[:, 0], out[:, 1] -> -(-1)^l out[:, 1]."""
    q = _case(lmax=3, lmax_out=3, seed=11)
    base = _run(q)
    sg = (-1.0) ** _degrees(q.lmax)
    X = q.node_feats.astype(np.float64).copy()
    XE = q.edge_feats.astype(np.float64).copy()
    X[:, 0] *= sg; X[:, 1] *= -sg
    XE[:, 0] *= sg; XE[:, 1] *= -sg
    inv = _run(q, node_feats=X, edge_feats=XE)
    so = (-1.0) ** _degrees(q.lmax_out)
    assert np.abs(inv[:, 0] - base[:, 0] * so).max() <= 1e-12 * np.abs(base[:, 0]).max()
    assert np.abs(inv[:, 1] + base[:, 1] * so).max() <= 1e-12 * np.abs(base[:, 1]).max()


def test_rotation_equivariance():
    """Both slots of both fields rotate with D^l (a pseudo-tensor's coefficients "still rotate under D^l2", :228); both
    output slots rotate with D^l (App. B test 5, :633)."""
    q = _case(lmax=2, lmax_out=3, N=2, Ne=2, C=2, nodes=7, seed=13)
    base = _run(q)
    R = shref.random_rotation(np.random.default_rng(5))
    D = shref.wigner_D_real(max(q.lmax, q.lmax_out), R)
    Di = D[: (q.lmax + 1) ** 2, : (q.lmax + 1) ** 2]
    Do = D[: (q.lmax_out + 1) ** 2, : (q.lmax_out + 1) ** 2]
    X = np.einsum("ab,...b->...a", Di, q.node_feats.astype(np.float64))
    XE = np.einsum("ab,...b->...a", Di, q.edge_feats.astype(np.float64))
    rot = _run(q, node_feats=X, edge_feats=XE)
    want = np.einsum("ab,...b->...a", Do, base)
    assert np.abs(rot - want).max() <= 1e-11 * np.abs(want).max()


def test_edge_order_and_empty_receivers():
    q = _case(lmax=2, lmax_out=2, seed=17)
    base = _run(q)
    assert np.abs(base[q.degree == 0]).max() == 0.0
    # reversing the in-edges of every receiver changes nothing beyond rounding (the sum over j in Eq.(28))
    rp = np.searchsorted(q.edge_index[1], np.arange(q.nodes + 1))
    perm = np.concatenate([np.arange(rp[i], rp[i + 1])[::-1] for i in range(q.nodes)]).astype(np.int64)
    out = orc.message_field_parity(q.node_feats, q.edge_index[:, perm], q.edge_feats[perm], q.W_edge, q.W_node, q.W_out,
                                   q.lmax, q.lmax_out)
    assert np.abs(out - base).max() <= 1e-12 * np.abs(base).max()

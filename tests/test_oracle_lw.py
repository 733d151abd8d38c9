"""Pins of the l-dependent-weight oracle functions (oracle_onsite_lw / oracle_message_lw), CPU only.

Pinned to the l-shared functions (themselves pinned in test_oracle_pipeline.py): equal weights for every degree reduce to
them exactly; a weight stack that is non-zero at one degree selects that degree of the input (Eq.(35) PAPER.md:322:
c_{cnl} acts on A_{nlm} of the same l) / of the output (Eq.(41) :346: lambda_c^{(nl)} acts on T_{clm} of the same l);
the projections done per degree in numpy around the l-shared oracle with identity weights; Wigner-D equivariance.
"""
import numpy as np

from oracle import cgtp_oracle as orc
from paper_2605_15073_b200 import synthetic
from tests import shref


def _lof(lmax):
    return np.concatenate([np.full(2 * l + 1, l) for l in range(lmax + 1)])


def test_onsite_lw_reduces_and_selects_degrees():
    lmax, lo, N, C = 3, 4, 3, 4
    inp = synthetic.make_onsite(lmax, lo, N, C, batch=4, seed=41, parity_mask=[0, 1, 1, 0])
    base = orc.onsite(inp.A, inp.B, inp.W_a, inp.W_b, inp.W_out, lmax, lo, inp.parity_mask)
    rep = lambda W, n: np.repeat(W[None].astype(np.float64), n, axis=0)
    got = orc.onsite_lw(inp.A, inp.B, rep(inp.W_a, lmax + 1), rep(inp.W_b, lmax + 1), rep(inp.W_out, lo + 1), lmax, lo,
                        inp.parity_mask)
    assert np.array_equal(got, base)
    lv, lvo = _lof(lmax), _lof(lo)
    for l0 in range(lmax + 1):
        Wa = np.zeros((lmax + 1, C, N))
        Wa[l0] = inp.W_a
        got = orc.onsite_lw(inp.A, inp.B, Wa, rep(inp.W_b, lmax + 1), rep(inp.W_out, lo + 1), lmax, lo, inp.parity_mask)
        ref = orc.onsite(inp.A * (lv == l0), inp.B, inp.W_a, inp.W_b, inp.W_out, lmax, lo, inp.parity_mask)
        assert np.abs(got - ref).max() < 1e-13 and np.abs(ref).max() > 1e-3
    for l0 in range(lo + 1):
        Wo = np.zeros((lo + 1, N, C))
        Wo[l0] = inp.W_out
        got = orc.onsite_lw(inp.A, inp.B, rep(inp.W_a, lmax + 1), rep(inp.W_b, lmax + 1), Wo, lmax, lo, inp.parity_mask)
        assert np.abs(got - base * (lvo == l0)).max() < 1e-13


def test_onsite_lw_vs_numpy_projections_around_the_shared_oracle():
    lmax, N, C = 3, 3, 4
    inp = synthetic.make_onsite(lmax, lmax, N, C, batch=3, seed=43)
    (Wa, Wb), Wo = synthetic.lw_weights(lmax, lmax, N, C, seed=43)
    got = orc.onsite_lw(inp.A, inp.B, Wa, Wb, Wo, lmax, lmax, inp.parity_mask)
    lv = _lof(lmax)
    Ha = np.einsum("qcn,bnq->bcq", Wa[lv].astype(float), inp.A.astype(float))
    Hb = np.einsum("qcn,bnq->bcq", Wb[lv].astype(float), inp.B.astype(float))
    eye = np.eye(C)
    T = orc.onsite(Ha, Hb, eye, eye, eye, lmax, lmax, inp.parity_mask)  # [b, s, c, lm]: sector s holds its channels
    ref = np.einsum("qnc,bscq->bsnq", Wo[lv].astype(float), T)
    assert np.abs(got - ref).max() < 1e-12 and np.abs(ref).max() > 1e-2
    # rotation: weights act within a degree, so the result still rotates with D^l
    R = shref.random_rotation(np.random.default_rng(2))
    D = shref.wigner_D_real(lmax, R)
    rot = orc.onsite_lw(np.einsum("ab,...b->...a", D, inp.A.astype(float)), np.einsum("ab,...b->...a", D, inp.B.astype(float)),
                        Wa, Wb, Wo, lmax, lmax, inp.parity_mask)
    assert np.abs(rot - np.einsum("ab,...b->...a", D, got)).max() < 1e-11


def test_message_lw_reduces_and_matches_numpy_projections():
    lmax, N, C = 3, 3, 4
    m = synthetic.make_message(lmax, lmax, N, C, nodes=6, degree=np.array([2, 0, 3, 1, 2, 4]), seed=45,
                               parity_mask=[1, 0, 0, 1])
    base = orc.message(m.node_feats, m.edge_index, m.edge_vec, m.edge_radial, m.W_node, m.W_out, lmax, lmax, m.parity_mask)
    rep = lambda W: np.repeat(W[None].astype(np.float64), lmax + 1, axis=0)
    got = orc.message_lw(m.node_feats, m.edge_index, m.edge_vec, m.edge_radial, rep(m.W_node), rep(m.W_out), lmax, lmax,
                         m.parity_mask)
    assert np.abs(got - base).max() < 1e-13
    (Wn,), Wo = synthetic.lw_weights(lmax, lmax, N, C, seed=45, n_in=1)
    got = orc.message_lw(m.node_feats, m.edge_index, m.edge_vec, m.edge_radial, Wn, Wo, lmax, lmax, m.parity_mask)
    lv = _lof(lmax)
    H = np.einsum("qcn,jnq->jcq", Wn[lv].astype(float), m.node_feats.astype(float))
    eye = np.eye(C)
    T = orc.message(H, m.edge_index, m.edge_vec, m.edge_radial, eye, eye, lmax, lmax, m.parity_mask)
    ref = np.einsum("qnc,iscq->isnq", Wo[lv].astype(float), T)
    assert np.abs(got - ref).max() < 1e-12 and np.abs(ref).max() > 1e-2


def test_message_lwr_radial_per_degree():
    """l1-dependent radial factor (Eq.(46)): equal values for every l1 reduce to message_lw; the general
    case against a direct contraction of the pinned real coupling tables (real_coupling_dense) in numpy."""
    lmax, N, C = 3, 3, 4
    m = synthetic.make_message(lmax, lmax, N, C, nodes=5, degree=np.array([2, 0, 3, 1, 2]), seed=47,
                               parity_mask=[1, 0, 0, 1])
    (Wn,), Wo = synthetic.lw_weights(lmax, lmax, N, C, seed=47, n_in=1)
    rep = np.repeat(m.edge_radial[:, :, None].astype(float), lmax + 1, axis=2)
    a = orc.message_lwr(m.node_feats, m.edge_index, m.edge_vec, rep, Wn, Wo, lmax, lmax, m.parity_mask)
    b = orc.message_lw(m.node_feats, m.edge_index, m.edge_vec, m.edge_radial, Wn, Wo, lmax, lmax, m.parity_mask)
    assert np.abs(a - b).max() < 1e-13
    rad = np.random.default_rng(3).standard_normal((m.E, C, lmax + 1))
    got = orc.message_lwr(m.node_feats, m.edge_index, m.edge_vec, rad, Wn, Wo, lmax, lmax, m.parity_mask)
    lv = _lof(lmax)
    H = np.einsum("qcn,jnq->jcq", Wn[lv].astype(float), m.node_feats.astype(float))
    tabs = [orc.real_coupling_dense(lmax, lmax, False), orc.real_coupling_dense(lmax, lmax, True)]
    T = np.zeros((m.nodes, C, (lmax + 1) ** 2))
    for e in range(m.E):
        j, i = m.edge_index[:, e]
        Y = shref.real_sh_xyz(lmax, m.edge_vec[e].astype(float))
        for c in range(C):
            T[i, c] += np.einsum("abo,a,b->o", tabs[int(m.parity_mask[c])], rad[e, c][lv] * Y, H[j, c])
    ref = np.zeros_like(got)
    for s in (0, 1):
        sel = m.parity_mask == s
        ref[:, s] = np.einsum("qnc,icq->inq", Wo[lv].astype(float)[:, :, sel], T[:, sel])
    assert np.abs(got - ref).max() < 1e-12 and np.abs(ref).max() > 1e-2

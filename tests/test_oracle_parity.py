"""Pins of the parity-slot oracle functions (oracle_message_parity / oracle_onsite_parity), CPU only.

Pinned to: the paper's dispatch check (App. B test 7: "With l1 = 0 and I on p2 = +1, every
p_out = +1 output sector receives a non-zero contribution while p_out = -1 vanishes exactly.  Switching to
l1 = 1 flips this."), the slot rules Eq.(44) (:385), Eq.(45) (:390), Eq.(56) (:432) read off the support of
the result, the reduction to the natural-parity functions (Cases A-D of Sec. VI, :197-:232; those functions
are pinned in test_oracle_pipeline.py), inversion with the parity labels of the slots, SO(3) equivariance.
"""
import numpy as np
import pytest

from oracle import cgtp_oracle as orc
from paper_2605_15073_b200 import synthetic
from tests import shref


def _lsign(lmax):
    return np.concatenate([np.full(2 * l + 1, (-1.0) ** l) for l in range(lmax + 1)])


def _lof(lmax):
    return np.concatenate([np.full(2 * l + 1, l) for l in range(lmax + 1)])


def _abs_parity(slot, l):
    """Parity label of slot `slot` at degree l: slot 0 natural (-1)^l, slot 1 opposite."""
    return (-1) ** (slot + l)


def _mp(m, X=None, ev=None, er=None, Wn=None, Wo=None, rl=None, lw=None):
    return orc.message_parity(m.node_feats if X is None else X, m.edge_index, m.edge_vec if ev is None else ev,
                              m.edge_radial if er is None else er, m.W_node if Wn is None else Wn,
                              m.W_out if Wo is None else Wo, m.lmax, m.lmax_out, rl, lw)


@pytest.mark.parametrize("l1", [0, 1])
def test_message_dispatch_rule_b7(l1):
    """One bond, lmax = 2, edge restricted to a single degree l1, I populated on p2 = +1 only (:647)."""
    lmax = 2
    m = synthetic.make_message_parity(lmax, lmax, N=1, C=1, nodes=2, degree=np.array([1, 0]), seed=5)
    lv = _lof(lmax)
    X = np.zeros_like(m.node_feats, dtype=np.float64)
    for s in (0, 1):  # p2 = +1 entries only
        for q, l in enumerate(lv):
            if _abs_parity(s, l) == +1:
                X[:, s, :, q] = m.node_feats[:, s, :, q]
    lw = np.zeros(lmax + 1)
    lw[l1] = 1.0
    out = _mp(m, X=X, lw=lw)[0]  # [2, N, Lo2]
    p_expected = (-1) ** l1  # p = (-1)^{l1} p2
    hit = False
    for s in (0, 1):
        for q, l in enumerate(lv):
            if _abs_parity(s, l) == p_expected:
                hit = hit or np.abs(out[s, :, q]).max() > 1e-3
            else:
                assert np.all(out[s, :, q] == 0.0), (s, l)
    assert hit
    # every output degree of the surviving parity is reached (l1 = 0: l = l2; l1 = 1: l = l2 +- 1 alpha, l = l2 beta)
    for l in range(lmax + 1):
        s = 0 if _abs_parity(0, l) == p_expected else 1
        assert np.abs(out[s][:, lv == l]).max() > 1e-4, l


@pytest.mark.parametrize("cat", [0, 1])
def test_message_slot_rule_eq44_eq56(cat):
    """Populate one (slot, l2) block of I and keep one category's output weights: the outputs that light up obey
    p2 = p (-1)^{l+l2} for alpha (Eq.(44)) and the opposite slot for beta (Eq.(56))."""
    lmax = 3
    m = synthetic.make_message_parity(lmax, lmax, N=2, C=3, nodes=4, degree=2, seed=9)
    lv = _lof(lmax)
    Wo = m.W_out.astype(np.float64).copy()
    Wo[4 * (1 - cat):4 * (1 - cat) + 4] = 0.0  # silence the other category
    for s_in in (0, 1):
        for l2 in range(lmax + 1):
            X = np.zeros_like(m.node_feats, dtype=np.float64)
            X[:, s_in][:, :, lv == l2] = m.node_feats[:, s_in][:, :, lv == l2]
            out = _mp(m, X=X, Wo=Wo)
            p2 = _abs_parity(s_in, l2)
            seen = 0
            for s in (0, 1):
                for l in range(lmax + 1):
                    blk = np.abs(out[:, s][:, :, lv == l]).max()
                    p = _abs_parity(s, l)
                    rule = p * (-1) ** (l + l2) * (1 if cat == 0 else -1)
                    if rule == p2 and (cat == 0 or (l > 0 and l2 > 0)):  # Q needs l1, l2, l >= 1 (:585)
                        assert blk > 1e-6, (s_in, l2, s, l)
                        seen += 1
                    elif rule != p2:
                        assert blk == 0.0, (s_in, l2, s, l)
            assert seen >= lmax or (cat == 1 and l2 == 0)


def test_message_reduces_to_natural_parity_cases_abcd():
    """Slot 1 empty -> Cases A (alpha -> sector 0) and B (beta -> sector 1); slot 0 empty -> Cases C (alpha ->
    sector 1) and D (beta -> sector 0); each run's weights act on its own output-l parity (Eq.(54), (55))."""
    lmax, N, C = 3, 3, 4
    m = synthetic.make_message_parity(lmax, lmax, N, C, nodes=6, degree=np.array([2, 0, 3, 1, 2, 4]), seed=3)
    lv = _lof(lmax)
    for s_in in (0, 1):
        X = np.zeros_like(m.node_feats, dtype=np.float64)
        X[:, s_in] = m.node_feats[:, s_in]
        got = _mp(m, X=X)
        for cat in (0, 1):
            s_out = s_in ^ cat
            for tau in (0, 1):
                run = 4 * cat + 2 * s_out + tau
                ref = orc.message(m.node_feats[:, s_in], m.edge_index, m.edge_vec, m.edge_radial[:, run],
                                  m.W_node[run], m.W_out[run], lmax, lmax, np.full(C, cat, np.uint8))
                sel = (lv % 2) == tau
                # the other category writes the other sector, so sector s_out at these l holds this run alone
                assert np.abs(got[:, s_out][:, :, sel] - ref[:, cat][:, :, sel]).max() < 1e-12
                assert np.abs(ref[:, cat][:, :, sel]).max() > 1e-3 or (cat == 1 and lmax == 0)


def test_message_parity_inversion_rotation_subset():
    lmax, N, C, nodes = 3, 3, 2, 6
    m = synthetic.make_message_parity(lmax, lmax, N, C, nodes, degree=3, seed=14)
    base = _mp(m)
    sign = _lsign(lmax)
    # inversion: a slot with parity label p2 picks up p2; the edge vector flips; sector s at degree l picks
    # its label (-1)^{s+l}  (Table I :86-:93)
    Xi = m.node_feats.astype(np.float64).copy()
    Xi[:, 0] *= sign
    Xi[:, 1] *= -sign
    inv = _mp(m, X=Xi, ev=-m.edge_vec.astype(np.float64))
    assert np.abs(inv[:, 0] - base[:, 0] * sign).max() < 1e-12
    assert np.abs(inv[:, 1] + base[:, 1] * sign).max() < 1e-12
    assert np.abs(base[:, 0]).max() > 1e-2 and np.abs(base[:, 1]).max() > 1e-2
    # rotation: both slots and both sectors rotate with D^l (pseudo-tensors rotate like tensors, :228)
    R = shref.random_rotation(np.random.default_rng(5))
    D = shref.wigner_D_real(lmax, R)
    rot = _mp(m, X=np.einsum("ab,...b->...a", D, m.node_feats.astype(np.float64)), ev=m.edge_vec.astype(np.float64) @ R.T)
    assert np.abs(rot - np.einsum("ab,...b->...a", D, base)).max() < 1e-11
    sub = _mp(m, rl=[4, 1])
    assert np.array_equal(sub, base[[4, 1]])


def test_onsite_parity_reduces_to_natural_parity_runs():
    """Only slots (s1, s2) populated: run (cat, s1, s2, tau) is the natural-parity contraction with that run's
    weights, restricted to (-1)^l = sigma and written to the sector whose label is p1 p2 (Eq.(1) :29)."""
    lmax, N, C = 3, 3, 2
    q = synthetic.make_onsite_parity(lmax, lmax, N, C, batch=3, seed=17)
    lv = _lof(lmax)
    full = np.zeros((3, 2, N, (lmax + 1) ** 2))
    for s1 in (0, 1):
        for s2 in (0, 1):
            A = np.zeros_like(q.A, dtype=np.float64)
            B = np.zeros_like(q.B, dtype=np.float64)
            A[:, s1] = q.A[:, s1]
            B[:, s2] = q.B[:, s2]
            got = orc.onsite_parity(A, B, q.W_a, q.W_b, q.W_out, lmax, lmax)
            full += got
            for cat in (0, 1):
                s_out = s1 ^ s2 ^ cat
                for tau in (0, 1):
                    run = 8 * cat + 4 * s1 + 2 * s2 + tau
                    ref = orc.onsite(q.A[:, s1], q.B[:, s2], q.W_a[run], q.W_b[run], q.W_out[run], lmax, lmax,
                                     np.full(C, cat, np.uint8))
                    sel = (lv % 2) == tau
                    assert np.abs(got[:, s_out][:, :, sel] - ref[:, cat][:, :, sel]).max() < 1e-12
    # bilinear: the four slot pairs add up to the full result
    assert np.abs(full - orc.onsite_parity(q.A, q.B, q.W_a, q.W_b, q.W_out, lmax, lmax)).max() < 1e-11


def test_onsite_parity_inversion_rotation():
    lmax, N, C = 2, 2, 3
    q = synthetic.make_onsite_parity(lmax, 2 * lmax - 1, N, C, batch=2, seed=19)
    lo = 2 * lmax - 1
    base = orc.onsite_parity(q.A, q.B, q.W_a, q.W_b, q.W_out, lmax, lo)
    sign, sign_o = _lsign(lmax), _lsign(lo)
    Ai, Bi = q.A.astype(np.float64).copy(), q.B.astype(np.float64).copy()
    for Z in (Ai, Bi):
        Z[:, 0] *= sign
        Z[:, 1] *= -sign
    inv = orc.onsite_parity(Ai, Bi, q.W_a, q.W_b, q.W_out, lmax, lo)
    assert np.abs(inv[:, 0] - base[:, 0] * sign_o).max() < 1e-12
    assert np.abs(inv[:, 1] + base[:, 1] * sign_o).max() < 1e-12
    R = shref.random_rotation(np.random.default_rng(6))
    D, Do = shref.wigner_D_real(lmax, R), shref.wigner_D_real(lo, R)
    rot = orc.onsite_parity(np.einsum("ab,...b->...a", D, q.A.astype(np.float64)),
                            np.einsum("ab,...b->...a", D, q.B.astype(np.float64)), q.W_a, q.W_b, q.W_out, lmax, lo)
    assert np.abs(rot - np.einsum("ab,...b->...a", Do, base)).max() < 1e-11

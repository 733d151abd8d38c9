"""Parity of cgtp_message_field (two feature fields, Eq.(28) :236, Sec. VII C f :471)
against the FP64 oracle, through the C ABI.  Bar: max|out - ref| / max|ref| <= 1e-5 per sector (FP32); segmentation
bit-exact (an edge attributed to the wrong receiver fails the value check at O(1))."""
import numpy as np
import pytest
import torch

from oracle import cgtp_oracle as orc
from paper_2605_15073_b200 import binding as cg
from paper_2605_15073_b200 import synthetic
from tests import shref
from tests.parity_util import TOL, cuda as _cuda, sample_rows, sector_errs

pytestmark = pytest.mark.gpu


def run_field(m, XE, W_edge, **kw):
    out = cg.cgtp_message_field(_cuda(m.node_feats), _cuda(m.edge_index), _cuda(XE), _cuda(W_edge), _cuda(m.W_node),
                                _cuda(m.W_out), m.lmax, m.lmax_out, m.N, W_edge.shape[1], m.C, m.parity_mask, **kw)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def oracle_field(m, XE, W_edge):
    return orc.message_field(m.node_feats, m.edge_index, XE, W_edge, m.W_node, m.W_out, m.lmax, m.lmax_out, m.parity_mask)


def sector_err(got, ref):
    """max over the sectors of the R14 / R22 error norm (tests/parity_util.py)."""
    return max(sector_errs(got, ref))


def _ragged(nodes, hi, seed):
    d = np.random.default_rng(seed).integers(0, hi + 1, size=nodes)
    d[0] = 0
    d[-1] = 0
    return d


# several CTAs and a ragged tail of columns; compiled and non-compiled bands (5 -> 6, 7 -> 8); lmax_out != lmax;
# band 12 takes the generic core; ragged degrees with empty receivers (first and last node included)
@pytest.mark.parametrize("lmax,lmax_out,N,Ne,C,nodes,degree", [
    (2, 2, 8, 4, 8, 40, 3), (4, 4, 16, 8, 12, 61, "ragged"), (6, 6, 16, 16, 16, 50, 5), (8, 8, 8, 8, 8, 20, 4),
    (3, 5, 6, 3, 5, 33, "ragged"), (5, 3, 4, 4, 6, 17, 2), (7, 7, 8, 2, 4, 9, 3), (1, 2, 2, 2, 2, 5, 1),
    (12, 12, 4, 4, 4, 6, 2), (4, 0, 8, 8, 8, 12, 3),
    # channel counts per parity that are multiples of the core's column-group width (32, or 16 from band 8 up and for
    # the odd channels at 6): the sender's field is read in place through the edge list, no gathered copy
    (4, 4, 16, 8, 64, 37, "ragged"), (8, 8, 8, 4, 32, 11, 3), (6, 6, 8, 8, 64, 13, 4), (2, 3, 8, 8, 64, 29, "ragged"),
])
def test_field_vs_oracle(lmax, lmax_out, N, Ne, C, nodes, degree):
    deg = _ragged(nodes, 6, lmax) if degree == "ragged" else degree
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, deg, seed=100 * lmax + lmax_out)
    XE, W_edge = synthetic.make_edge_field(m, Ne, seed=lmax)
    got = run_field(m, XE, W_edge, check=True)
    ref = oracle_field(m, XE, W_edge)
    assert got.shape == ref.shape
    assert sector_err(got, ref) <= TOL, sector_err(got, ref)
    assert np.array_equal(got, run_field(m, XE, W_edge))  # bitwise reproducible


@pytest.mark.parametrize("mask_kind", ["even", "odd", "mixed"])
def test_field_masks(mask_kind):
    lmax, lmax_out, N, Ne, C, nodes = 3, 3, 8, 4, 7, 25
    mask = {"even": np.zeros(C, np.uint8), "odd": np.ones(C, np.uint8),
            "mixed": np.array([1, 0, 0, 1, 1, 0, 1], np.uint8)}[mask_kind]
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, 4, seed=2, parity_mask=mask)
    XE, W_edge = synthetic.make_edge_field(m, Ne, seed=2)
    got = run_field(m, XE, W_edge)
    ref = oracle_field(m, XE, W_edge)
    assert sector_err(got, ref) <= TOL


def test_field_edge_chunks_straddle_segments():
    # C = 1024 -> chunks of 4096 edges; degree 7 puts segment boundaries inside chunks and segments across them
    lmax, lmax_out, N, Ne, C, nodes = 1, 1, 2, 2, 1024, 1300
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, 7, seed=4)
    assert m.E > 2 * 4096 and 4096 % 7 != 0
    XE, W_edge = synthetic.make_edge_field(m, Ne, seed=4)
    got = run_field(m, XE, W_edge, check=True)
    ref = oracle_field(m, XE, W_edge)
    assert sector_err(got, ref) <= TOL


def test_field_no_edges_and_bad_graph():
    lmax, lmax_out, N, Ne, C, nodes = 2, 2, 4, 4, 4, 6
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, 0, seed=1)
    XE, W_edge = synthetic.make_edge_field(m, Ne, seed=1)
    assert m.E == 0
    got = run_field(m, XE, W_edge, check=True)
    assert got.shape == (nodes, 2, N, 9) and np.abs(got).max() == 0.0
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, 2, seed=1)
    XE, W_edge = synthetic.make_edge_field(m, Ne, seed=1)
    m.edge_index = m.edge_index[:, ::-1].copy()  # receivers descending
    with pytest.raises(cg.CgtpError):
        run_field(m, XE, W_edge, check=True)
    m = synthetic.make_message(lmax, lmax_out, N, 64, nodes, 2, seed=1)   # in-place sender reads (C/2 = 32)
    XE, W_edge = synthetic.make_edge_field(m, Ne, seed=1)
    m.edge_index[0, 3] = nodes + 5                                        # sender out of range
    with pytest.raises(cg.CgtpError):
        run_field(m, XE, W_edge, check=True)
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, 2, seed=1)
    XE, W_edge = synthetic.make_edge_field(m, Ne, seed=1)
    with pytest.raises(cg.CgtpError):  # workspace too small
        m2 = synthetic.make_message(lmax, lmax_out, N, C, nodes, 2, seed=1)
        run_field(m2, XE, W_edge, workspace=torch.empty(512, dtype=torch.uint8, device="cuda"))


def test_field_RY_edge_fields_match_cgtp_message():
    lmax, lmax_out, N, Ne, C, nodes = 4, 4, 16, 8, 16, 64
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, 5, seed=7)
    _, W_edge = synthetic.make_edge_field(m, Ne, seed=7)
    R = np.random.default_rng(3).standard_normal((m.E, Ne)).astype(np.float32)
    ev = m.edge_vec.astype(np.float64)
    Y = shref.real_sh_xyz(lmax, ev / np.linalg.norm(ev, axis=1, keepdims=True))
    XE = (R[:, :, None] * Y[:, None, :]).astype(np.float32)
    got = run_field(m, XE, W_edge)
    er = (R.astype(np.float64) @ W_edge.astype(np.float64).T).astype(np.float32)
    ref = cg.cgtp_message(_cuda(m.node_feats), _cuda(m.edge_index), _cuda(m.edge_vec), _cuda(er), _cuda(m.W_node),
                          _cuda(m.W_out), lmax, lmax_out, N, C, m.parity_mask)
    torch.cuda.synchronize()
    assert sector_err(got, ref.cpu().numpy().astype(np.float64)) <= 2 * TOL


def test_field_rotation_equivariance_on_device():
    lmax, lmax_out, N, Ne, C, nodes = 4, 4, 8, 8, 8, 30
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, 4, seed=9)
    XE, W_edge = synthetic.make_edge_field(m, Ne, seed=9)
    base = run_field(m, XE, W_edge).astype(np.float64)
    D = shref.wigner_D_real(lmax_out, shref.random_rotation(np.random.default_rng(4)))
    L2 = (lmax + 1) ** 2
    rot = lambda x: np.einsum("ab,...b->...a", D[:L2, :L2], x.astype(np.float64)).astype(np.float32)
    m.node_feats = rot(m.node_feats)
    got = run_field(m, rot(XE), W_edge).astype(np.float64)
    want = np.einsum("ab,...b->...a", D, base)
    assert sector_err(got, want) <= TOL


def test_field_full_size_bench_configuration_sampled_receivers():
    """The workload bench.py times (`edge_field`: graph of BASELINE.json configs[2], N = C = Ne = 128, lmax 4, half odd
    channels, in-place sender reads): sampled receivers (first, last, strided, seeded-random) against the oracle, which
    evaluates the same edge list restricted to those receivers; exchange-free invariant on the full output: the odd
    sector has no l = 0 component."""
    lmax, N, Ne, C, nodes, degree = 4, 128, 128, 128, 2048, 16
    m = synthetic.make_message(lmax, lmax, N, C, nodes, degree, seed=0)
    XE, W_edge = synthetic.make_edge_field(m, Ne, seed=0)
    got = run_field(m, XE, W_edge, check=True)
    recv = sample_rows(nodes, 128, seed=0)
    keep = np.isin(m.edge_index[1], recv)
    ref = orc.message_field(m.node_feats, m.edge_index[:, keep], XE[keep], W_edge, m.W_node, m.W_out, lmax, lmax,
                            m.parity_mask)
    assert sector_err(got[recv], ref[recv]) <= TOL, sector_err(got[recv], ref[recv])
    assert np.abs(got[:, 1, :, 0]).max() <= TOL * np.abs(got[:, 1]).max()


def test_field_bipartite_shards_reproduce_the_full_call():
    from paper_2605_15073_b200 import parallel
    lmax, lmax_out, N, Ne, C, nodes = 4, 4, 8, 8, 64, 50
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, _ragged(nodes, 7, 3), seed=12)
    XE, W_edge = synthetic.make_edge_field(m, Ne, seed=12)
    full = run_field(m, XE, W_edge)
    rp = parallel.row_ptr_from_receivers(m.edge_index[1], nodes)
    bounds = parallel.shard_receivers(rp, 3)
    rows = []
    for r in range(3):
        sh = parallel.make_field_shard(torch.from_numpy(m.node_feats), torch.from_numpy(m.edge_index), torch.from_numpy(XE),
                                       bounds, r)
        out = cg.cgtp_message_field_bipartite(_cuda(m.node_feats), sh.edge_index.cuda(), sh.edge_feats.cuda(), _cuda(W_edge),
                                              _cuda(m.W_node), _cuda(m.W_out), lmax, lmax_out, N, Ne, C, m.parity_mask,
                                              sh.hi - sh.lo, check=True)
        torch.cuda.synchronize()
        rows.append(out.cpu().numpy())
    assert np.array_equal(np.concatenate(rows), full)  # bit-identical rows


@pytest.mark.parametrize("lmax,lmax_out,N,Ne,C,nodes", [(4, 4, 16, 8, 64, 30), (3, 5, 6, 4, 5, 21), (6, 6, 8, 8, 16, 12)])
def test_field_lw_vs_oracle(lmax, lmax_out, N, Ne, C, nodes):
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, _ragged(nodes, 5, lmax), seed=31 + lmax)
    XE, _ = synthetic.make_edge_field(m, Ne, seed=31)
    (Wn,), Wo = synthetic.lw_weights(lmax, lmax_out, N, C, seed=31, n_in=1)
    (We,), _ = synthetic.lw_weights(lmax, lmax_out, Ne, C, seed=37, n_in=1)
    out = cg.cgtp_message_field_lw(_cuda(m.node_feats), _cuda(m.edge_index), _cuda(XE), _cuda(We), _cuda(Wn), _cuda(Wo),
                                   lmax, lmax_out, N, Ne, C, m.parity_mask, check=True)
    torch.cuda.synchronize()
    ref = orc.message_field_lw(m.node_feats, m.edge_index, XE, We, Wn, Wo, lmax, lmax_out, m.parity_mask)
    assert sector_err(out.cpu().numpy(), ref) <= TOL


def test_field_configs4_graph_sampled_receivers():
    """The graph of BASELINE.json configs[4] (16384 nodes, 524288 edges, lmax 8, N = C = 128, half odd) with an edge
    field of 8 channels: 16 edge chunks, 16-column groups reading the sender's field in place; >= 128 sampled receivers
    against the oracle on the edge list restricted to them."""
    lmax, N, Ne, C, nodes, degree = 8, 128, 8, 128, 16384, 32
    m = synthetic.make_message(lmax, lmax, N, C, nodes, degree, r_max=6.0, seed=0)
    XE, W_edge = synthetic.make_edge_field(m, Ne, seed=0)
    got = run_field(m, XE, W_edge, check=True)
    # >= 128 receivers, both sides of every chunk boundary (chunks of 2^22 / C = 32768 edges = 1024 receivers)
    bounds = [b + d for b in range(1024, nodes, 1024) for d in (-1, 0)]
    recv = sample_rows(nodes, 128, seed=1, extra=bounds)
    assert recv.size >= 128
    keep = np.isin(m.edge_index[1], recv)
    ref = orc.message_field(m.node_feats, m.edge_index[:, keep], XE[keep], W_edge, m.W_node, m.W_out, lmax, lmax,
                            m.parity_mask)
    assert sector_err(got[recv], ref[recv]) <= TOL, sector_err(got[recv], ref[recv])
    assert np.abs(got[:, 1, :, 0]).max() <= TOL * np.abs(got[:, 1]).max()


# ------------------------------------------------ two parity-bearing fields with slot axes
def run_field_parity(q, **kw):
    out = cg.cgtp_message_field_parity(_cuda(q.node_feats), _cuda(q.edge_index), _cuda(q.edge_feats), _cuda(q.W_edge),
                                       _cuda(q.W_node), _cuda(q.W_out), q.lmax, q.lmax_out, q.N, q.Ne, q.C, **kw)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("lmax,lmax_out,N,Ne,C,nodes", [
    (0, 0, 2, 2, 2, 5),
    (1, 2, 3, 2, 2, 17),     # odd N * L2: slot blocks not 16-byte aligned -> generic projection kernel
    (2, 2, 8, 4, 8, 40),
    (3, 5, 4, 3, 3, 21),     # lmax_out > lmax
    (4, 4, 8, 8, 8, 30),     # 16 columns per parity block: sender fields read in place through the edge list
    (6, 6, 8, 4, 4, 25),
    (8, 8, 4, 4, 4, 12),
])
def test_field_parity_slots_vs_oracle(lmax, lmax_out, N, Ne, C, nodes):
    """cgtp_message_field_parity (Eq.(28) with the parity labels of both fields, Sec. VII C f :471) against the
    term-by-term oracle: 16 runs, ragged graphs with empty first receiver and a long last segment."""
    rng = np.random.default_rng(600 + lmax)
    deg = rng.integers(0, 7, nodes)
    deg[0] = 0
    deg[-1] = 19
    q = synthetic.make_field_parity(lmax, lmax_out, N, Ne, C, nodes, deg, seed=600 + lmax)
    got = run_field_parity(q, check=True)
    ref = orc.message_field_parity(q.node_feats, q.edge_index, q.edge_feats, q.W_edge, q.W_node, q.W_out, lmax, lmax_out)
    assert sector_err(got, ref) <= TOL, sector_errs(got, ref)
    assert np.abs(got[deg == 0]).max() == 0.0
    assert np.array_equal(got, run_field_parity(q))  # bitwise reproducible


def test_field_parity_reduces_to_the_natural_parity_call():
    """Slot 1 of both fields empty: sector 0 / 1 at (-1)^l = sigma equal cgtp_message_field with the weights of the runs
    (alpha, 0, 0, tau) / (beta, 0, 0, tau) -- the two entry points agree to rounding."""
    lmax, N, Ne, C, nodes = 4, 8, 4, 4, 30
    q = synthetic.make_field_parity(lmax, lmax, N, Ne, C, nodes, _ragged(nodes, 6, 2), seed=77)
    q.node_feats[:, 1] = 0
    q.edge_feats[:, 1] = 0
    got = run_field_parity(q)
    lv = np.concatenate([np.full(2 * l + 1, l) for l in range(lmax + 1)])
    for tau in (0, 1):
        We = np.concatenate([q.W_edge[tau], q.W_edge[8 + tau]])
        Wn = np.concatenate([q.W_node[tau], q.W_node[8 + tau]])
        Wo = np.concatenate([q.W_out[tau], q.W_out[8 + tau]], axis=1)
        nat = cg.cgtp_message_field(_cuda(q.node_feats[:, 0]), _cuda(q.edge_index), _cuda(q.edge_feats[:, 0]), _cuda(We),
                                    _cuda(Wn), _cuda(Wo), lmax, lmax, N, Ne, 2 * C, [0] * C + [1] * C).cpu().numpy()
        sel = (lv % 2) == tau
        for s in (0, 1):
            d = np.abs(got[:, s][:, :, sel] - nat[:, s][:, :, sel]).max()
            assert d <= 2e-6 * np.abs(nat[:, s]).max(), (tau, s, d)


def test_field_parity_inversion_rotation_and_errors_on_gpu():
    lmax, N, Ne, C, nodes = 4, 4, 4, 4, 20
    q = synthetic.make_field_parity(lmax, lmax, N, Ne, C, nodes, 5, seed=91)
    base = run_field_parity(q).astype(np.float64)
    sign = np.concatenate([np.full(2 * l + 1, (-1.0) ** l) for l in range(lmax + 1)]).astype(np.float32)
    qi = synthetic.make_field_parity(lmax, lmax, N, Ne, C, nodes, 5, seed=91)
    qi.node_feats[:, 0] *= sign
    qi.node_feats[:, 1] *= -sign
    qi.edge_feats[:, 0] *= sign
    qi.edge_feats[:, 1] *= -sign
    inv = run_field_parity(qi)
    assert np.abs(inv[:, 0] - base[:, 0] * sign).max() < TOL * np.abs(base[:, 0]).max()
    assert np.abs(inv[:, 1] + base[:, 1] * sign).max() < TOL * np.abs(base[:, 1]).max()
    D = shref.wigner_D_real(lmax, shref.random_rotation(np.random.default_rng(8)))
    qr = synthetic.make_field_parity(lmax, lmax, N, Ne, C, nodes, 5, seed=91)
    qr.node_feats = np.einsum("ab,...b->...a", D, q.node_feats.astype(np.float64)).astype(np.float32)
    qr.edge_feats = np.einsum("ab,...b->...a", D, q.edge_feats.astype(np.float64)).astype(np.float32)
    rot = run_field_parity(qr)
    assert sector_err(rot, np.einsum("ab,...b->...a", D, base)) <= TOL
    bad = synthetic.make_field_parity(lmax, lmax, N, Ne, C, nodes, 5, seed=91)
    bad.edge_index[1] = bad.edge_index[1][::-1].copy()
    with pytest.raises(cg.CgtpError) as ei:
        run_field_parity(bad, check=True)
    assert ei.value.code == cg.ERR_GRAPH
    assert np.abs(run_field_parity(bad)).max() == 0.0  # zeros plus the flag


# ------------------------------------------------------------ neighbour sum on the grid inside the core vs per-edge passes
@pytest.fixture
def default_path_after():
    yield
    cg.cgtp_set_kernel_path(0)


@pytest.mark.parametrize("lmax,lmax_out,N,Ne,C,nodes,degree", [
    (2, 2, 8, 4, 32, 40, "ragged"), (4, 4, 16, 8, 64, 61, "ragged"), (6, 6, 16, 16, 32, 50, 5), (8, 8, 8, 8, 32, 20, 40),
    (3, 5, 6, 3, 32, 33, "ragged"),
])
def test_field_per_edge_path_vs_oracle(lmax, lmax_out, N, Ne, C, nodes, degree, default_path_after):
    """The per-edge form (one full core pass per edge + pooling kernel, CGTP_PATH_FIELD_PER_EDGE) stays covered: against the
    oracle, and against the default form (neighbour sum on the grid inside the core) to rounding."""
    deg = _ragged(nodes, 9, lmax) if degree == "ragged" else degree
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, deg, seed=70 + lmax)
    XE, W_edge = synthetic.make_edge_field(m, Ne, seed=70)
    ref = oracle_field(m, XE, W_edge)
    got = run_field(m, XE, W_edge, check=True)
    assert sector_err(got, ref) <= TOL
    cg.cgtp_set_kernel_path(cg.PATH_FIELD_PER_EDGE)
    n0 = cg.cgtp_launch_count()
    alt = run_field(m, XE, W_edge, check=True)
    n1 = cg.cgtp_launch_count()
    assert sector_err(alt, ref) <= TOL
    cg.cgtp_set_kernel_path(0)
    run_field(m, XE, W_edge)
    assert cg.cgtp_launch_count() - n1 <= n1 - n0  # the default form has no pooling launches where its group width divides the channels


def test_field_configs4_graph_every_element_both_forms(default_path_after):
    """The configs[4] graph (16 edge chunks, segments meeting chunk boundaries): the two forms agree on every element."""
    lmax, N, Ne, C, nodes, degree = 8, 128, 8, 128, 16384, 32
    m = synthetic.make_message(lmax, lmax, N, C, nodes, degree, r_max=6.0, seed=0)
    XE, W_edge = synthetic.make_edge_field(m, Ne, seed=0)
    T = [_cuda(x) for x in (m.node_feats, m.edge_index, XE, W_edge, m.W_node, m.W_out)]
    f = lambda: cg.cgtp_message_field(*T, lmax, lmax, N, Ne, C, m.parity_mask, check=True)
    a = f().clone()
    cg.cgtp_set_kernel_path(cg.PATH_FIELD_PER_EDGE)
    b = f()
    for s in (0, 1):
        assert ((a[:, s] - b[:, s]).abs().max() / b[:, s].abs().max()).item() < TOL

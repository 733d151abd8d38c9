"""Parity of the CUDA path (through the C ABI, via paper_2605_15073_b200.binding) against the FP64 oracle.

Bar (BASELINE.json north_star; R14): per parity sector, max|out - ref| / max|ref| <= 1e-5 for
FP32; indexing / segmentation bit-exact.  All inputs are seeded and synthetic (synthetic.py).
"""
import numpy as np
import pytest
import torch

from oracle import cgtp_oracle as orc
from paper_2605_15073_b200 import binding as cg
from paper_2605_15073_b200 import synthetic
from tests import shref
from tests.parity_util import TOL, cuda as _cuda, sector_errs as sector_err

pytestmark = pytest.mark.gpu


def run_onsite(inp, **kw):
    out = cg.cgtp_onsite(_cuda(inp.A), _cuda(inp.B), _cuda(inp.W_a), _cuda(inp.W_b), _cuda(inp.W_out),
                         inp.lmax, inp.lmax_out, inp.N, inp.C, inp.parity_mask, **kw)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def run_message(m, **kw):
    out = cg.cgtp_message(_cuda(m.node_feats), _cuda(m.edge_index), _cuda(m.edge_vec), _cuda(m.edge_radial),
                          _cuda(m.W_node), _cuda(m.W_out), m.lmax, m.lmax_out, m.N, m.C, m.parity_mask, **kw)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def oracle_onsite(inp, idx=None):
    A, B = (inp.A, inp.B) if idx is None else (inp.A[idx], inp.B[idx])
    return orc.onsite(A, B, inp.W_a, inp.W_b, inp.W_out, inp.lmax, inp.lmax_out, inp.parity_mask)


def oracle_message(m, recv=None):
    return orc.message(m.node_feats, m.edge_index, m.edge_vec, m.edge_radial, m.W_node, m.W_out, m.lmax, m.lmax_out,
                       m.parity_mask, recv)


# ------------------------------------------------------------------------------------------ on-site
def test_onsite_config0_full():
    """BASELINE.json configs[0]: lmax=2, N=8, C=8, batch=64, even+odd, seed 0."""
    inp = synthetic.config(0)
    got, ref = run_onsite(inp), oracle_onsite(inp)
    e = sector_err(got, ref)
    assert max(e) < TOL, e
    assert np.abs(ref[:, 1, :, 0]).max() == 0.0 and np.abs(got[:, 1, :, 0]).max() < 1e-6  # odd sector: no l=0


@pytest.mark.parametrize("lmax,lmax_out,N,C,batch,mask", [
    (0, 0, 4, 4, 3, [0, 1, 0, 1]),
    (1, 1, 5, 6, 37, [0, 1, 1, 0, 1, 0]),
    (1, 2, 4, 4, 9, [1, 0, 0, 1]),
    (2, 4, 3, 5, 11, [1, 1, 0, 1, 0]),
    (3, 3, 7, 9, 130, [0, 0, 1, 0, 1, 1, 1, 0, 0]),
    (3, 5, 4, 4, 20, [0, 1, 0, 1]),
    (4, 2, 6, 8, 33, [1, 0, 1, 0, 1, 0, 1, 0]),
    (5, 5, 8, 8, 65, [0, 0, 0, 0, 1, 1, 1, 1]),
    (7, 7, 4, 6, 19, [0, 1, 0, 1, 0, 1]),      # band 7 runs on the LB=8 instantiation
    (9, 9, 4, 4, 7, [0, 0, 1, 1]),             # band 9 -> LB=10
    (4, 4, 8, 8, 40, [0] * 8),                 # all even: sector 1 must be zero
    (4, 4, 8, 8, 40, [1] * 8),                 # all odd: sector 0 must be zero
    (6, 6, 40, 33, 50, None),                  # N, C not multiples of the GEMM tiles
    (16, 16, 40, 40, 3, None),                 # 289 coefficients > one 256-column tile of proj_fast (sub-tiles)
    (2, 2, 72, 136, 61, None),                 # several row blocks, ragged last atom group and row slab
    (5, 5, 12, 20, 9, [0] * 10 + [1] * 10),    # K = 12 / 10: small K chunks
    (3, 3, 8, 8, 300, [0, 0, 0, 1, 1, 1, 1, 1]),  # odd number of even channels: generic projection kernel
])
def test_onsite_small_shapes(lmax, lmax_out, N, C, batch, mask):
    inp = synthetic.make_onsite(lmax, lmax_out, N, C, batch, seed=100 + lmax * 7 + lmax_out, parity_mask=mask)
    got, ref = run_onsite(inp), oracle_onsite(inp)
    e = sector_err(got, ref)
    assert max(e) < TOL, e
    for s in (0, 1):
        if np.abs(ref[:, s]).max() == 0.0:
            assert np.abs(got[:, s]).max() == 0.0


@pytest.fixture
def default_path_after():
    yield
    cg.cgtp_set_kernel_path(0)


@pytest.mark.parametrize("lmax,lmax_out,N,C,batch,mask", [
    (2, 2, 8, 8, 64, None),                        # configs[0]: 8 atoms per tile, two buffers, all groups per barrier
    (2, 2, 8, 8, 61, None),                        # ragged last tile
    (1, 1, 4, 8, 19, [0] * 4 + [1] * 4),           # odd lmax: aligned coefficient rows (L2 = 4)
    (3, 2, 8, 16, 33, [0] * 8 + [1] * 8),          # lmax_out < lmax, L2 = 16
    (4, 4, 32, 32, 300, None),                     # configs[3] shape at lmax 4
    (4, 4, 16, 32, 77, [0] * 24 + [1] * 8),        # unbalanced sectors: 24 pointwise + 8 curl channels
    (5, 5, 8, 16, 21, [1] * 16),                   # all odd: every warp on the curl sub-group; sector 0 must be zero
    (6, 6, 8, 16, 21, [0] * 16),                   # all even
    (6, 6, 64, 64, 301, None),                     # configs[1] shape: tight layout (one A/B buffer under the F planes)
    (6, 4, 32, 64, 150, None),                     # N != C, lmax_out < lmax
    (7, 7, 8, 32, 40, None),                       # band 7 on the LB = 8 instantiation, aligned rows (L2 = 64)
    (8, 8, 8, 16, 30, [0] * 16),                   # band 8 fits with one parity only (the F planes of both do not)
])
def test_onsite_fused_kernel_shapes(lmax, lmax_out, N, C, batch, mask, default_path_after):
    """The single-kernel step (onsite_fused.cu) forced for every shape it supports (CGTP_PATH_FUSED_ONSITE), against the
    oracle; then the four-launch step on the same inputs (the two must agree to rounding)."""
    inp = synthetic.make_onsite(lmax, lmax_out, N, C, batch, seed=900 + 10 * lmax + lmax_out, parity_mask=mask)
    ref = oracle_onsite(inp)
    cg.cgtp_set_kernel_path(cg.PATH_FUSED_ONSITE)
    n0 = cg.cgtp_launch_count()
    got = run_onsite(inp)
    assert cg.cgtp_launch_count() - n0 == 1  # one launch: the fused kernel took the shape
    e = sector_err(got, ref)
    assert max(e) < TOL, e
    for s in (0, 1):
        if np.abs(ref[:, s]).max() == 0.0:
            assert np.abs(got[:, s]).max() == 0.0
    assert np.array_equal(got, run_onsite(inp))  # bitwise reproducible
    cg.cgtp_set_kernel_path(cg.PATH_UNFUSED_ONSITE)
    n0 = cg.cgtp_launch_count()
    alt = run_onsite(inp)
    assert cg.cgtp_launch_count() - n0 >= 3
    e = sector_err(alt, ref)
    assert max(e) < TOL, e


@pytest.mark.parametrize("lmax,lmax_out,N,C,batch,mask", [
    (1, 1, 8, 8, 70, None),
    (2, 2, 8, 16, 129, None),
    (3, 3, 8, 8, 300, [0, 0, 0, 1, 1, 1, 1, 1]),   # 3 even + 5 odd channels: ragged column groups in both parities
    (4, 4, 32, 32, 300, None),                     # configs[3] shape at lmax 4
    (4, 2, 8, 8, 33, None),                        # lmax_out < lmax: T shorter than H
    (2, 4, 8, 8, 33, None),                        # lmax_out > lmax: band limit 4 kernel, H has 9 coefficients
    (5, 5, 8, 16, 65, None),                       # H re-read from shared memory per grid row (band limits 5, 6)
    (3, 6, 8, 8, 21, None),                        # band limit 6: register core for the odd channels only
    (6, 6, 16, 16, 47, [1] * 16),                  # all odd at band limit 6
    (4, 4, 8, 8, 1, None),                         # one atom: a single partly filled group
])
def test_onsite_register_and_shared_memory_cores(lmax, lmax_out, N, C, batch, mask, default_path_after):
    """S2a-S4b at small band limits have two cores: one thread per column with everything in registers (onsite_reg.cu, the
    library's choice for band limits <= 5 and the odd channels at 6) and the warp-scheduled shared-memory core
    (onsite_core.cu, CGTP_PATH_SMEM_CORE).  Both against the oracle on the four-launch step."""
    inp = synthetic.make_onsite(lmax, lmax_out, N, C, batch, seed=700 + 10 * lmax + lmax_out, parity_mask=mask)
    ref = oracle_onsite(inp)
    outs = []
    for flags in (cg.PATH_UNFUSED_ONSITE, cg.PATH_UNFUSED_ONSITE | cg.PATH_SMEM_CORE):
        cg.cgtp_set_kernel_path(flags)
        got = run_onsite(inp)
        e = sector_err(got, ref)
        assert max(e) < TOL, (flags, e)
        assert np.array_equal(got, run_onsite(inp))  # bitwise reproducible
        outs.append(got)
    assert not np.array_equal(outs[0], outs[1])  # two different kernels did run (different summation orders)


def test_onsite_config1_full():
    """BASELINE.json configs[1] (the bench workload): lmax=6, N=C=64, batch=4096, every output checked."""
    inp = synthetic.config(1)
    got, ref = run_onsite(inp), oracle_onsite(inp)
    e = sector_err(got, ref)
    assert max(e) < TOL, e


@pytest.mark.parametrize("lmax,N,C,batch", [(6, 64, 64, 4099), (5, 32, 32, 9001)])
def test_onsite_window_tiles_ragged(lmax, N, C, batch):
    """Projection tiles that are windows of the flattened (atom, lm) columns (proj_fast.cu): atoms straddle tile
    boundaries and the last window is ragged; every output checked."""
    inp = synthetic.make_onsite(lmax, lmax, N, C, batch, seed=610 + lmax)
    got, ref = run_onsite(inp), oracle_onsite(inp)
    e = sector_err(got, ref)
    assert max(e) < TOL, e


def test_onsite_invariants_full_size():
    """Properties that hold at any size, on the bench workload: exchange symmetry, self-coupled vanishing
    (Eq.(27)) and bitwise run-to-run reproducibility."""
    inp = synthetic.config(1)
    A, B, Wa, Wb, Wo = map(_cuda, (inp.A, inp.B, inp.W_a, inp.W_b, inp.W_out))
    f = lambda a, b, wa, wb: cg.cgtp_onsite(a, b, wa, wb, Wo, inp.lmax, inp.lmax_out, inp.N, inp.C, inp.parity_mask)
    base = f(A, B, Wa, Wb).clone()
    again = f(A, B, Wa, Wb)
    assert torch.equal(base, again)
    sw = f(B, A, Wb, Wa)
    scale0, scale1 = base[:, 0].abs().max().item(), base[:, 1].abs().max().item()
    assert (sw[:, 0] - base[:, 0]).abs().max().item() < TOL * scale0
    assert (sw[:, 1] + base[:, 1]).abs().max().item() < TOL * scale1
    selfc = f(A, A, Wa, Wa)
    assert selfc[:, 1].abs().max().item() < TOL * scale1
    assert selfc[:, 0].abs().max().item() > 0.1 * scale0


def test_onsite_equivariance():
    """R15: rotate A, B with the real Wigner-D of a random rotation; outputs rotate with D, per sector."""
    lmax = 6
    inp = synthetic.make_onsite(lmax, lmax, 16, 16, 64, seed=5)
    base = run_onsite(inp).astype(np.float64)
    R = shref.random_rotation(np.random.default_rng(17))
    D = shref.wigner_D_real(lmax, R)
    rot_in = synthetic.make_onsite(lmax, lmax, 16, 16, 64, seed=5)
    rot_in.A = np.einsum("ab,...b->...a", D, inp.A.astype(np.float64)).astype(np.float32)
    rot_in.B = np.einsum("ab,...b->...a", D, inp.B.astype(np.float64)).astype(np.float32)
    rot = run_onsite(rot_in).astype(np.float64)
    e = sector_err(rot, np.einsum("ab,...b->...a", D, base))
    assert max(e) < TOL, e


def test_onsite_host_entry_matches_device_entry():
    inp = synthetic.make_onsite(4, 4, 16, 16, 3000, seed=9)
    dev = run_onsite(inp)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    host = cg.cgtp_onsite_host(pin(inp.A), pin(inp.B), pin(inp.W_a), pin(inp.W_b), pin(inp.W_out), 4, 4, 16, 16,
                               inp.parity_mask).numpy()
    # the host entry works in batch chunks, and the library chooses the kernels per call size (onsite_fused.cu for small
    # calls): the two results agree to rounding, not bit for bit
    for s in (0, 1):
        assert np.abs(dev[:, s] - host[:, s]).max() <= 2e-6 * np.abs(dev[:, s]).max()
    host2 = cg.cgtp_onsite_host(pin(inp.A), pin(inp.B), pin(inp.W_a), pin(inp.W_b), pin(inp.W_out), 4, 4, 16, 16,
                                inp.parity_mask).numpy()
    assert np.array_equal(host, host2)


def test_onsite_argument_errors():
    inp = synthetic.make_onsite(2, 2, 4, 4, 4, seed=1)
    A, B, Wa, Wb, Wo = map(_cuda, (inp.A, inp.B, inp.W_a, inp.W_b, inp.W_out))
    with pytest.raises(cg.CgtpError) as ei:
        cg.cgtp_onsite(A, B, Wa, Wb, Wo, 2, 2, 4, 4, [0, 1, 2, 0])
    assert ei.value.code == cg.ERR_INVALID
    big = synthetic.make_onsite(2, 2, 4, 4, 1, seed=1)
    with pytest.raises(cg.CgtpError) as ei:  # lmax_out > 2 lmax
        cg.cgtp_onsite(A, B, Wa, Wb, Wo, 2, 5, 4, 4, big.parity_mask,
                       out=torch.empty((4, 2, 4, 36), device="cuda"))
    assert ei.value.code == cg.ERR_INVALID
    with pytest.raises(cg.CgtpError) as ei:  # band limit above the compiled maximum
        L2 = (cg.cgtp_max_lmax() + 2) ** 2
        z = torch.zeros((1, 4, L2), device="cuda")
        cg.cgtp_onsite(z, z, Wa, Wb, Wo, cg.cgtp_max_lmax() + 1, cg.cgtp_max_lmax() + 1, 4, 4, big.parity_mask)
    assert ei.value.code == cg.ERR_UNSUPPORTED
    with pytest.raises(TypeError):  # CPU tensors are refused: no CPU fallback
        cg.cgtp_onsite(A.cpu(), B, Wa, Wb, Wo, 2, 2, 4, 4, inp.parity_mask)
    empty = torch.zeros((0, 4, 9), device="cuda")
    out = cg.cgtp_onsite(empty, empty, Wa, Wb, Wo, 2, 2, 4, 4, inp.parity_mask)
    assert out.shape == (0, 2, 4, 9)


# ------------------------------------------------------------------------------------- segmentation
def test_segments_bit_exact_and_graph_errors():
    rng = np.random.default_rng(0)
    nodes = 1000
    deg = rng.integers(0, 9, nodes)
    deg[[0, 17, 999]] = 0
    m = synthetic.make_message(2, 2, 4, 4, nodes, deg, seed=3)
    rc, ref = orc.segments(m.edge_index, nodes)
    assert rc == 0
    row_ptr, status = cg.cgtp_build_segments(_cuda(m.edge_index), nodes)
    assert status.item() == 0
    assert np.array_equal(row_ptr.cpu().numpy(), ref)
    # empty edge list
    row_ptr, status = cg.cgtp_build_segments(torch.zeros((2, 0), dtype=torch.int64, device="cuda"), 5)
    assert status.item() == 0 and np.array_equal(row_ptr.cpu().numpy(), np.zeros(6, np.int64))
    # unsorted receivers / out-of-range sender
    bad = m.edge_index.copy()
    bad[1, 10], bad[1, 400] = bad[1, 400], bad[1, 10]
    assert cg.cgtp_build_segments(_cuda(bad), nodes)[1].item() == cg.ERR_GRAPH
    assert orc.segments(bad, nodes)[0] == 4
    bad = m.edge_index.copy()
    bad[0, 5] = nodes
    assert cg.cgtp_build_segments(_cuda(bad), nodes)[1].item() == cg.ERR_GRAPH


# ----------------------------------------------------------------------------------- message passing
@pytest.mark.parametrize("lmax,lmax_out,N,C,nodes,mask", [
    (0, 0, 4, 4, 6, [0, 1, 0, 1]),
    (1, 1, 4, 4, 9, [0, 1, 1, 0]),
    (2, 2, 5, 6, 40, [0, 1, 1, 0, 1, 0]),
    (3, 3, 8, 8, 30, None),
    (2, 4, 4, 4, 12, [1, 0, 0, 1]),
    (4, 2, 4, 6, 12, [0, 0, 1, 1, 1, 0]),
    (5, 5, 8, 8, 25, [1] * 8),
    (6, 6, 8, 8, 25, [0] * 8),
    (7, 7, 4, 4, 10, None),
])
def test_message_small_ragged_graphs(lmax, lmax_out, N, C, nodes, mask):
    rng = np.random.default_rng(lmax * 13 + nodes)
    deg = rng.integers(0, 20, nodes)
    deg[0] = 0
    deg[nodes // 2] = 0
    deg[-1] = 0 if nodes % 2 else 11
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, deg, seed=200 + lmax, parity_mask=mask)
    got, ref = run_message(m, check=True), oracle_message(m)
    e = sector_err(got, ref)
    assert max(e) < TOL, e
    assert np.abs(got[deg == 0]).max() == 0.0  # receivers without edges -> zeros


@pytest.mark.parametrize("lmax,lmax_out,N,C,deg,mask", [
    # one receiver with more in-edges than the producer warp's batch (32) and the geometry chunk
    (3, 3, 8, 8, [70, 0, 33, 1, 32, 8], None),
    # more even channels than one CTA block of the edge kernel holds (several channel blocks)
    (6, 6, 4, 132, [5, 0, 9, 3], [0] * 130 + [1] * 2),
    # sub-blocks with a ragged last channel group
    (8, 8, 4, 14, [4, 7, 0, 2], [0] * 9 + [1] * 5),
    # the largest grid the library supports (lmax = lmax_out = 20: 473 float4 quads per field)
    (20, 20, 4, 2, [2, 0, 3], [0, 1]),
])
def test_message_edge_kernel_shapes(lmax, lmax_out, N, C, deg, mask):
    """Shapes that exercise the tiling limits of the TMA-ring edge kernel (edge_ring.cu)."""
    deg = np.asarray(deg)
    m = synthetic.make_message(lmax, lmax_out, N, C, len(deg), deg, seed=300 + lmax, parity_mask=mask)
    got, ref = run_message(m, check=True), oracle_message(m)
    e = sector_err(got, ref)
    assert max(e) < TOL, e
    assert np.abs(got[deg == 0]).max() == 0.0


def test_message_config2_full_even_and_halfhalf():
    """BASELINE.json configs[2]: 2048 nodes x 16 in-edges, lmax=4, N=C=128; all-even as the config states
    plus the half/half variant."""
    m = synthetic.config(2)
    got, ref = run_message(m, check=True), oracle_message(m)
    e = sector_err(got, ref)
    assert e[0] < TOL and np.abs(got[:, 1]).max() == 0.0, e
    m.parity_mask = synthetic.half_mask(m.C)
    got, ref = run_message(m, check=True), oracle_message(m)
    e = sector_err(got, ref)
    assert max(e) < TOL, e


def test_message_reproducible_and_graph_error():
    m = synthetic.make_message(4, 4, 16, 16, 300, 12, seed=8)
    a = run_message(m)
    b = run_message(m)
    assert np.array_equal(a, b)
    bad = synthetic.make_message(4, 4, 16, 16, 300, 12, seed=8)
    bad.edge_index[1] = bad.edge_index[1][::-1].copy()
    with pytest.raises(cg.CgtpError) as ei:
        run_message(bad, check=True)
    assert ei.value.code == cg.ERR_GRAPH
    out = run_message(bad)
    assert np.abs(out).max() == 0.0


def test_message_equivariance_and_inversion():
    lmax = 4
    m = synthetic.make_message(lmax, lmax, 8, 8, 50, 10, seed=31)
    base = run_message(m).astype(np.float64)
    R = shref.random_rotation(np.random.default_rng(23))
    D = shref.wigner_D_real(lmax, R)
    mr = synthetic.make_message(lmax, lmax, 8, 8, 50, 10, seed=31)
    mr.node_feats = np.einsum("ab,...b->...a", D, m.node_feats.astype(np.float64)).astype(np.float32)
    mr.edge_vec = (m.edge_vec.astype(np.float64) @ R.T).astype(np.float32)
    rot = run_message(mr).astype(np.float64)
    e = sector_err(rot, np.einsum("ab,...b->...a", D, base))
    assert max(e) < TOL, e
    sign = np.concatenate([np.full(2 * l + 1, (-1.0) ** l) for l in range(lmax + 1)]).astype(np.float32)
    mi = synthetic.make_message(lmax, lmax, 8, 8, 50, 10, seed=31)
    mi.node_feats = m.node_feats * sign
    mi.edge_vec = -m.edge_vec
    inv = run_message(mi).astype(np.float64)
    assert np.abs(inv[:, 0] - base[:, 0] * sign).max() < TOL * np.abs(base[:, 0]).max()
    assert np.abs(inv[:, 1] + base[:, 1] * sign).max() < TOL * np.abs(base[:, 1]).max()


def test_message_host_entry_matches_device_entry():
    m = synthetic.make_message(3, 3, 8, 8, 200, 7, seed=2)
    dev = run_message(m)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    host = cg.cgtp_message_host(pin(m.node_feats), pin(m.edge_index), pin(m.edge_vec), pin(m.edge_radial),
                                pin(m.W_node), pin(m.W_out), 3, 3, 8, 8, m.parity_mask).numpy()
    assert np.array_equal(dev, host)


def test_message_bipartite_shards_reproduce_the_full_call():
    """Receiver sharding on one GPU: each shard's cgtp_message_bipartite call over its own
    in-edges (global senders, local receivers) gives exactly the rows of the unsharded call, and matches the oracle."""
    from paper_2605_15073_b200 import parallel
    rng = np.random.default_rng(21)
    deg = rng.integers(0, 14, 61)
    deg[[0, 30]] = 0
    m = synthetic.make_message(3, 3, 8, 8, 61, deg, seed=91)
    full = run_message(m, check=True)
    ref = oracle_message(m)
    assert max(sector_err(full, ref)) < TOL
    rp = parallel.row_ptr_from_receivers(m.edge_index[1], m.nodes)
    bounds = parallel.shard_receivers(rp, 3)
    t = torch.from_numpy
    for r in range(3):
        s = parallel.make_shard(t(m.node_feats), t(m.edge_index), t(m.edge_vec), t(m.edge_radial), bounds, r)
        got = cg.cgtp_message_bipartite(_cuda(m.node_feats), s.edge_index.cuda(), s.edge_vec.cuda(), s.edge_radial.cuda(),
                                        _cuda(m.W_node), _cuda(m.W_out), m.lmax, m.lmax_out, m.N, m.C, m.parity_mask,
                                        s.hi - s.lo, check=True)
        torch.cuda.synchronize()
        assert np.array_equal(got.cpu().numpy(), full[s.lo:s.hi])
    # a sender index outside [0, n_send) is a graph error
    bad = m.edge_index.copy()
    bad[0, 0] = m.nodes
    with pytest.raises(cg.CgtpError) as ei:
        cg.cgtp_message_bipartite(_cuda(m.node_feats), _cuda(bad), _cuda(m.edge_vec), _cuda(m.edge_radial),
                                  _cuda(m.W_node), _cuda(m.W_out), m.lmax, m.lmax_out, m.N, m.C, m.parity_mask,
                                  m.nodes, check=True)
    assert ei.value.code == cg.ERR_GRAPH


# ------------------------------------------------------------------------- tensor-core math modes
@pytest.fixture
def fp32_mode_after():
    yield
    cg.cgtp_set_math_mode(cg.MATH_FP32)


@pytest.mark.parametrize("lmax,N,C,batch", [
    (2, 8, 8, 64),       # configs[0] shape: one partial tile
    (4, 24, 40, 70),     # K = 24 / 20: zero-padded K chunk; 40 channels padded to 64 TMEM columns
    (6, 64, 64, 300),    # configs[1] shape, several tiles per CTA ring
    (3, 136, 72, 40),    # K = 136: three K chunks accumulate in TMEM
])
def test_onsite_tensor_core_math_modes(lmax, N, C, batch, fp32_mode_after):
    """cgtp_set_math_mode: the 3xTF32 tcgen05 projections meet the FP32 parity bar, single-pass TF32 lands at the
    ~1e-3 the TF32 mantissa allows, and switching back restores the FP32 path bit for bit."""
    inp = synthetic.make_onsite(lmax, lmax, N, C, batch, seed=500 + lmax)
    ref = oracle_onsite(inp)
    base = run_onsite(inp)
    cg.cgtp_set_math_mode(cg.MATH_3XTF32)
    assert cg.cgtp_get_math_mode() == cg.MATH_3XTF32
    e3 = sector_err(run_onsite(inp), ref)
    assert max(e3) < TOL, e3
    cg.cgtp_set_math_mode(cg.MATH_TF32)
    e1 = sector_err(run_onsite(inp), ref)
    assert 1e-5 < max(e1) < 2e-2, e1
    cg.cgtp_set_math_mode(cg.MATH_FP32)
    assert np.array_equal(run_onsite(inp), base)
    with pytest.raises(cg.CgtpError):
        cg.cgtp_set_math_mode(7)


def test_message_tensor_core_math_mode(fp32_mode_after):
    m = synthetic.make_message(4, 4, 128, 128, 96, 6, seed=17)
    ref = oracle_message(m)
    cg.cgtp_set_math_mode(cg.MATH_3XTF32)
    e3 = sector_err(run_message(m, check=True), ref)
    assert max(e3) < TOL, e3


# ------------------------------------------------------------- parity-labelled inputs
def run_onsite_parity(q):
    out = cg.cgtp_onsite_parity(_cuda(q.A), _cuda(q.B), _cuda(q.W_a), _cuda(q.W_b), _cuda(q.W_out), q.lmax,
                                q.lmax_out, q.N, q.C)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def run_message_parity(m, **kw):
    out = cg.cgtp_message_parity(_cuda(m.node_feats), _cuda(m.edge_index), _cuda(m.edge_vec), _cuda(m.edge_radial),
                                 _cuda(m.W_node), _cuda(m.W_out), m.lmax, m.lmax_out, m.N, m.C, **kw)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("lmax,lmax_out,N,C,batch", [
    (0, 0, 2, 2, 5),
    (1, 2, 3, 2, 37),     # odd N * L2: slot blocks not 16-byte aligned -> generic projection kernel
    (2, 2, 8, 8, 64),     # configs[0] shape with both slots
    (3, 5, 4, 3, 33),
    (6, 6, 16, 8, 300),   # fast core + fast projections, several tiles and a ragged tail
    (10, 10, 4, 2, 9),
])
def test_onsite_parity_slots(lmax, lmax_out, N, C, batch):
    """cgtp_onsite_parity (PAPER.md VII C e :469) against the term-by-term oracle, 16 runs."""
    q = synthetic.make_onsite_parity(lmax, lmax_out, N, C, batch, seed=400 + lmax)
    got = run_onsite_parity(q)
    ref = orc.onsite_parity(q.A, q.B, q.W_a, q.W_b, q.W_out, lmax, lmax_out)
    e = sector_err(got, ref)
    assert max(e) < TOL, e
    assert np.array_equal(got, run_onsite_parity(q))  # bitwise reproducible


def test_onsite_parity_reduces_to_natural_call():
    """Slot 1 of both inputs empty: sector 0 / 1 at (-1)^l = sigma equal cgtp_onsite with the weights of the runs
    (alpha, 0, 0, tau) / (beta, 0, 0, tau) -- the two entry points agree to rounding."""
    lmax, N, C, batch = 4, 8, 4, 50
    q = synthetic.make_onsite_parity(lmax, lmax, N, C, batch, seed=77)
    q.A[:, 1] = 0
    q.B[:, 1] = 0
    got = run_onsite_parity(q)
    lv = np.concatenate([np.full(2 * l + 1, l) for l in range(lmax + 1)])
    for tau in (0, 1):
        Wa = np.concatenate([q.W_a[tau], q.W_a[8 + tau]])
        Wb = np.concatenate([q.W_b[tau], q.W_b[8 + tau]])
        Wo = np.concatenate([q.W_out[tau], q.W_out[8 + tau]], axis=1)
        nat = cg.cgtp_onsite(_cuda(q.A[:, 0]), _cuda(q.B[:, 0]), _cuda(Wa), _cuda(Wb), _cuda(Wo), lmax, lmax, N, 2 * C,
                             [0] * C + [1] * C).cpu().numpy()
        sel = (lv % 2) == tau
        for s in (0, 1):
            d = np.abs(got[:, s][:, :, sel] - nat[:, s][:, :, sel]).max()
            assert d <= 2e-6 * np.abs(nat[:, s]).max(), (tau, s, d)


@pytest.mark.parametrize("lmax,lmax_out,N,C,nodes", [
    (0, 0, 2, 2, 5),
    (2, 2, 3, 3, 17),
    (3, 4, 4, 2, 12),
    (4, 4, 8, 8, 40),
    (8, 8, 4, 5, 10),
])
def test_message_parity_slots(lmax, lmax_out, N, C, nodes):
    """cgtp_message_parity (PAPER.md VII C a-c) against the term-by-term oracle, 8 runs, ragged graphs."""
    rng = np.random.default_rng(500 + lmax)
    deg = rng.integers(0, 12, nodes)
    deg[0] = 0
    deg[-1] = 35
    m = synthetic.make_message_parity(lmax, lmax_out, N, C, nodes, deg, seed=500 + lmax)
    got = run_message_parity(m, check=True)
    ref = orc.message_parity(m.node_feats, m.edge_index, m.edge_vec, m.edge_radial, m.W_node, m.W_out, lmax, lmax_out)
    e = sector_err(got, ref)
    assert max(e) < TOL, e
    assert np.abs(got[deg == 0]).max() == 0.0
    assert np.array_equal(got, run_message_parity(m))


def test_message_parity_inversion_on_gpu():
    """Parity labels on the device path: slot s at degree l carries (-1)^(s+l) (Table I PAPER.md:86-:93)."""
    lmax, N, C, nodes = 5, 8, 4, 20
    m = synthetic.make_message_parity(lmax, lmax, N, C, nodes, 6, seed=91)
    base = run_message_parity(m)
    sign = np.concatenate([np.full(2 * l + 1, (-1.0) ** l) for l in range(lmax + 1)]).astype(np.float32)
    m.node_feats[:, 0] *= sign
    m.node_feats[:, 1] *= -sign
    m.edge_vec = -m.edge_vec
    inv = run_message_parity(m)
    assert np.abs(inv[:, 0] - base[:, 0] * sign).max() < 1e-5 * np.abs(base[:, 0]).max()
    assert np.abs(inv[:, 1] + base[:, 1] * sign).max() < 1e-5 * np.abs(base[:, 1]).max()


# --------------------------------------------------------------- l-dependent CP weights
@pytest.mark.parametrize("lmax,lmax_out,N,C,batch,mask", [
    (0, 0, 2, 2, 5, [0, 1]),
    (2, 2, 8, 8, 64, None),
    (3, 5, 5, 3, 33, [1, 0, 1]),      # odd N: unaligned atom blocks -> generic projection kernel
    (6, 6, 16, 16, 700, None),        # fast projections with a column offset, several tiles, ragged tail
    (10, 10, 4, 4, 9, None),
])
def test_onsite_lw(lmax, lmax_out, N, C, batch, mask):
    """cgtp_onsite_lw: c_{cnl} / lambda_c^{(nl)} per degree (Eq.(35), Eq.(41) :346) against the oracle."""
    inp = synthetic.make_onsite(lmax, lmax_out, N, C, batch, seed=700 + lmax, parity_mask=mask)
    (Wa, Wb), Wo = synthetic.lw_weights(lmax, lmax_out, N, C, seed=700 + lmax)
    out = cg.cgtp_onsite_lw(_cuda(inp.A), _cuda(inp.B), _cuda(Wa), _cuda(Wb), _cuda(Wo), lmax, lmax_out, N, C,
                            inp.parity_mask)
    got = out.cpu().numpy()
    ref = orc.onsite_lw(inp.A, inp.B, Wa, Wb, Wo, lmax, lmax_out, inp.parity_mask)
    e = sector_err(got, ref)
    assert max(e) < TOL, e
    # equal weights for every degree: the l-shared entry point, to rounding
    rep = lambda W, n: np.ascontiguousarray(np.repeat(W[None], n, axis=0))
    same = cg.cgtp_onsite_lw(_cuda(inp.A), _cuda(inp.B), _cuda(rep(inp.W_a, lmax + 1)), _cuda(rep(inp.W_b, lmax + 1)),
                             _cuda(rep(inp.W_out, lmax_out + 1)), lmax, lmax_out, N, C, inp.parity_mask).cpu().numpy()
    base = run_onsite(inp)
    for s in (0, 1):
        assert np.abs(same[:, s] - base[:, s]).max() <= 2e-6 * max(np.abs(base[:, s]).max(), 1e-30)


@pytest.mark.parametrize("lmax,lmax_out,N,C,nodes,mask", [
    (1, 1, 4, 4, 9, [0, 1, 1, 0]),
    (3, 4, 4, 6, 20, None),
    (6, 6, 8, 8, 40, None),
    (8, 8, 16, 8, 30, [0] * 3 + [1] * 5),
])
def test_message_lw(lmax, lmax_out, N, C, nodes, mask):
    """cgtp_message_lw: W_node[l], W_out[l] per degree (Eq.(47), Eq.(55) :427) against the oracle."""
    rng = np.random.default_rng(800 + lmax)
    deg = rng.integers(0, 10, nodes)
    deg[0] = 0
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, deg, seed=800 + lmax, parity_mask=mask)
    (Wn,), Wo = synthetic.lw_weights(lmax, lmax_out, N, C, seed=800 + lmax, n_in=1)
    out = cg.cgtp_message_lw(_cuda(m.node_feats), _cuda(m.edge_index), _cuda(m.edge_vec), _cuda(m.edge_radial), _cuda(Wn),
                             _cuda(Wo), lmax, lmax_out, N, C, m.parity_mask, check=True)
    got = out.cpu().numpy()
    ref = orc.message_lw(m.node_feats, m.edge_index, m.edge_vec, m.edge_radial, Wn, Wo, lmax, lmax_out, m.parity_mask)
    e = sector_err(got, ref)
    assert max(e) < TOL, e
    assert np.abs(got[deg == 0]).max() == 0.0


@pytest.mark.parametrize("lmax,lmax_out,N,C,nodes,mask", [
    (0, 0, 4, 4, 6, [0, 1, 0, 1]),
    (1, 2, 4, 4, 9, [0, 1, 1, 0]),
    (3, 3, 4, 6, 20, None),
    (4, 4, 8, 40, 12, [0] * 30 + [1] * 10),   # several channel blocks per receiver
    (8, 8, 8, 8, 16, None),
    (12, 12, 4, 3, 5, [0, 1, 1]),
])
def test_message_lwr(lmax, lmax_out, N, C, nodes, mask):
    """cgtp_message_lwr: l-dependent weights and the l1-dependent radial factor R~_{jicl1} (Eq.(46))."""
    rng = np.random.default_rng(900 + lmax)
    deg = rng.integers(0, 12, nodes)
    deg[0] = 0
    deg[-1] = 19
    m = synthetic.make_message(lmax, lmax_out, N, C, nodes, deg, seed=900 + lmax, parity_mask=mask)
    (Wn,), Wo = synthetic.lw_weights(lmax, lmax_out, N, C, seed=900 + lmax, n_in=1)
    rad = (m.edge_radial[:, :, None] * rng.uniform(0.5, 1.5, (m.E, C, lmax + 1))).astype(np.float32)
    out = cg.cgtp_message_lwr(_cuda(m.node_feats), _cuda(m.edge_index), _cuda(m.edge_vec), _cuda(rad), _cuda(Wn),
                              _cuda(Wo), lmax, lmax_out, N, C, m.parity_mask, check=True)
    got = out.cpu().numpy()
    ref = orc.message_lwr(m.node_feats, m.edge_index, m.edge_vec, rad, Wn, Wo, lmax, lmax_out, m.parity_mask)
    e = sector_err(got, ref)
    assert max(e) < TOL, e
    assert np.abs(got[deg == 0]).max() == 0.0
    again = cg.cgtp_message_lwr(_cuda(m.node_feats), _cuda(m.edge_index), _cuda(m.edge_vec), _cuda(rad), _cuda(Wn),
                                _cuda(Wo), lmax, lmax_out, N, C, m.parity_mask).cpu().numpy()
    assert np.array_equal(got, again)  # bitwise reproducible


def test_message_lwr_equivariance_and_inversion():
    """The full parameterisation on the device path (cgtp_message_lwr) under a random rotation and under inversion: weights
    and radial factor act within a degree, so both sectors still rotate with D^l (App. B test 5 PAPER.md:633) and pick up
    their parity labels (Table I :86-:93)."""
    lmax, N, C, nodes = 5, 8, 8, 40
    m = synthetic.make_message(lmax, lmax, N, C, nodes, 9, seed=33)
    (Wn,), Wo = synthetic.lw_weights(lmax, lmax, N, C, seed=33, n_in=1)
    rad = (m.edge_radial[:, :, None] * np.random.default_rng(4).uniform(0.5, 1.5, (m.E, C, lmax + 1))).astype(np.float32)

    def run(X, ev):
        return cg.cgtp_message_lwr(_cuda(X.astype(np.float32)), _cuda(m.edge_index), _cuda(ev.astype(np.float32)), _cuda(rad),
                                   _cuda(Wn), _cuda(Wo), lmax, lmax, N, C, m.parity_mask).cpu().numpy().astype(np.float64)

    base = run(m.node_feats, m.edge_vec)
    R = shref.random_rotation(np.random.default_rng(29))
    D = shref.wigner_D_real(lmax, R)
    rot = run(np.einsum("ab,...b->...a", D, m.node_feats.astype(np.float64)), m.edge_vec.astype(np.float64) @ R.T)
    e = sector_err(rot, np.einsum("ab,...b->...a", D, base))
    assert max(e) < TOL, e
    sign = np.concatenate([np.full(2 * l + 1, (-1.0) ** l) for l in range(lmax + 1)])
    inv = run(m.node_feats * sign, -m.edge_vec)
    assert np.abs(inv[:, 0] - base[:, 0] * sign).max() < TOL * np.abs(base[:, 0]).max()
    assert np.abs(inv[:, 1] + base[:, 1] * sign).max() < TOL * np.abs(base[:, 1]).max()

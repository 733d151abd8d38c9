"""Multi-rank host logic (paper_2605_15073_b200/parallel.py) on CPU: world_size-2 gloo runs of the
message-passing shard plan + all-gather, and the pure index arithmetic of the batch / receiver splits.

The GPU kernels are not involved: `message_sharded` is given the FP64 oracle as its `compute` step, so the
test checks that sharding + the exchange reproduce the unsharded result row for row."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import cgtp_oracle as orc
from paper_2605_15073_b200 import parallel, synthetic


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _problem():
    rng = np.random.default_rng(11)
    deg = rng.integers(0, 9, 23)
    deg[0] = 0
    deg[7] = 17
    return synthetic.make_message(2, 2, 3, 4, 23, deg, seed=77, parity_mask=[0, 1, 1, 0])


def _oracle_compute(feats, ei, ev, er, Wn, Wo, lmax, lmax_out, N, C, mask, n_recv):
    out = orc.message(feats.numpy(), ei.numpy(), ev.numpy(), er.numpy(), Wn.numpy(), Wo.numpy(), lmax, lmax_out, mask,
                      np.arange(n_recv))
    return torch.from_numpy(out)


def _worker(rank: int, world: int, port: int, result_dir: str):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        m = _problem()
        t = torch.from_numpy
        rp = parallel.row_ptr_from_receivers(m.edge_index[1], m.nodes)
        bounds = parallel.shard_receivers(rp, world)
        shard = parallel.make_shard(t(m.node_feats), t(m.edge_index), t(m.edge_vec), t(m.edge_radial), bounds, rank)
        # the exchange step on its own: every rank ends up with all node features, in node order
        feats = parallel.all_gather_node_feats(shard.node_feats, bounds)
        assert torch.equal(feats, t(m.node_feats))
        out = parallel.message_sharded(shard, bounds, t(m.W_node), t(m.W_out), m.lmax, m.lmax_out, m.N, m.C,
                                       m.parity_mask, compute=_oracle_compute)
        assert out.shape[0] == shard.hi - shard.lo
        np.save(os.path.join(result_dir, f"out{rank}.npy"), out.numpy())
        np.save(os.path.join(result_dir, f"bounds{rank}.npy"), bounds)
        dist.barrier()
    finally:
        dist.destroy_process_group()


def _field_oracle_compute(feats, ei, xe, We, Wn, Wo, lmax, lmax_out, N, Ne, C, mask, n_recv):
    # receivers are local rows 0 .. n_recv-1 of a graph whose senders index all nodes: evaluate on the sender count
    out = orc.message_field(feats.numpy(), ei.numpy(), xe.numpy(), We.numpy(), Wn.numpy(), Wo.numpy(), lmax, lmax_out, mask)
    return torch.from_numpy(out[:n_recv])


def _field_worker(rank: int, world: int, port: int, result_dir: str):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        m = _problem()
        XE, W_edge = synthetic.make_edge_field(m, 2, seed=5)
        t = torch.from_numpy
        rp = parallel.row_ptr_from_receivers(m.edge_index[1], m.nodes)
        bounds = parallel.shard_receivers(rp, world)
        shard = parallel.make_field_shard(t(m.node_feats), t(m.edge_index), t(XE), bounds, rank)
        assert shard.edge_feats.shape[0] == shard.edge_index.shape[1]
        out = parallel.message_field_sharded(shard, bounds, t(W_edge), t(m.W_node), t(m.W_out), m.lmax, m.lmax_out, m.N, 2,
                                             m.C, m.parity_mask, compute=_field_oracle_compute)
        np.save(os.path.join(result_dir, f"fout{rank}.npy"), out.numpy())
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_message_field_sharded_world2_matches_unsharded(tmp_path):
    world = 2
    mp.spawn(_field_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    m = _problem()
    XE, W_edge = synthetic.make_edge_field(m, 2, seed=5)
    ref = orc.message_field(m.node_feats, m.edge_index, XE, W_edge, m.W_node, m.W_out, m.lmax, m.lmax_out, m.parity_mask)
    got = np.concatenate([np.load(tmp_path / f"fout{r}.npy") for r in range(world)])
    assert got.shape == ref.shape
    assert np.array_equal(got, ref)


@pytest.mark.timeout(300)
def test_message_sharded_world2_matches_unsharded(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    m = _problem()
    ref = orc.message(m.node_feats, m.edge_index, m.edge_vec, m.edge_radial, m.W_node, m.W_out, m.lmax, m.lmax_out,
                      m.parity_mask)
    b0, b1 = np.load(tmp_path / "bounds0.npy"), np.load(tmp_path / "bounds1.npy")
    assert np.array_equal(b0, b1) and b0[0] == 0 and b0[-1] == m.nodes
    got = np.concatenate([np.load(tmp_path / f"out{r}.npy") for r in range(world)])
    assert got.shape == ref.shape
    assert np.array_equal(got, ref)  # same FP64 arithmetic per receiver -> identical, not merely close


def test_shard_batch_partitions_exactly():
    for batch in (0, 1, 7, 4096, 4099):
        for world in (1, 2, 3, 8):
            spans = [parallel.shard_batch(batch, world, r) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == batch
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1


def test_shard_receivers_is_contiguous_and_balanced():
    rng = np.random.default_rng(5)
    deg = rng.integers(0, 40, 1000)
    deg[100:200] = 0
    rp = np.concatenate([[0], np.cumsum(deg)]).astype(np.int64)
    for world in (1, 2, 4, 8):
        b = parallel.shard_receivers(rp, world)
        assert b.shape == (world + 1,) and b[0] == 0 and b[-1] == 1000 and np.all(np.diff(b) >= 0)
        cost = np.array([(rp[b[r + 1]] - rp[b[r]]) + 4.0 * (b[r + 1] - b[r]) for r in range(world)])
        assert cost.max() <= cost.mean() * 1.05 + 44.0  # within one node of the ideal cut
        # edge slices tile the edge list
        sl = [parallel.local_edge_slice(rp, b[r], b[r + 1]) for r in range(world)]
        assert sl[0][0] == 0 and sl[-1][1] == rp[-1] and all(x[1] == y[0] for x, y in zip(sl, sl[1:]))
    # more ranks than nodes: empty ranges are allowed
    b = parallel.shard_receivers(np.array([0, 3, 3, 5], np.int64), 8)
    assert b[0] == 0 and b[-1] == 3 and np.all(np.diff(b) >= 0)


def test_row_ptr_matches_oracle_segments_and_rejects_unsorted():
    m = _problem()
    status, ref = orc.segments(m.edge_index, m.nodes)
    assert status == 0
    assert np.array_equal(parallel.row_ptr_from_receivers(m.edge_index[1], m.nodes), ref)
    bad = m.edge_index[1].copy()
    bad[[0, -1]] = bad[[-1, 0]]
    with pytest.raises(ValueError):
        parallel.row_ptr_from_receivers(bad, m.nodes)


def test_make_shard_rebases_receivers_only():
    m = _problem()
    t = torch.from_numpy
    rp = parallel.row_ptr_from_receivers(m.edge_index[1], m.nodes)
    bounds = parallel.shard_receivers(rp, 3)
    seen = 0
    for r in range(3):
        s = parallel.make_shard(t(m.node_feats), t(m.edge_index), t(m.edge_vec), t(m.edge_radial), bounds, r)
        e0, e1 = parallel.local_edge_slice(rp, s.lo, s.hi)
        assert torch.equal(s.edge_index[0], t(m.edge_index)[0, e0:e1])            # senders stay global
        assert torch.equal(s.edge_index[1] + s.lo, t(m.edge_index)[1, e0:e1])     # receivers are local
        assert s.edge_index.shape[1] == 0 or (s.edge_index[1].min() >= 0 and s.edge_index[1].max() < s.hi - s.lo)
        seen += s.edge_index.shape[1]
    assert seen == m.E

"""Seeded synthetic workloads shaped like the paper's benchmarks (PAPER.md:479, :685 use random
inputs only) and like BASELINE.json's five configs.  DESIGN.md "Input recipe" states the recipe.

This module serves the tests, bench.py and the oracle alike and holds NONE of the method's
arithmetic: it only draws random numbers (numpy Generator, one independent child stream per tensor,
spawned from the seed in a fixed order) and evaluates the radial basis that the *caller* of the
library is responsible for (edge_radial is an input of cgtp_message).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


def _streams(seed: int, n: int):
    return [np.random.default_rng(s) for s in np.random.SeedSequence(seed).spawn(n)]


def half_mask(C: int) -> np.ndarray:
    """parity_mask with the first half of the rank channels even (0) and the second half odd (1)."""
    m = np.zeros(C, np.uint8)
    m[C // 2:] = 1
    return m


@dataclass
class OnsiteInputs:
    lmax: int
    lmax_out: int
    N: int
    C: int
    batch: int
    A: np.ndarray
    B: np.ndarray
    W_a: np.ndarray
    W_b: np.ndarray
    W_out: np.ndarray
    parity_mask: np.ndarray


def make_onsite(lmax: int, lmax_out: int, N: int, C: int, batch: int, seed: int = 0,
                parity_mask=None) -> OnsiteInputs:
    """A,B ~ N(0,1) per real-SH coefficient; W_a,W_b[C,N] ~ N(0,1/sqrt(N)); W_out[N,C] ~ N(0,1/sqrt(C))."""
    L2 = (lmax + 1) ** 2
    rA, rB, rWa, rWb, rWo = _streams(seed, 5)
    A = rA.standard_normal((batch, N, L2), dtype=np.float32)
    B = rB.standard_normal((batch, N, L2), dtype=np.float32)
    W_a = (rWa.standard_normal((C, N), dtype=np.float32) / np.float32(np.sqrt(N))).astype(np.float32)
    W_b = (rWb.standard_normal((C, N), dtype=np.float32) / np.float32(np.sqrt(N))).astype(np.float32)
    W_out = (rWo.standard_normal((N, C), dtype=np.float32) / np.float32(np.sqrt(C))).astype(np.float32)
    mask = half_mask(C) if parity_mask is None else np.ascontiguousarray(parity_mask, dtype=np.uint8)
    return OnsiteInputs(lmax, lmax_out, N, C, batch, A, B, W_a, W_b, W_out, mask)


@dataclass
class NbodyInputs:
    nu: int
    lmax: int
    lmax_out: int
    N: int
    C: int
    batch: int
    X: np.ndarray      # [nu, batch, N, (lmax+1)^2]
    W_in: np.ndarray   # [nu, C, N]
    W_out: np.ndarray  # [N, C]


def make_nbody(nu: int, lmax: int, lmax_out: int, N: int, C: int, batch: int, seed: int = 0) -> NbodyInputs:
    """nu feature sets ~ N(0,1) per real-SH coefficient; W_in[s][C,N] ~ N(0,1/sqrt(N)); W_out[N,C] ~ N(0,1/sqrt(C))."""
    L2 = (lmax + 1) ** 2
    rX, rW, rWo = _streams(seed, 3)
    X = rX.standard_normal((nu, batch, N, L2), dtype=np.float32)
    W_in = (rW.standard_normal((nu, C, N), dtype=np.float32) / np.float32(np.sqrt(N))).astype(np.float32)
    W_out = (rWo.standard_normal((N, C), dtype=np.float32) / np.float32(np.sqrt(C))).astype(np.float32)
    return NbodyInputs(nu, lmax, lmax_out, N, C, batch, X, W_in, W_out)


@dataclass
class MessageInputs:
    lmax: int
    lmax_out: int
    N: int
    C: int
    nodes: int
    E: int
    node_feats: np.ndarray
    edge_index: np.ndarray
    edge_vec: np.ndarray
    edge_radial: np.ndarray
    W_node: np.ndarray
    W_out: np.ndarray
    parity_mask: np.ndarray
    degree: np.ndarray = field(default=None)


def bessel_basis(r: np.ndarray, r_cut: float, n_basis: int = 8) -> np.ndarray:
    """b_k(r) = sqrt(2/r_c) sin(k pi r / r_c) / r, k = 1..n_basis (input generation only, R13)."""
    k = np.arange(1, n_basis + 1, dtype=np.float64)[None, :]
    r = r.astype(np.float64)[:, None]
    return np.sqrt(2.0 / r_cut) * np.sin(k * np.pi * r / r_cut) / r


def make_message(lmax: int, lmax_out: int, N: int, C: int, nodes: int, degree, r_min: float = 0.8,
                 r_max: float = 5.0, seed: int = 0, parity_mask=None) -> MessageInputs:
    """Random graph: `degree` in-edges per node (an int, or an int array [nodes] for ragged graphs),
    receiver-sorted, senders uniform random != receiver; edge vectors uniform on S^2 with lengths
    U[r_min, r_max]; edge_radial = 8 Bessel functions (cutoff r_max) x Gaussian [8,C] weights."""
    L2 = (lmax + 1) ** 2
    rX, rS, rD, rL, rRw, rWn, rWo = _streams(seed, 7)
    deg = np.full(nodes, degree, np.int64) if np.isscalar(degree) else np.asarray(degree, np.int64)
    assert deg.shape == (nodes,)
    recv = np.repeat(np.arange(nodes, dtype=np.int64), deg)
    E = int(recv.shape[0])
    # uniform sender != receiver: draw from nodes-1 values and skip over the receiver
    snd = rS.integers(0, max(nodes - 1, 1), size=E, dtype=np.int64)
    if nodes > 1:
        snd = snd + (snd >= recv)
    edge_index = np.stack([snd, recv]).astype(np.int64)
    d = rD.standard_normal((E, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    length = rL.uniform(r_min, r_max, size=E)
    edge_vec = (d * length[:, None]).astype(np.float32)
    w_rad = rRw.standard_normal((8, C)) / np.sqrt(8.0)
    edge_radial = (bessel_basis(length, r_max, 8) @ w_rad).astype(np.float32)
    node_feats = rX.standard_normal((nodes, N, L2), dtype=np.float32)
    W_node = (rWn.standard_normal((C, N), dtype=np.float32) / np.float32(np.sqrt(N))).astype(np.float32)
    W_out = (rWo.standard_normal((N, C), dtype=np.float32) / np.float32(np.sqrt(C))).astype(np.float32)
    mask = half_mask(C) if parity_mask is None else np.ascontiguousarray(parity_mask, dtype=np.uint8)
    return MessageInputs(lmax, lmax_out, N, C, nodes, E, node_feats, edge_index, edge_vec, edge_radial,
                         W_node, W_out, mask, deg)


def make_edge_field(m: MessageInputs, Ne: int, seed: int = 0):
    """Edge feature field of the two-field coupling Eq.(28) for the graph `m`: edge_feats [E, Ne, L2]
    ~N(0,1) per real-SH coefficient (a deeper layer's edge message, no longer of the form R.Y) and its CP projection
    weights W_edge [C, Ne] ~N(0, 1/sqrt(Ne)).  Holds none of the method's arithmetic."""
    rF, rW = _streams(seed + 7919, 2)
    L2 = (m.lmax + 1) ** 2
    edge_feats = rF.standard_normal((m.E, Ne, L2), dtype=np.float32)
    W_edge = (rW.standard_normal((m.C, Ne), dtype=np.float32) / np.float32(np.sqrt(Ne))).astype(np.float32)
    return edge_feats, W_edge


# ---------------------------------------------------------------------------------------------
# Parity-labelled inputs (Sec. VI, VII C a-c, e): a parity-slot axis on the
# features (slot 0 natural parity (-1)^l, slot 1 opposite) and one independent weight set per run.
# ---------------------------------------------------------------------------------------------
@dataclass
class OnsiteParityInputs:
    lmax: int
    lmax_out: int
    N: int
    C: int
    batch: int
    A: np.ndarray      # [batch, 2, N, L2]
    B: np.ndarray      # [batch, 2, N, L2]
    W_a: np.ndarray    # [16, C, N]
    W_b: np.ndarray    # [16, C, N]
    W_out: np.ndarray  # [16, N, C]


def make_onsite_parity(lmax: int, lmax_out: int, N: int, C: int, batch: int, seed: int = 0) -> OnsiteParityInputs:
    """Same distributions as make_onsite, with both parity slots populated and 16 weight sets."""
    L2 = (lmax + 1) ** 2
    rA, rB, rWa, rWb, rWo = _streams(seed, 5)
    A = rA.standard_normal((batch, 2, N, L2), dtype=np.float32)
    B = rB.standard_normal((batch, 2, N, L2), dtype=np.float32)
    W_a = (rWa.standard_normal((16, C, N), dtype=np.float32) / np.float32(np.sqrt(N))).astype(np.float32)
    W_b = (rWb.standard_normal((16, C, N), dtype=np.float32) / np.float32(np.sqrt(N))).astype(np.float32)
    W_out = (rWo.standard_normal((16, N, C), dtype=np.float32) / np.float32(np.sqrt(C))).astype(np.float32)
    return OnsiteParityInputs(lmax, lmax_out, N, C, batch, A, B, W_a, W_b, W_out)


@dataclass
class MessageParityInputs:
    lmax: int
    lmax_out: int
    N: int
    C: int
    nodes: int
    E: int
    node_feats: np.ndarray   # [nodes, 2, N, L2]
    edge_index: np.ndarray   # [2, E]
    edge_vec: np.ndarray     # [E, 3]
    edge_radial: np.ndarray  # [E, 8, C]
    W_node: np.ndarray       # [8, C, N]
    W_out: np.ndarray        # [8, N, C]
    degree: np.ndarray = field(default=None)


def make_message_parity(lmax: int, lmax_out: int, N: int, C: int, nodes: int, degree, r_min: float = 0.8,
                        r_max: float = 5.0, seed: int = 0) -> MessageParityInputs:
    """The graph and edge vectors of make_message (same seed -> same graph); node features in both parity
    slots; per run one Gaussian [8, C] radial weight matrix, W_node and W_out."""
    g = make_message(lmax, lmax_out, 1, 1, nodes, degree, r_min, r_max, seed)
    L2 = (lmax + 1) ** 2
    rX, rRw, rWn, rWo = _streams(seed + 7919, 4)
    length = np.linalg.norm(g.edge_vec.astype(np.float64), axis=1)
    w_rad = rRw.standard_normal((8, 8 * C)) / np.sqrt(8.0)
    edge_radial = (bessel_basis(length, r_max, 8) @ w_rad).astype(np.float32).reshape(g.E, 8, C)
    node_feats = rX.standard_normal((nodes, 2, N, L2), dtype=np.float32)
    W_node = (rWn.standard_normal((8, C, N), dtype=np.float32) / np.float32(np.sqrt(N))).astype(np.float32)
    W_out = (rWo.standard_normal((8, N, C), dtype=np.float32) / np.float32(np.sqrt(C))).astype(np.float32)
    return MessageParityInputs(lmax, lmax_out, N, C, nodes, g.E, node_feats, g.edge_index, g.edge_vec, edge_radial,
                               W_node, W_out, g.degree)


@dataclass
class FieldParityInputs:
    lmax: int
    lmax_out: int
    N: int
    Ne: int
    C: int
    nodes: int
    E: int
    node_feats: np.ndarray   # [nodes, 2, N, L2]
    edge_index: np.ndarray   # [2, E]
    edge_feats: np.ndarray   # [E, 2, Ne, L2]
    W_edge: np.ndarray       # [16, C, Ne]
    W_node: np.ndarray       # [16, C, N]
    W_out: np.ndarray        # [16, N, C]
    degree: np.ndarray


def make_field_parity(lmax: int, lmax_out: int, N: int, Ne: int, C: int, nodes: int, degree, seed: int = 0) -> FieldParityInputs:
    """Two parity-bearing fields (Eq.(28), Sec. VII C f :471): the graph of make_message (same seed -> same
    graph), node and edge feature fields ~N(0,1) in both parity slots, one weight set per run (16 runs)."""
    g = make_message(lmax, lmax_out, 1, 1, nodes, degree, 0.8, 5.0, seed)
    L2 = (lmax + 1) ** 2
    rX, rE, rWe, rWn, rWo = _streams(seed + 104729, 5)
    node_feats = rX.standard_normal((nodes, 2, N, L2), dtype=np.float32)
    edge_feats = rE.standard_normal((g.E, 2, Ne, L2), dtype=np.float32)
    W_edge = (rWe.standard_normal((16, C, Ne), dtype=np.float32) / np.float32(np.sqrt(Ne))).astype(np.float32)
    W_node = (rWn.standard_normal((16, C, N), dtype=np.float32) / np.float32(np.sqrt(N))).astype(np.float32)
    W_out = (rWo.standard_normal((16, N, C), dtype=np.float32) / np.float32(np.sqrt(C))).astype(np.float32)
    return FieldParityInputs(lmax, lmax_out, N, Ne, C, nodes, g.E, node_feats, g.edge_index, edge_feats, W_edge, W_node,
                             W_out, g.degree)


# ---------------------------------------------------------------------------------------------
# l-dependent CP weights (Eq.(35) :322, Eq.(41) :346, Eq.(47) :398): the same inputs as
# make_onsite / make_message with one weight matrix per degree l.
# ---------------------------------------------------------------------------------------------
def lw_weights(lmax: int, lmax_out: int, N: int, C: int, seed: int, n_in: int = 2):
    """n_in input weight stacks [lmax+1, C, N] ~ N(0, 1/sqrt(N)) and one output stack [lmax_out+1, N, C] ~ N(0, 1/sqrt(C))."""
    rs = _streams(seed + 104729, n_in + 1)
    w_in = [(r.standard_normal((lmax + 1, C, N), dtype=np.float32) / np.float32(np.sqrt(N))).astype(np.float32)
            for r in rs[:n_in]]
    w_out = (rs[n_in].standard_normal((lmax_out + 1, N, C), dtype=np.float32) / np.float32(np.sqrt(C))).astype(np.float32)
    return w_in, w_out


# BASELINE.json configs (index = position in BASELINE.json "configs").
def config(idx: int, lmax: int | None = None, seed: int = 0):
    if idx == 0:
        return make_onsite(2, 2, 8, 8, 64, seed)
    if idx == 1:
        return make_onsite(6, 6, 64, 64, 4096, seed)
    if idx == 2:
        return make_message(4, 4, 128, 128, 2048, 16, 0.8, 5.0, seed, parity_mask=np.zeros(128, np.uint8))
    if idx == 3:
        assert lmax in (2, 4, 8, 12, 16, 20)
        return make_onsite(lmax, lmax, 32, 32, 16384, seed)
    if idx == 4:
        return make_message(8, 8, 128, 128, 16384, 32, 0.8, 6.0, seed)
    raise ValueError(idx)

"""ctypes front end of the FP64 CPU oracle (oracle/cgtp_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and the cpu_baseline /
--impl reference legs of bench.py.  The product package never imports this module and this
module never imports the product package.

Every function converts its inputs to float64 and calls the C routine of the same name; no
arithmetic of the method lives in this file.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cgtp_oracle.c")
_LIB = os.path.join(_HERE, "libcgtp_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C99 + OpenMP).  Returns the path of the shared object."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build())
    d, i, i64 = ctypes.c_double, ctypes.c_int, ctypes.c_int64
    p = ctypes.c_void_p
    lib.oracle_wigner3j.restype = d
    lib.oracle_wigner3j.argtypes = [i] * 6
    lib.oracle_cg.restype = d
    lib.oracle_cg.argtypes = [i] * 6
    lib.oracle_cg000_closed.restype = d
    lib.oracle_cg000_closed.argtypes = [i] * 3
    lib.oracle_gaunt_complex.restype = d
    lib.oracle_gaunt_complex.argtypes = [i] * 6
    lib.oracle_kappa_inv_imag.restype = d
    lib.oracle_kappa_inv_imag.argtypes = [i] * 3
    lib.oracle_q_complex_imag.restype = d
    lib.oracle_q_complex_imag.argtypes = [i] * 6
    lib.oracle_real_coupling.restype = i64
    lib.oracle_real_coupling.argtypes = [i, i, i, p, p, p, p, p]
    lib.oracle_real_sh.restype = None
    lib.oracle_real_sh.argtypes = [i, d, d, d, p]
    lib.oracle_segments.restype = i
    lib.oracle_segments.argtypes = [p, i64, i64, p]
    lib.oracle_onsite.restype = i
    lib.oracle_onsite.argtypes = [p, p, p, p, p, i, i, i, i, p, p, i64]
    lib.oracle_message.restype = i
    lib.oracle_message.argtypes = [p, p, p, p, p, p, i, i, i, i, p, p, i64, i64, p, i64]
    lib.oracle_message_parity.restype = i
    lib.oracle_message_parity.argtypes = [p, p, p, p, p, p, p, i, i, i, i, p, i64, i64, p, i64]
    lib.oracle_onsite_parity.restype = i
    lib.oracle_onsite_parity.argtypes = [p, p, p, p, p, i, i, i, i, p, i64]
    lib.oracle_onsite_lw.restype = i
    lib.oracle_onsite_lw.argtypes = [p, p, p, p, p, i, i, i, i, p, p, i64]
    lib.oracle_message_lw.restype = i
    lib.oracle_message_lw.argtypes = [p, p, p, p, p, p, i, i, i, i, p, p, i64, i64]
    lib.oracle_message_lwr.restype = i
    lib.oracle_message_lwr.argtypes = lib.oracle_message_lw.argtypes
    lib.oracle_onsite_nbody.restype = i
    lib.oracle_onsite_nbody.argtypes = [p, p, p, i, i, i, i, i, p, i64]
    lib.oracle_message_field.restype = i
    lib.oracle_message_field.argtypes = [p, p, p, p, p, p, i, i, i, i, i, p, p, i64, i64]
    lib.oracle_message_field_lw.restype = i
    lib.oracle_message_field_lw.argtypes = lib.oracle_message_field.argtypes
    lib.oracle_message_field_parity.restype = i
    lib.oracle_message_field_parity.argtypes = [p, p, p, p, p, p, i, i, i, i, i, p, i64, i64]
    lib.oracle_num_threads.restype = i
    lib.oracle_num_threads.argtypes = []
    _lib = lib
    return lib


def _f64(a):
    return np.ascontiguousarray(np.asarray(a), dtype=np.float64)


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def wigner3j(j1, j2, j3, m1, m2, m3) -> float:
    return _load().oracle_wigner3j(j1, j2, j3, m1, m2, m3)


def cg(l1, m1, l2, m2, l, m) -> float:
    return _load().oracle_cg(l1, m1, l2, m2, l, m)


def cg000_closed(l1, l2, l) -> float:
    return _load().oracle_cg000_closed(l1, l2, l)


def gaunt_complex(l1, m1, l2, m2, l, m) -> float:
    return _load().oracle_gaunt_complex(l1, m1, l2, m2, l, m)


def kappa_inv_imag(l1, l2, l) -> float:
    return _load().oracle_kappa_inv_imag(l1, l2, l)


def q_complex_imag(l1, m1, l2, m2, l, m) -> float:
    return _load().oracle_q_complex_imag(l1, m1, l2, m2, l, m)


def real_coupling(lmax: int, lmax_out: int, odd: bool):
    """Sparse real-basis coupling tensor (i1, i2, io, val, max_imag)."""
    lib = _load()
    mi = ctypes.c_double(0.0)
    nnz = lib.oracle_real_coupling(lmax, lmax_out, int(odd), None, None, None, None, ctypes.byref(mi))
    if nnz < 0:
        raise RuntimeError("oracle coupling cache full")
    i1 = np.empty(nnz, np.int32)
    i2 = np.empty(nnz, np.int32)
    io = np.empty(nnz, np.int32)
    val = np.empty(nnz, np.float64)
    lib.oracle_real_coupling(lmax, lmax_out, int(odd), _ptr(i1), _ptr(i2), _ptr(io), _ptr(val), ctypes.byref(mi))
    return i1, i2, io, val, mi.value


def real_coupling_dense(lmax: int, lmax_out: int, odd: bool) -> np.ndarray:
    i1, i2, io, val, _ = real_coupling(lmax, lmax_out, odd)
    t = np.zeros(((lmax + 1) ** 2, (lmax + 1) ** 2, (lmax_out + 1) ** 2))
    t[i1, i2, io] = val
    return t


def real_sh(lmax: int, xyz) -> np.ndarray:
    """Real spherical harmonics Y[(lmax+1)^2] of one direction (need not be normalised)."""
    out = np.empty((lmax + 1) ** 2, np.float64)
    x, y, z = (float(v) for v in xyz)
    _load().oracle_real_sh(lmax, x, y, z, _ptr(out))
    return out


def segments(edge_index, nodes: int):
    """CSR offsets row_ptr[nodes+1] of a receiver-sorted edge list; returns (status, row_ptr)."""
    ei = np.ascontiguousarray(np.asarray(edge_index), dtype=np.int64)
    E = ei.shape[1]
    rp = np.zeros(nodes + 1, np.int64)
    rc = _load().oracle_segments(_ptr(ei), E, nodes, _ptr(rp))
    return rc, rp


def onsite(A, B, W_a, W_b, W_out, lmax, lmax_out, parity_mask) -> np.ndarray:
    """out[batch, 2, N, (lmax_out+1)^2] in float64."""
    A, B, W_a, W_b, W_out = map(_f64, (A, B, W_a, W_b, W_out))
    batch, N, L2 = A.shape
    C = W_a.shape[0]
    assert L2 == (lmax + 1) ** 2 and B.shape == A.shape
    assert W_a.shape == (C, N) and W_b.shape == (C, N) and W_out.shape == (N, C)
    mask = np.ascontiguousarray(np.asarray(parity_mask), dtype=np.uint8)
    assert mask.shape == (C,)
    out = np.zeros((batch, 2, N, (lmax_out + 1) ** 2), np.float64)
    rc = _load().oracle_onsite(_ptr(A), _ptr(B), _ptr(W_a), _ptr(W_b), _ptr(W_out), lmax, lmax_out, N, C,
                               _ptr(mask), _ptr(out), batch)
    if rc:
        raise RuntimeError(f"oracle_onsite failed with code {rc}")
    return out


def message(node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, parity_mask,
            recv_list=None) -> np.ndarray:
    """out[n_recv or nodes, 2, N, (lmax_out+1)^2] in float64."""
    X, ev, er, W_node, W_out = map(_f64, (node_feats, edge_vec, edge_radial, W_node, W_out))
    ei = np.ascontiguousarray(np.asarray(edge_index), dtype=np.int64)
    nodes, N, L2 = X.shape
    E = ei.shape[1]
    C = W_node.shape[0]
    assert L2 == (lmax + 1) ** 2 and ev.shape == (E, 3) and er.shape == (E, C)
    assert W_node.shape == (C, N) and W_out.shape == (N, C)
    mask = np.ascontiguousarray(np.asarray(parity_mask), dtype=np.uint8)
    if recv_list is None:
        rl, nr, rlp = None, nodes, None
    else:
        rl = np.ascontiguousarray(np.asarray(recv_list), dtype=np.int64)
        nr, rlp = rl.shape[0], _ptr(rl)
    out = np.zeros((nr, 2, N, (lmax_out + 1) ** 2), np.float64)
    rc = _load().oracle_message(_ptr(X), _ptr(ei), _ptr(ev), _ptr(er), _ptr(W_node), _ptr(W_out), lmax, lmax_out,
                                N, C, _ptr(mask), _ptr(out), nodes, E, rlp, nr if rl is not None else 0)
    if rc:
        raise RuntimeError(f"oracle_message failed with code {rc}")
    return out


def onsite_parity(A, B, W_a, W_b, W_out, lmax, lmax_out) -> np.ndarray:
    """Parity-labelled on-site contraction (Sec. VII C e).  A, B [batch,2,N,L2] (slot 0 natural, 1 opposite parity);
    W_a, W_b [16,C,N], W_out [16,N,C], run = 8*cat + 4*s1 + 2*s2 + tau.  out[batch,2,N,(lmax_out+1)^2]."""
    A, B, W_a, W_b, W_out = map(_f64, (A, B, W_a, W_b, W_out))
    batch, two, N, L2 = A.shape
    C = W_a.shape[1]
    assert two == 2 and L2 == (lmax + 1) ** 2 and B.shape == A.shape
    assert W_a.shape == (16, C, N) and W_b.shape == (16, C, N) and W_out.shape == (16, N, C)
    out = np.zeros((batch, 2, N, (lmax_out + 1) ** 2), np.float64)
    rc = _load().oracle_onsite_parity(_ptr(A), _ptr(B), _ptr(W_a), _ptr(W_b), _ptr(W_out), lmax, lmax_out, N, C,
                                      _ptr(out), batch)
    if rc:
        raise RuntimeError(f"oracle_onsite_parity failed with code {rc}")
    return out


def message_parity(node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, recv_list=None,
                   l1_weight=None) -> np.ndarray:
    """Parity-labelled message passing (Sec. VII C a-c).  node_feats [nodes,2,N,L2]; edge_radial [E,8,C];
    W_node [8,C,N]; W_out [8,N,C]; run = 4*cat + 2*s_out + tau.  out[n_recv or nodes,2,N,(lmax_out+1)^2]."""
    X, ev, er, W_node, W_out = map(_f64, (node_feats, edge_vec, edge_radial, W_node, W_out))
    ei = np.ascontiguousarray(np.asarray(edge_index), dtype=np.int64)
    nodes, two, N, L2 = X.shape
    E = ei.shape[1]
    C = W_node.shape[1]
    assert two == 2 and L2 == (lmax + 1) ** 2 and ev.shape == (E, 3) and er.shape == (E, 8, C)
    assert W_node.shape == (8, C, N) and W_out.shape == (8, N, C)
    if recv_list is None:
        rl, nr, rlp = None, nodes, None
    else:
        rl = np.ascontiguousarray(np.asarray(recv_list), dtype=np.int64)
        nr, rlp = rl.shape[0], _ptr(rl)
    lw = None if l1_weight is None else _f64(l1_weight)
    assert lw is None or lw.shape == (lmax + 1,)
    out = np.zeros((nr, 2, N, (lmax_out + 1) ** 2), np.float64)
    rc = _load().oracle_message_parity(_ptr(X), _ptr(ei), _ptr(ev), _ptr(er), None if lw is None else _ptr(lw),
                                       _ptr(W_node), _ptr(W_out), lmax, lmax_out, N, C, _ptr(out), nodes, E, rlp,
                                       nr if rl is not None else 0)
    if rc:
        raise RuntimeError(f"oracle_message_parity failed with code {rc}")
    return out


def onsite_lw(A, B, W_a, W_b, W_out, lmax, lmax_out, parity_mask) -> np.ndarray:
    """On-site contraction with l-dependent CP weights (Eq.(35), (41)): W_a, W_b [lmax+1, C, N], W_out [lmax_out+1, N, C]."""
    A, B, W_a, W_b, W_out = map(_f64, (A, B, W_a, W_b, W_out))
    batch, N, L2 = A.shape
    C = W_a.shape[1]
    assert L2 == (lmax + 1) ** 2 and B.shape == A.shape
    assert W_a.shape == (lmax + 1, C, N) and W_b.shape == (lmax + 1, C, N) and W_out.shape == (lmax_out + 1, N, C)
    mask = np.ascontiguousarray(np.asarray(parity_mask), dtype=np.uint8)
    assert mask.shape == (C,)
    out = np.zeros((batch, 2, N, (lmax_out + 1) ** 2), np.float64)
    rc = _load().oracle_onsite_lw(_ptr(A), _ptr(B), _ptr(W_a), _ptr(W_b), _ptr(W_out), lmax, lmax_out, N, C,
                                  _ptr(mask), _ptr(out), batch)
    if rc:
        raise RuntimeError(f"oracle_onsite_lw failed with code {rc}")
    return out


def message_lw(node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, parity_mask) -> np.ndarray:
    """Message passing with l-dependent node / output weights: W_node [lmax+1, C, N], W_out [lmax_out+1, N, C]."""
    X, ev, er, W_node, W_out = map(_f64, (node_feats, edge_vec, edge_radial, W_node, W_out))
    ei = np.ascontiguousarray(np.asarray(edge_index), dtype=np.int64)
    nodes, N, L2 = X.shape
    E = ei.shape[1]
    C = W_node.shape[1]
    assert L2 == (lmax + 1) ** 2 and ev.shape == (E, 3) and er.shape == (E, C)
    assert W_node.shape == (lmax + 1, C, N) and W_out.shape == (lmax_out + 1, N, C)
    mask = np.ascontiguousarray(np.asarray(parity_mask), dtype=np.uint8)
    out = np.zeros((nodes, 2, N, (lmax_out + 1) ** 2), np.float64)
    rc = _load().oracle_message_lw(_ptr(X), _ptr(ei), _ptr(ev), _ptr(er), _ptr(W_node), _ptr(W_out), lmax, lmax_out,
                                   N, C, _ptr(mask), _ptr(out), nodes, E)
    if rc:
        raise RuntimeError(f"oracle_message_lw failed with code {rc}")
    return out


def message_lwr(node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, parity_mask) -> np.ndarray:
    """Message passing in the paper's full parameterisation: W_node [lmax+1, C, N], W_out [lmax_out+1, N, C] and the
    l1-dependent radial factor edge_radial [E, C, lmax+1] (Eq.(46))."""
    X, ev, er, W_node, W_out = map(_f64, (node_feats, edge_vec, edge_radial, W_node, W_out))
    ei = np.ascontiguousarray(np.asarray(edge_index), dtype=np.int64)
    nodes, N, L2 = X.shape
    E = ei.shape[1]
    C = W_node.shape[1]
    assert L2 == (lmax + 1) ** 2 and ev.shape == (E, 3) and er.shape == (E, C, lmax + 1)
    assert W_node.shape == (lmax + 1, C, N) and W_out.shape == (lmax_out + 1, N, C)
    mask = np.ascontiguousarray(np.asarray(parity_mask), dtype=np.uint8)
    out = np.zeros((nodes, 2, N, (lmax_out + 1) ** 2), np.float64)
    rc = _load().oracle_message_lwr(_ptr(X), _ptr(ei), _ptr(ev), _ptr(er), _ptr(W_node), _ptr(W_out), lmax, lmax_out,
                                    N, C, _ptr(mask), _ptr(out), nodes, E)
    if rc:
        raise RuntimeError(f"oracle_message_lwr failed with code {rc}")
    return out


def onsite_nbody(X, W_in, W_out, lmax, lmax_out) -> np.ndarray:
    """nu-body pointwise product: X [nu, batch, N, (lmax+1)^2], W_in [nu, C, N], W_out [N, C]
    -> out[batch, N, (lmax_out+1)^2] in float64."""
    X, W_in, W_out = map(_f64, (X, W_in, W_out))
    nu, batch, N, L2 = X.shape
    C = W_in.shape[1]
    assert L2 == (lmax + 1) ** 2 and W_in.shape == (nu, C, N) and W_out.shape == (N, C)
    out = np.zeros((batch, N, (lmax_out + 1) ** 2), np.float64)
    rc = _load().oracle_onsite_nbody(_ptr(X), _ptr(W_in), _ptr(W_out), nu, lmax, lmax_out, N, C, _ptr(out), batch)
    if rc:
        raise RuntimeError(f"oracle_onsite_nbody failed with code {rc}")
    return out


def message_field(node_feats, edge_index, edge_feats, W_edge, W_node, W_out, lmax, lmax_out, parity_mask) -> np.ndarray:
    """Two-field coupling Eq.(28): node_feats [nodes,N,L2], edge_feats [E,Ne,L2], W_edge [C,Ne], W_node [C,N],
    W_out [N,C]; out [nodes, 2, N, (lmax_out+1)^2] in float64."""
    X, XE, W_edge, W_node, W_out = map(_f64, (node_feats, edge_feats, W_edge, W_node, W_out))
    ei = np.ascontiguousarray(np.asarray(edge_index), dtype=np.int64)
    nodes, N, L2 = X.shape
    E, Ne, _ = XE.shape
    C = W_node.shape[0]
    assert L2 == (lmax + 1) ** 2 and XE.shape == (E, Ne, L2) and ei.shape == (2, E)
    assert W_edge.shape == (C, Ne) and W_node.shape == (C, N) and W_out.shape == (N, C)
    mask = np.ascontiguousarray(np.asarray(parity_mask), dtype=np.uint8)
    assert mask.shape == (C,)
    out = np.zeros((nodes, 2, N, (lmax_out + 1) ** 2), np.float64)
    rc = _load().oracle_message_field(_ptr(X), _ptr(ei), _ptr(XE), _ptr(W_edge), _ptr(W_node), _ptr(W_out), lmax,
                                      lmax_out, N, Ne, C, _ptr(mask), _ptr(out), nodes, E)
    if rc:
        raise RuntimeError(f"oracle_message_field failed with code {rc}")
    return out


def message_field_parity(node_feats, edge_index, edge_feats, W_edge, W_node, W_out, lmax, lmax_out) -> np.ndarray:
    """Two parity-bearing fields, Eq.(28) with slot axes: node_feats [nodes,2,N,L2], edge_feats [E,2,Ne,L2] (slot 0 natural,
    1 opposite parity); W_edge [16,C,Ne], W_node [16,C,N], W_out [16,N,C], run = 8*cat + 4*s1 + 2*s2 + tau (s1: edge slot,
    s2: node slot).  out [nodes, 2, N, (lmax_out+1)^2]."""
    X, XE, W_edge, W_node, W_out = map(_f64, (node_feats, edge_feats, W_edge, W_node, W_out))
    ei = np.ascontiguousarray(np.asarray(edge_index), dtype=np.int64)
    nodes, two, N, L2 = X.shape
    E, two_e, Ne, _ = XE.shape
    C = W_node.shape[1]
    assert two == 2 and two_e == 2 and L2 == (lmax + 1) ** 2 and XE.shape == (E, 2, Ne, L2) and ei.shape == (2, E)
    assert W_edge.shape == (16, C, Ne) and W_node.shape == (16, C, N) and W_out.shape == (16, N, C)
    out = np.zeros((nodes, 2, N, (lmax_out + 1) ** 2), np.float64)
    rc = _load().oracle_message_field_parity(_ptr(X), _ptr(ei), _ptr(XE), _ptr(W_edge), _ptr(W_node), _ptr(W_out), lmax,
                                             lmax_out, N, Ne, C, _ptr(out), nodes, E)
    if rc:
        raise RuntimeError(f"oracle_message_field_parity failed with code {rc}")
    return out


def message_field_lw(node_feats, edge_index, edge_feats, W_edge, W_node, W_out, lmax, lmax_out, parity_mask) -> np.ndarray:
    """Two-field coupling with l-dependent weights: W_edge [lmax+1,C,Ne], W_node [lmax+1,C,N], W_out [lmax_out+1,N,C]."""
    X, XE, W_edge, W_node, W_out = map(_f64, (node_feats, edge_feats, W_edge, W_node, W_out))
    ei = np.ascontiguousarray(np.asarray(edge_index), dtype=np.int64)
    nodes, N, L2 = X.shape
    E, Ne, _ = XE.shape
    C = W_node.shape[1]
    assert L2 == (lmax + 1) ** 2 and XE.shape == (E, Ne, L2) and ei.shape == (2, E)
    assert W_edge.shape == (lmax + 1, C, Ne) and W_node.shape == (lmax + 1, C, N) and W_out.shape == (lmax_out + 1, N, C)
    mask = np.ascontiguousarray(np.asarray(parity_mask), dtype=np.uint8)
    assert mask.shape == (C,)
    out = np.zeros((nodes, 2, N, (lmax_out + 1) ** 2), np.float64)
    rc = _load().oracle_message_field_lw(_ptr(X), _ptr(ei), _ptr(XE), _ptr(W_edge), _ptr(W_node), _ptr(W_out), lmax,
                                         lmax_out, N, Ne, C, _ptr(mask), _ptr(out), nodes, E)
    if rc:
        raise RuntimeError(f"oracle_message_field_lw failed with code {rc}")
    return out


def num_threads() -> int:
    return _load().oracle_num_threads()

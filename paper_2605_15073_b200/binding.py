"""Thin ctypes binding of libcgtp.so (the C ABI of include/cgtp.h).

Argument marshalling only: every step of the hot path runs in the CUDA kernels of csrc/.  PyTorch is
used for device memory (tensors, the workspace) and streams.  There is no CPU fallback: if the shared
library is missing or the tensors are not CUDA tensors, the call raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libcgtp.so")

OK, ERR_INVALID, ERR_UNSUPPORTED, ERR_CUDA, ERR_GRAPH = 0, 1, 2, 3, 4


class CgtpError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"cgtp error {code}: {msg}")
        self.code = code


_lib = None


def lib() -> ctypes.CDLL:
    """Loads libcgtp.so (built by `python -m paper_2605_15073_b200.build`).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} not found: build it with `python -m paper_2605_15073_b200.build` "
                          "(there is no CPU fallback)")
    L = ctypes.CDLL(_LIB_PATH)
    vp, i, i64, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_size_t
    L.cgtp_version.restype = i
    L.cgtp_last_error.restype = ctypes.c_char_p
    L.cgtp_max_lmax.restype = i
    L.cgtp_grid_shape.restype = i
    L.cgtp_grid_shape.argtypes = [i, i, ctypes.POINTER(i), ctypes.POINTER(i)]
    L.cgtp_onsite_workspace_bytes.restype = sz
    L.cgtp_onsite_workspace_bytes.argtypes = [i, i, i, i, i64]
    L.cgtp_onsite.restype = i
    L.cgtp_onsite.argtypes = [vp, vp, vp, vp, vp, i, i, i, i, vp, vp, i64, vp, sz, vp]
    L.cgtp_onsite_static.restype = i
    L.cgtp_onsite_static.argtypes = [vp, vp, vp, vp, vp, i, i, i, i, vp, vp, i64, vp]
    L.cgtp_message_workspace_bytes.restype = sz
    L.cgtp_message_workspace_bytes.argtypes = [i, i, i, i, vp, i64, i64]
    L.cgtp_message.restype = i
    L.cgtp_message.argtypes = [vp, vp, vp, vp, vp, vp, i, i, i, i, vp, vp, i64, i64, vp, sz, vp]
    L.cgtp_message_bipartite_workspace_bytes.restype = sz
    L.cgtp_message_bipartite_workspace_bytes.argtypes = [i, i, i, i, vp, i64, i64, i64]
    L.cgtp_message_bipartite.restype = i
    L.cgtp_message_bipartite.argtypes = [vp, vp, vp, vp, vp, vp, i, i, i, i, vp, vp, i64, i64, i64, vp, sz, vp]
    L.cgtp_onsite_parity_workspace_bytes.restype = sz
    L.cgtp_onsite_parity_workspace_bytes.argtypes = [i, i, i, i, i64]
    L.cgtp_onsite_parity.restype = i
    L.cgtp_onsite_parity.argtypes = [vp, vp, vp, vp, vp, i, i, i, i, vp, i64, vp, sz, vp]
    L.cgtp_message_parity_workspace_bytes.restype = sz
    L.cgtp_message_parity_workspace_bytes.argtypes = [i, i, i, i, i64, i64]
    L.cgtp_message_parity.restype = i
    L.cgtp_message_parity.argtypes = [vp, vp, vp, vp, vp, vp, i, i, i, i, vp, i64, i64, vp, sz, vp]
    L.cgtp_message_field_workspace_bytes.restype = sz
    L.cgtp_message_field_workspace_bytes.argtypes = [i, i, i, i, i, i64, i64]
    L.cgtp_message_field.restype = i
    L.cgtp_message_field.argtypes = [vp, vp, vp, vp, vp, vp, i, i, i, i, i, vp, vp, i64, i64, vp, sz, vp]
    L.cgtp_message_field_lw.restype = i
    L.cgtp_message_field_lw.argtypes = L.cgtp_message_field.argtypes
    L.cgtp_message_field_bipartite_workspace_bytes.restype = sz
    L.cgtp_message_field_bipartite_workspace_bytes.argtypes = [i, i, i, i, i, i64, i64, i64]
    L.cgtp_message_field_bipartite.restype = i
    L.cgtp_message_field_bipartite.argtypes = [vp, vp, vp, vp, vp, vp, i, i, i, i, i, vp, vp, i64, i64, i64, vp, sz, vp]
    L.cgtp_message_field_parity_workspace_bytes.restype = sz
    L.cgtp_message_field_parity_workspace_bytes.argtypes = [i, i, i, i, i, i64, i64]
    L.cgtp_message_field_parity.restype = i
    L.cgtp_message_field_parity.argtypes = [vp, vp, vp, vp, vp, vp, i, i, i, i, i, vp, i64, i64, vp, sz, vp]
    L.cgtp_onsite_nbody_workspace_bytes.restype = sz
    L.cgtp_onsite_nbody_workspace_bytes.argtypes = [i, i, i, i, i, i64]
    L.cgtp_onsite_nbody.restype = i
    L.cgtp_onsite_nbody.argtypes = [vp, vp, vp, i, i, i, i, i, vp, i64, vp, sz, vp]
    L.cgtp_grid_shape_nu.restype = i
    L.cgtp_grid_shape_nu.argtypes = [i, i, i, ctypes.POINTER(i), ctypes.POINTER(i)]
    L.cgtp_onsite_lw.restype = i
    L.cgtp_onsite_lw.argtypes = L.cgtp_onsite.argtypes
    L.cgtp_message_lwr.restype = i
    L.cgtp_message_lwr.argtypes = L.cgtp_message.argtypes
    L.cgtp_message_lw.restype = i
    L.cgtp_message_lw.argtypes = L.cgtp_message.argtypes
    L.cgtp_message_status.restype = i
    L.cgtp_message_status.argtypes = [vp, vp]
    L.cgtp_build_segments.restype = i
    L.cgtp_build_segments.argtypes = [vp, i64, i64, vp, vp, vp]
    L.cgtp_onsite_host.restype = i
    L.cgtp_onsite_host.argtypes = [vp, vp, vp, vp, vp, i, i, i, i, vp, vp, i64, vp]
    L.cgtp_message_host.restype = i
    L.cgtp_message_host.argtypes = [vp, vp, vp, vp, vp, vp, i, i, i, i, vp, vp, i64, i64, vp]
    L.cgtp_set_math_mode.restype = i
    L.cgtp_set_math_mode.argtypes = [i]
    L.cgtp_get_math_mode.restype = i
    L.cgtp_set_kernel_path.restype = i
    L.cgtp_set_kernel_path.argtypes = [i]
    L.cgtp_get_kernel_path.restype = i
    L.cgtp_fma_peak.restype = i
    L.cgtp_fma_peak.argtypes = [i, ctypes.c_double, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double), vp]
    L.cgtp_launch_count.restype = i64
    L.cgtp_profile_kinds.restype = i
    L.cgtp_profile_kind_name.restype = ctypes.c_char_p
    L.cgtp_profile_kind_name.argtypes = [i]
    L.cgtp_profile_enable.restype = i
    L.cgtp_profile_enable.argtypes = [i]
    L.cgtp_profile_collect.restype = i
    L.cgtp_profile_collect.argtypes = [vp, vp]
    _lib = L
    return L


def _check(rc: int):
    if rc != OK:
        raise CgtpError(rc, lib().cgtp_last_error().decode())


def _mask(parity_mask, C: int) -> np.ndarray:
    m = np.ascontiguousarray(np.asarray(parity_mask), dtype=np.uint8)
    if m.shape != (C,):
        raise ValueError(f"parity_mask must have shape ({C},)")
    return m


def _dev(t: torch.Tensor, dtype, name: str) -> torch.Tensor:
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name} must be contiguous {dtype}")
    return t


def _stream_ptr(stream) -> int:
    s = torch.cuda.current_stream() if stream is None else stream
    return s.cuda_stream


def _out(out, shape, device) -> torch.Tensor:
    """The caller's `out` (contiguous FP32 CUDA tensor of exactly `shape`: the kernels write all of it) or a new one."""
    if out is None:
        return torch.empty(shape, dtype=torch.float32, device=device)
    _dev(out, torch.float32, "out")
    if tuple(out.shape) != tuple(shape) or out.device != device:
        raise ValueError(f"out must be a tensor of shape {tuple(shape)} on {device}, got {tuple(out.shape)} on {out.device}")
    return out


_ws_cache: dict = {}


def _workspace(device, nbytes: int, stream=None) -> torch.Tensor:
    """One grow-only scratch buffer per (device, stream): calls issued on different streams never share scratch, and a
    buffer that is replaced by a larger one is handed back to the caching allocator only after the work queued on its
    stream has run (record_stream).  torch allocations are 512-byte aligned."""
    with torch.cuda.device(device):
        s = torch.cuda.current_stream() if stream is None else stream
        key = (device.index if device.index is not None else torch.cuda.current_device(), s.cuda_stream)
        ws = _ws_cache.get(key)
        if ws is None or ws.numel() < nbytes:
            _ws_cache.pop(key, None)
            ws = None  # drops the old buffer; its record_stream defers reuse until the stream has passed this point
            ws = torch.empty(int(nbytes), dtype=torch.uint8, device=device)
            ws.record_stream(s)
            _ws_cache[key] = ws
    return ws


def cgtp_version() -> int:
    return lib().cgtp_version()


def cgtp_max_lmax() -> int:
    return lib().cgtp_max_lmax()


def cgtp_grid_shape(lmax: int, lmax_out: int):
    U, V = ctypes.c_int(0), ctypes.c_int(0)
    _check(lib().cgtp_grid_shape(lmax, lmax_out, ctypes.byref(U), ctypes.byref(V)))
    return U.value, V.value


def cgtp_onsite_workspace_bytes(lmax, lmax_out, N, C, batch) -> int:
    return lib().cgtp_onsite_workspace_bytes(lmax, lmax_out, N, C, batch)


def cgtp_onsite(A, B, W_a, W_b, W_out, lmax, lmax_out, N, C, parity_mask, out=None, workspace=None, stream=None):
    """out[batch, 2, N, (lmax_out+1)^2] = on-site contracted CG product (see include/cgtp.h)."""
    f32 = torch.float32
    A, B = _dev(A, f32, "A"), _dev(B, f32, "B")
    W_a, W_b, W_out = _dev(W_a, f32, "W_a"), _dev(W_b, f32, "W_b"), _dev(W_out, f32, "W_out")
    batch = A.shape[0]
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    if tuple(A.shape) != (batch, N, L2) or tuple(B.shape) != (batch, N, L2):
        raise ValueError("A, B must be [batch, N, (lmax+1)^2]")
    if tuple(W_a.shape) != (C, N) or tuple(W_b.shape) != (C, N) or tuple(W_out.shape) != (N, C):
        raise ValueError("W_a, W_b must be [C, N] and W_out [N, C]")
    mask = _mask(parity_mask, C)
    out = _out(out, (batch, 2, N, Lo2), A.device)
    nbytes = cgtp_onsite_workspace_bytes(lmax, lmax_out, N, C, batch)
    ws = _workspace(A.device, nbytes, stream) if workspace is None else workspace
    with torch.cuda.device(A.device):
        rc = lib().cgtp_onsite(A.data_ptr(), B.data_ptr(), W_a.data_ptr(), W_b.data_ptr(), W_out.data_ptr(),
                               lmax, lmax_out, N, C, mask.ctypes.data, out.data_ptr(), batch,
                               ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc)
    return out


STATIC_SCRATCH_BYTES = 16 << 20


def cgtp_onsite_static(A, B, W_a, W_b, W_out, lmax, lmax_out, N, C, parity_mask, out, stream=None):
    """cgtp_onsite without any device allocation (include/cgtp.h): scratch in a 16 MiB file-scope device array, limits
    max(lmax, lmax_out) <= 4 and C <= 256.  `out` [batch, 2, N, (lmax_out+1)^2] is the caller's (this wrapper allocates
    nothing either).  All calls share the array: calls that overlap on the GPU race."""
    f32 = torch.float32
    A, B = _dev(A, f32, "A"), _dev(B, f32, "B")
    W_a, W_b, W_out = _dev(W_a, f32, "W_a"), _dev(W_b, f32, "W_b"), _dev(W_out, f32, "W_out")
    batch = A.shape[0]
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    if tuple(A.shape) != (batch, N, L2) or tuple(B.shape) != (batch, N, L2):
        raise ValueError("A, B must be [batch, N, (lmax+1)^2]")
    if tuple(W_a.shape) != (C, N) or tuple(W_b.shape) != (C, N) or tuple(W_out.shape) != (N, C):
        raise ValueError("W_a, W_b must be [C, N] and W_out [N, C]")
    mask = _mask(parity_mask, C)
    if out is None:
        raise ValueError("cgtp_onsite_static allocates nothing: pass `out`")
    out = _out(out, (batch, 2, N, Lo2), A.device)
    with torch.cuda.device(A.device):
        rc = lib().cgtp_onsite_static(A.data_ptr(), B.data_ptr(), W_a.data_ptr(), W_b.data_ptr(), W_out.data_ptr(),
                                      lmax, lmax_out, N, C, mask.ctypes.data, out.data_ptr(), batch, _stream_ptr(stream))
    _check(rc)
    return out


def cgtp_grid_shape_nu(lmax: int, lmax_out: int, nu: int):
    U, V = ctypes.c_int(0), ctypes.c_int(0)
    _check(lib().cgtp_grid_shape_nu(lmax, lmax_out, nu, ctypes.byref(U), ctypes.byref(V)))
    return U.value, V.value


def cgtp_onsite_nbody_workspace_bytes(nu, lmax, lmax_out, N, C, batch) -> int:
    return lib().cgtp_onsite_nbody_workspace_bytes(nu, lmax, lmax_out, N, C, batch)


def cgtp_onsite_nbody(X, W_in, W_out, nu, lmax, lmax_out, N, C, out=None, workspace=None, stream=None):
    """out[batch, N, (lmax_out+1)^2] = nu-body pointwise product of X[nu, batch, N, (lmax+1)^2] (see include/cgtp.h)."""
    f32 = torch.float32
    X, W_in, W_out = _dev(X, f32, "X"), _dev(W_in, f32, "W_in"), _dev(W_out, f32, "W_out")
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    if X.dim() != 4 or X.shape[0] != nu or X.shape[2] != N or X.shape[3] != L2:
        raise ValueError("X must be [nu, batch, N, (lmax+1)^2]")
    batch = X.shape[1]
    if tuple(W_in.shape) != (nu, C, N) or tuple(W_out.shape) != (N, C):
        raise ValueError("W_in must be [nu, C, N] and W_out [N, C]")
    out = _out(out, (batch, N, Lo2), X.device)
    nbytes = cgtp_onsite_nbody_workspace_bytes(nu, lmax, lmax_out, N, C, batch)
    ws = _workspace(X.device, nbytes, stream) if workspace is None else workspace
    with torch.cuda.device(X.device):
        rc = lib().cgtp_onsite_nbody(X.data_ptr(), W_in.data_ptr(), W_out.data_ptr(), nu, lmax, lmax_out, N, C,
                                     out.data_ptr(), batch, ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc)
    return out


def cgtp_message_workspace_bytes(lmax, lmax_out, N, C, parity_mask, nodes, E) -> int:
    mask = _mask(parity_mask, C)
    return lib().cgtp_message_workspace_bytes(lmax, lmax_out, N, C, mask.ctypes.data, nodes, E)


def cgtp_message(node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, N, C, parity_mask,
                 out=None, workspace=None, stream=None, check: bool = False):
    """out[nodes, 2, N, (lmax_out+1)^2] = parity-aware message passing (see include/cgtp.h).
    check=True synchronises and raises CgtpError(ERR_GRAPH) for an unsorted / out-of-range edge list."""
    f32 = torch.float32
    X = _dev(node_feats, f32, "node_feats")
    ei = _dev(edge_index, torch.int64, "edge_index")
    ev, er = _dev(edge_vec, f32, "edge_vec"), _dev(edge_radial, f32, "edge_radial")
    W_node, W_out = _dev(W_node, f32, "W_node"), _dev(W_out, f32, "W_out")
    nodes, E = X.shape[0], ei.shape[1]
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    if tuple(X.shape) != (nodes, N, L2):
        raise ValueError("node_feats must be [nodes, N, (lmax+1)^2]")
    if tuple(ei.shape) != (2, E) or tuple(ev.shape) != (E, 3) or tuple(er.shape) != (E, C):
        raise ValueError("edge_index [2,E], edge_vec [E,3], edge_radial [E,C] expected")
    if tuple(W_node.shape) != (C, N) or tuple(W_out.shape) != (N, C):
        raise ValueError("W_node must be [C, N] and W_out [N, C]")
    mask = _mask(parity_mask, C)
    out = _out(out, (nodes, 2, N, Lo2), X.device)
    nbytes = lib().cgtp_message_workspace_bytes(lmax, lmax_out, N, C, mask.ctypes.data, nodes, E)
    ws = _workspace(X.device, nbytes, stream) if workspace is None else workspace
    sp = _stream_ptr(stream)
    with torch.cuda.device(X.device):
        rc = lib().cgtp_message(X.data_ptr(), ei.data_ptr(), ev.data_ptr(), er.data_ptr(), W_node.data_ptr(),
                                W_out.data_ptr(), lmax, lmax_out, N, C, mask.ctypes.data, out.data_ptr(), nodes, E,
                                ws.data_ptr(), ws.numel(), sp)
        _check(rc)
        if check:
            _check(lib().cgtp_message_status(ws.data_ptr(), sp))
    return out


def cgtp_message_field_workspace_bytes(lmax, lmax_out, N, Ne, C, nodes, E) -> int:
    return lib().cgtp_message_field_workspace_bytes(lmax, lmax_out, N, Ne, C, nodes, E)


def cgtp_message_field_lw(node_feats, edge_index, edge_feats, W_edge, W_node, W_out, lmax, lmax_out, N, Ne, C,
                          parity_mask, out=None, workspace=None, stream=None, check: bool = False):
    """cgtp_message_field with l-dependent weights W_edge [lmax+1,C,Ne], W_node [lmax+1,C,N], W_out [lmax_out+1,N,C]."""
    return cgtp_message_field(node_feats, edge_index, edge_feats, W_edge, W_node, W_out, lmax, lmax_out, N, Ne, C,
                              parity_mask, out=out, workspace=workspace, stream=stream, check=check, _lw=True)


def cgtp_message_field(node_feats, edge_index, edge_feats, W_edge, W_node, W_out, lmax, lmax_out, N, Ne, C,
                       parity_mask, out=None, workspace=None, stream=None, check: bool = False, _lw: bool = False):
    """out[nodes, 2, N, (lmax_out+1)^2] = two-field coupling Eq.(28) (edge feature field x sender feature; see
    include/cgtp.h).  check=True synchronises and raises CgtpError(ERR_GRAPH) for an invalid edge list."""
    f32 = torch.float32
    X, XE = _dev(node_feats, f32, "node_feats"), _dev(edge_feats, f32, "edge_feats")
    ei = _dev(edge_index, torch.int64, "edge_index")
    W_edge, W_node, W_out = _dev(W_edge, f32, "W_edge"), _dev(W_node, f32, "W_node"), _dev(W_out, f32, "W_out")
    nodes, E = X.shape[0], ei.shape[1]
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    if tuple(X.shape) != (nodes, N, L2) or tuple(XE.shape) != (E, Ne, L2) or tuple(ei.shape) != (2, E):
        raise ValueError("node_feats [nodes,N,(lmax+1)^2], edge_feats [E,Ne,(lmax+1)^2], edge_index [2,E] expected")
    pre_in, pre_out = ((lmax + 1,), (lmax_out + 1,)) if _lw else ((), ())
    if (tuple(W_edge.shape) != pre_in + (C, Ne) or tuple(W_node.shape) != pre_in + (C, N)
            or tuple(W_out.shape) != pre_out + (N, C)):
        raise ValueError("W_edge must be [C, Ne], W_node [C, N] and W_out [N, C] (with a leading degree axis for _lw)")
    mask = _mask(parity_mask, C)
    out = _out(out, (nodes, 2, N, Lo2), X.device)
    nbytes = cgtp_message_field_workspace_bytes(lmax, lmax_out, N, Ne, C, nodes, E)
    ws = _workspace(X.device, nbytes, stream) if workspace is None else workspace
    sp = _stream_ptr(stream)
    with torch.cuda.device(X.device):
        entry = lib().cgtp_message_field_lw if _lw else lib().cgtp_message_field
        rc = entry(X.data_ptr(), ei.data_ptr(), XE.data_ptr(), W_edge.data_ptr(), W_node.data_ptr(),
                                      W_out.data_ptr(), lmax, lmax_out, N, Ne, C, mask.ctypes.data, out.data_ptr(),
                                      nodes, E, ws.data_ptr(), ws.numel(), sp)
        _check(rc)
        if check:
            _check(lib().cgtp_message_status(ws.data_ptr(), sp))
    return out


def cgtp_message_field_parity(node_feats, edge_index, edge_feats, W_edge, W_node, W_out, lmax, lmax_out, N, Ne, C, out=None,
                              workspace=None, stream=None, check: bool = False):
    """out[nodes, 2, N, (lmax_out+1)^2] = two parity-bearing fields, Eq.(28) with slot axes: node_feats [nodes,2,N,L2],
    edge_feats [E,2,Ne,L2], W_edge [16,C,Ne], W_node [16,C,N], W_out [16,N,C] (see include/cgtp.h)."""
    f32 = torch.float32
    X, XE = _dev(node_feats, f32, "node_feats"), _dev(edge_feats, f32, "edge_feats")
    ei = _dev(edge_index, torch.int64, "edge_index")
    W_edge, W_node, W_out = _dev(W_edge, f32, "W_edge"), _dev(W_node, f32, "W_node"), _dev(W_out, f32, "W_out")
    nodes, E = X.shape[0], ei.shape[1]
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    if tuple(X.shape) != (nodes, 2, N, L2) or tuple(XE.shape) != (E, 2, Ne, L2) or tuple(ei.shape) != (2, E):
        raise ValueError("node_feats [nodes,2,N,(lmax+1)^2], edge_feats [E,2,Ne,(lmax+1)^2], edge_index [2,E] expected")
    if tuple(W_edge.shape) != (16, C, Ne) or tuple(W_node.shape) != (16, C, N) or tuple(W_out.shape) != (16, N, C):
        raise ValueError("W_edge must be [16, C, Ne], W_node [16, C, N] and W_out [16, N, C]")
    out = _out(out, (nodes, 2, N, Lo2), X.device)
    nbytes = lib().cgtp_message_field_parity_workspace_bytes(lmax, lmax_out, N, Ne, C, nodes, E)
    ws = _workspace(X.device, nbytes, stream) if workspace is None else workspace
    sp = _stream_ptr(stream)
    with torch.cuda.device(X.device):
        rc = lib().cgtp_message_field_parity(X.data_ptr(), ei.data_ptr(), XE.data_ptr(), W_edge.data_ptr(), W_node.data_ptr(),
                                             W_out.data_ptr(), lmax, lmax_out, N, Ne, C, out.data_ptr(), nodes, E,
                                             ws.data_ptr(), ws.numel(), sp)
        _check(rc)
        if check:
            _check(lib().cgtp_message_status(ws.data_ptr(), sp))
    return out


def cgtp_message_field_bipartite(node_feats, edge_index, edge_feats, W_edge, W_node, W_out, lmax, lmax_out, N, Ne, C,
                                 parity_mask, n_recv, out=None, workspace=None, stream=None, check: bool = False):
    """out[n_recv, 2, N, (lmax_out+1)^2]: cgtp_message_field for one receiver shard -- senders index node_feats
    [n_send, N, L2] (all nodes), receivers are the local rows 0 .. n_recv-1 (see include/cgtp.h)."""
    f32 = torch.float32
    X, XE = _dev(node_feats, f32, "node_feats"), _dev(edge_feats, f32, "edge_feats")
    ei = _dev(edge_index, torch.int64, "edge_index")
    W_edge, W_node, W_out = _dev(W_edge, f32, "W_edge"), _dev(W_node, f32, "W_node"), _dev(W_out, f32, "W_out")
    n_send, E = X.shape[0], ei.shape[1]
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    if tuple(X.shape) != (n_send, N, L2) or tuple(XE.shape) != (E, Ne, L2) or tuple(ei.shape) != (2, E):
        raise ValueError("node_feats [n_send,N,(lmax+1)^2], edge_feats [E,Ne,(lmax+1)^2], edge_index [2,E] expected")
    if tuple(W_edge.shape) != (C, Ne) or tuple(W_node.shape) != (C, N) or tuple(W_out.shape) != (N, C):
        raise ValueError("W_edge must be [C, Ne], W_node [C, N] and W_out [N, C]")
    mask = _mask(parity_mask, C)
    out = _out(out, (n_recv, 2, N, Lo2), X.device)
    nbytes = lib().cgtp_message_field_bipartite_workspace_bytes(lmax, lmax_out, N, Ne, C, n_send, n_recv, E)
    ws = _workspace(X.device, nbytes, stream) if workspace is None else workspace
    sp = _stream_ptr(stream)
    with torch.cuda.device(X.device):
        rc = lib().cgtp_message_field_bipartite(X.data_ptr(), ei.data_ptr(), XE.data_ptr(), W_edge.data_ptr(),
                                                W_node.data_ptr(), W_out.data_ptr(), lmax, lmax_out, N, Ne, C,
                                                mask.ctypes.data, out.data_ptr(), n_send, n_recv, E, ws.data_ptr(),
                                                ws.numel(), sp)
        _check(rc)
        if check:
            _check(lib().cgtp_message_status(ws.data_ptr(), sp))
    return out


def cgtp_message_bipartite(node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, N, C,
                           parity_mask, n_recv: int, out=None, workspace=None, stream=None, check: bool = False):
    """out[n_recv, 2, N, (lmax_out+1)^2]: message passing onto n_recv receivers from the n_send =
    node_feats.shape[0] sender nodes (see include/cgtp.h); receivers in edge_index are local, in [0, n_recv)."""
    f32 = torch.float32
    X = _dev(node_feats, f32, "node_feats")
    ei = _dev(edge_index, torch.int64, "edge_index")
    ev, er = _dev(edge_vec, f32, "edge_vec"), _dev(edge_radial, f32, "edge_radial")
    W_node, W_out = _dev(W_node, f32, "W_node"), _dev(W_out, f32, "W_out")
    n_send, E = X.shape[0], ei.shape[1]
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    if tuple(X.shape) != (n_send, N, L2):
        raise ValueError("node_feats must be [n_send, N, (lmax+1)^2]")
    if tuple(ei.shape) != (2, E) or tuple(ev.shape) != (E, 3) or tuple(er.shape) != (E, C):
        raise ValueError("edge_index [2,E], edge_vec [E,3], edge_radial [E,C] expected")
    if tuple(W_node.shape) != (C, N) or tuple(W_out.shape) != (N, C):
        raise ValueError("W_node must be [C, N] and W_out [N, C]")
    mask = _mask(parity_mask, C)
    out = _out(out, (n_recv, 2, N, Lo2), X.device)
    nbytes = lib().cgtp_message_bipartite_workspace_bytes(lmax, lmax_out, N, C, mask.ctypes.data, n_send, n_recv, E)
    ws = _workspace(X.device, nbytes, stream) if workspace is None else workspace
    sp = _stream_ptr(stream)
    with torch.cuda.device(X.device):
        rc = lib().cgtp_message_bipartite(X.data_ptr(), ei.data_ptr(), ev.data_ptr(), er.data_ptr(), W_node.data_ptr(),
                                          W_out.data_ptr(), lmax, lmax_out, N, C, mask.ctypes.data, out.data_ptr(),
                                          n_send, n_recv, E, ws.data_ptr(), ws.numel(), sp)
        _check(rc)
        if check:
            _check(lib().cgtp_message_status(ws.data_ptr(), sp))
    return out


def cgtp_onsite_parity(A, B, W_a, W_b, W_out, lmax, lmax_out, N, C, out=None, workspace=None, stream=None):
    """out[batch, 2, N, (lmax_out+1)^2] = on-site contraction of parity-labelled inputs A, B [batch, 2, N, (lmax+1)^2]
    with the 16 weight sets W_a, W_b [16, C, N], W_out [16, N, C] (see include/cgtp.h)."""
    f32 = torch.float32
    A, B = _dev(A, f32, "A"), _dev(B, f32, "B")
    W_a, W_b, W_out = _dev(W_a, f32, "W_a"), _dev(W_b, f32, "W_b"), _dev(W_out, f32, "W_out")
    batch = A.shape[0]
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    if tuple(A.shape) != (batch, 2, N, L2) or tuple(B.shape) != (batch, 2, N, L2):
        raise ValueError("A, B must be [batch, 2, N, (lmax+1)^2]")
    if tuple(W_a.shape) != (16, C, N) or tuple(W_b.shape) != (16, C, N) or tuple(W_out.shape) != (16, N, C):
        raise ValueError("W_a, W_b must be [16, C, N] and W_out [16, N, C]")
    out = _out(out, (batch, 2, N, Lo2), A.device)
    nbytes = lib().cgtp_onsite_parity_workspace_bytes(lmax, lmax_out, N, C, batch)
    ws = _workspace(A.device, nbytes, stream) if workspace is None else workspace
    with torch.cuda.device(A.device):
        rc = lib().cgtp_onsite_parity(A.data_ptr(), B.data_ptr(), W_a.data_ptr(), W_b.data_ptr(), W_out.data_ptr(),
                                      lmax, lmax_out, N, C, out.data_ptr(), batch, ws.data_ptr(), ws.numel(),
                                      _stream_ptr(stream))
    _check(rc)
    return out


def cgtp_message_parity(node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, N, C,
                        out=None, workspace=None, stream=None, check: bool = False):
    """out[nodes, 2, N, (lmax_out+1)^2] = message passing with parity-labelled node features [nodes, 2, N, (lmax+1)^2],
    edge_radial [E, 8, C], W_node [8, C, N], W_out [8, N, C] (see include/cgtp.h)."""
    f32 = torch.float32
    X = _dev(node_feats, f32, "node_feats")
    ei = _dev(edge_index, torch.int64, "edge_index")
    ev, er = _dev(edge_vec, f32, "edge_vec"), _dev(edge_radial, f32, "edge_radial")
    W_node, W_out = _dev(W_node, f32, "W_node"), _dev(W_out, f32, "W_out")
    nodes, E = X.shape[0], ei.shape[1]
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    if tuple(X.shape) != (nodes, 2, N, L2):
        raise ValueError("node_feats must be [nodes, 2, N, (lmax+1)^2]")
    if tuple(ei.shape) != (2, E) or tuple(ev.shape) != (E, 3) or tuple(er.shape) != (E, 8, C):
        raise ValueError("edge_index [2,E], edge_vec [E,3], edge_radial [E,8,C] expected")
    if tuple(W_node.shape) != (8, C, N) or tuple(W_out.shape) != (8, N, C):
        raise ValueError("W_node must be [8, C, N] and W_out [8, N, C]")
    out = _out(out, (nodes, 2, N, Lo2), X.device)
    nbytes = lib().cgtp_message_parity_workspace_bytes(lmax, lmax_out, N, C, nodes, E)
    ws = _workspace(X.device, nbytes, stream) if workspace is None else workspace
    sp = _stream_ptr(stream)
    with torch.cuda.device(X.device):
        rc = lib().cgtp_message_parity(X.data_ptr(), ei.data_ptr(), ev.data_ptr(), er.data_ptr(), W_node.data_ptr(),
                                       W_out.data_ptr(), lmax, lmax_out, N, C, out.data_ptr(), nodes, E,
                                       ws.data_ptr(), ws.numel(), sp)
        _check(rc)
        if check:
            _check(lib().cgtp_message_status(ws.data_ptr(), sp))
    return out


def cgtp_onsite_lw(A, B, W_a, W_b, W_out, lmax, lmax_out, N, C, parity_mask, out=None, workspace=None, stream=None):
    """cgtp_onsite with l-dependent CP weights: W_a, W_b [lmax+1, C, N], W_out [lmax_out+1, N, C] (see include/cgtp.h)."""
    f32 = torch.float32
    A, B = _dev(A, f32, "A"), _dev(B, f32, "B")
    W_a, W_b, W_out = _dev(W_a, f32, "W_a"), _dev(W_b, f32, "W_b"), _dev(W_out, f32, "W_out")
    batch = A.shape[0]
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    if tuple(A.shape) != (batch, N, L2) or tuple(B.shape) != (batch, N, L2):
        raise ValueError("A, B must be [batch, N, (lmax+1)^2]")
    if tuple(W_a.shape) != (lmax + 1, C, N) or tuple(W_b.shape) != (lmax + 1, C, N) or tuple(W_out.shape) != (lmax_out + 1, N, C):
        raise ValueError("W_a, W_b must be [lmax+1, C, N] and W_out [lmax_out+1, N, C]")
    mask = _mask(parity_mask, C)
    out = _out(out, (batch, 2, N, Lo2), A.device)
    nbytes = cgtp_onsite_workspace_bytes(lmax, lmax_out, N, C, batch)
    ws = _workspace(A.device, nbytes, stream) if workspace is None else workspace
    with torch.cuda.device(A.device):
        rc = lib().cgtp_onsite_lw(A.data_ptr(), B.data_ptr(), W_a.data_ptr(), W_b.data_ptr(), W_out.data_ptr(),
                                  lmax, lmax_out, N, C, mask.ctypes.data, out.data_ptr(), batch,
                                  ws.data_ptr(), ws.numel(), _stream_ptr(stream))
    _check(rc)
    return out


def cgtp_message_lw(node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, N, C, parity_mask,
                    out=None, workspace=None, stream=None, check: bool = False, radial_l1: bool = False):
    """cgtp_message with l-dependent weights: W_node [lmax+1, C, N], W_out [lmax_out+1, N, C]; radial_l1=True calls
    cgtp_message_lwr: edge_radial [E, C, lmax+1], the l1-dependent radial factor (see include/cgtp.h)."""
    f32 = torch.float32
    X = _dev(node_feats, f32, "node_feats")
    ei = _dev(edge_index, torch.int64, "edge_index")
    ev, er = _dev(edge_vec, f32, "edge_vec"), _dev(edge_radial, f32, "edge_radial")
    W_node, W_out = _dev(W_node, f32, "W_node"), _dev(W_out, f32, "W_out")
    nodes, E = X.shape[0], ei.shape[1]
    L2, Lo2 = (lmax + 1) ** 2, (lmax_out + 1) ** 2
    if tuple(X.shape) != (nodes, N, L2):
        raise ValueError("node_feats must be [nodes, N, (lmax+1)^2]")
    if tuple(ei.shape) != (2, E) or tuple(ev.shape) != (E, 3) or tuple(er.shape) != ((E, C, lmax + 1) if radial_l1 else (E, C)):
        raise ValueError("edge_index [2,E], edge_vec [E,3], edge_radial [E,C] ([E,C,lmax+1] with radial_l1) expected")
    if tuple(W_node.shape) != (lmax + 1, C, N) or tuple(W_out.shape) != (lmax_out + 1, N, C):
        raise ValueError("W_node must be [lmax+1, C, N] and W_out [lmax_out+1, N, C]")
    mask = _mask(parity_mask, C)
    out = _out(out, (nodes, 2, N, Lo2), X.device)
    nbytes = lib().cgtp_message_workspace_bytes(lmax, lmax_out, N, C, mask.ctypes.data, nodes, E)
    ws = _workspace(X.device, nbytes, stream) if workspace is None else workspace
    sp = _stream_ptr(stream)
    with torch.cuda.device(X.device):
        fn = lib().cgtp_message_lwr if radial_l1 else lib().cgtp_message_lw
        rc = fn(X.data_ptr(), ei.data_ptr(), ev.data_ptr(), er.data_ptr(), W_node.data_ptr(),
                W_out.data_ptr(), lmax, lmax_out, N, C, mask.ctypes.data, out.data_ptr(), nodes, E,
                ws.data_ptr(), ws.numel(), sp)
        _check(rc)
        if check:
            _check(lib().cgtp_message_status(ws.data_ptr(), sp))
    return out


def cgtp_message_lwr(node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, N, C, parity_mask,
                     out=None, workspace=None, stream=None, check: bool = False):
    """Message passing with l-dependent weights and the l1-dependent radial factor edge_radial [E, C, lmax+1]."""
    return cgtp_message_lw(node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, N, C, parity_mask,
                           out=out, workspace=workspace, stream=stream, check=check, radial_l1=True)


def cgtp_message_status(workspace=None, device=None, stream=None) -> int:
    """Graph status word of the last message-passing call that used `workspace` (default: the binding's own scratch
    buffer of (device, stream)); synchronises the stream."""
    if workspace is None:
        device = torch.device("cuda", torch.cuda.current_device()) if device is None else device
        with torch.cuda.device(device):
            s = torch.cuda.current_stream() if stream is None else stream
            workspace = _ws_cache[(device.index, s.cuda_stream)]
            return lib().cgtp_message_status(workspace.data_ptr(), s.cuda_stream)
    return lib().cgtp_message_status(workspace.data_ptr(), _stream_ptr(stream))


def cgtp_build_segments(edge_index, nodes: int, stream=None):
    """Returns (row_ptr int64 [nodes+1], status int32 [1]) on the device of edge_index."""
    ei = _dev(edge_index, torch.int64, "edge_index")
    E = ei.shape[1]
    row_ptr = torch.empty(nodes + 1, dtype=torch.int64, device=ei.device)
    status = torch.empty(1, dtype=torch.int32, device=ei.device)
    with torch.cuda.device(ei.device):
        _check(lib().cgtp_build_segments(ei.data_ptr(), E, nodes, row_ptr.data_ptr(), status.data_ptr(),
                                         _stream_ptr(stream)))
    return row_ptr, status


def _host(t, dtype, name):
    if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name} must be a contiguous CPU tensor of {dtype}")
    return t


def cgtp_onsite_host(A, B, W_a, W_b, W_out, lmax, lmax_out, N, C, parity_mask, out=None, stream=None):
    """Host-buffer entry point (pinned CPU tensors recommended); returns a CPU tensor."""
    f32 = torch.float32
    A, B = _host(A, f32, "A"), _host(B, f32, "B")
    W_a, W_b, W_out = _host(W_a, f32, "W_a"), _host(W_b, f32, "W_b"), _host(W_out, f32, "W_out")
    batch = A.shape[0]
    mask = _mask(parity_mask, C)
    if out is None:
        out = torch.empty((batch, 2, N, (lmax_out + 1) ** 2), dtype=f32, pin_memory=True)
    rc = lib().cgtp_onsite_host(A.data_ptr(), B.data_ptr(), W_a.data_ptr(), W_b.data_ptr(), W_out.data_ptr(),
                                lmax, lmax_out, N, C, mask.ctypes.data, out.data_ptr(), batch, _stream_ptr(stream))
    _check(rc)
    return out


def cgtp_message_host(node_feats, edge_index, edge_vec, edge_radial, W_node, W_out, lmax, lmax_out, N, C,
                      parity_mask, out=None, stream=None):
    f32 = torch.float32
    X = _host(node_feats, f32, "node_feats")
    ei = _host(edge_index, torch.int64, "edge_index")
    ev, er = _host(edge_vec, f32, "edge_vec"), _host(edge_radial, f32, "edge_radial")
    W_node, W_out = _host(W_node, f32, "W_node"), _host(W_out, f32, "W_out")
    nodes, E = X.shape[0], ei.shape[1]
    mask = _mask(parity_mask, C)
    if out is None:
        out = torch.empty((nodes, 2, N, (lmax_out + 1) ** 2), dtype=f32, pin_memory=True)
    rc = lib().cgtp_message_host(X.data_ptr(), ei.data_ptr(), ev.data_ptr(), er.data_ptr(), W_node.data_ptr(),
                                 W_out.data_ptr(), lmax, lmax_out, N, C, mask.ctypes.data, out.data_ptr(), nodes, E,
                                 _stream_ptr(stream))
    _check(rc)
    return out


MATH_FP32, MATH_3XTF32, MATH_TF32 = 0, 1, 2
PATH_GENERIC_CORE, PATH_GENERIC_EDGE, PATH_GENERIC_PROJ, PATH_GENERIC_SYNTH, PATH_UNFUSED_ONSITE = 1, 2, 4, 8, 16
PATH_FUSED_ONSITE = 32
PATH_FIELD_PER_EDGE = 64
PATH_SMEM_CORE = 128
PATH_PLAIN_LAUNCH = 256


def cgtp_set_kernel_path(flags: int) -> None:
    """Test switch: force the generic kernel of a stage (PATH_* bits, include/cgtp.h); 0 = the specialised kernels."""
    _check(lib().cgtp_set_kernel_path(int(flags)))


def cgtp_get_kernel_path() -> int:
    return lib().cgtp_get_kernel_path()


def cgtp_fma_peak(packed: bool, ms_target: float = 20.0, stream=None):
    """(TFLOP/s, equivalent SM MHz) of the register-only FFMA (packed=False) / FFMA2 (packed=True) micro-kernel."""
    tf, mhz = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(lib().cgtp_fma_peak(int(bool(packed)), float(ms_target), ctypes.byref(tf), ctypes.byref(mhz),
                               _stream_ptr(stream)))
    return tf.value, mhz.value


def cgtp_set_math_mode(mode: int) -> None:
    """Arithmetic of the channel projections: MATH_FP32 (default), MATH_3XTF32 or MATH_TF32 (tcgen05)."""
    _check(lib().cgtp_set_math_mode(int(mode)))


def cgtp_get_math_mode() -> int:
    return lib().cgtp_get_math_mode()


def cgtp_launch_count() -> int:
    return lib().cgtp_launch_count()


def cgtp_profile_enable(on: bool) -> None:
    _check(lib().cgtp_profile_enable(int(on)))


def cgtp_profile_collect() -> dict:
    """{kind name: (milliseconds, launches)} accumulated since the last collect."""
    n = lib().cgtp_profile_kinds()
    ms = (ctypes.c_double * n)()
    cnt = (ctypes.c_int64 * n)()
    _check(lib().cgtp_profile_collect(ms, cnt))
    return {lib().cgtp_profile_kind_name(k).decode(): (ms[k], cnt[k]) for k in range(n) if cnt[k]}

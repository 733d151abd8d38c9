"""Race / out-of-bounds evidence without compute-sanitizer (the tool is closed on this GPU pool; the refusal is kept in
profiles/r02_sanitizer.md): every kernel family with mbarriers, TMA rings or named barriers is run repeatedly on identical
inputs -- a race between a bulk copy and a generic read, or between warp groups, shows up as a run that differs bit for bit --
with `out` and the workspace cut out of larger buffers whose guard bands must stay untouched (a stray store outside either
is caught), and with unrelated work on a second stream to perturb the timing."""
import numpy as np
import pytest
import torch

from paper_2605_15073_b200 import binding as cg
from paper_2605_15073_b200 import synthetic
from tests.parity_util import cuda

pytestmark = pytest.mark.gpu

GUARD = 4096          # bytes on each side
PATTERN = 0x5A


class Guarded:
    """A device buffer of `nbytes` bytes (256-byte aligned start) between two guard bands."""

    def __init__(self, nbytes):
        self.raw = torch.full((nbytes + 2 * GUARD + 512,), PATTERN, dtype=torch.uint8, device="cuda")
        off = GUARD + (-(self.raw.data_ptr() + GUARD)) % 256
        self.off, self.nbytes = off, nbytes
        self.view = self.raw[off: off + nbytes]

    def intact(self):
        lo, hi = self.raw[: self.off], self.raw[self.off + self.nbytes:]
        return bool((lo == PATTERN).all().item() and (hi == PATTERN).all().item())


def _stress(call, out_shape, ws_bytes, reps=12):
    nout = int(np.prod(out_shape)) * 4
    g_out, g_ws = Guarded(nout), Guarded(int(ws_bytes))
    out = g_out.view.view(torch.float32).view(out_shape)
    side = torch.cuda.Stream()
    noise = torch.empty(1 << 24, device="cuda")
    first = None
    for r in range(reps):
        out.fill_(float("nan"))
        if r % 2:
            with torch.cuda.stream(side):  # unrelated traffic on another stream: perturbs scheduling and L2
                noise.normal_()
        call(out, g_ws.view)
        torch.cuda.synchronize()
        assert torch.isfinite(out).all(), f"run {r}: output not fully written"
        assert g_out.intact() and g_ws.intact(), f"run {r}: store outside out / workspace"
        if first is None:
            first = out.clone()
        else:
            assert torch.equal(first, out), f"run {r} differs bit for bit from run 0"
    return first


@pytest.fixture(autouse=True)
def defaults_after():
    yield
    cg.cgtp_set_kernel_path(0)
    cg.cgtp_set_math_mode(cg.MATH_FP32)


@pytest.mark.parametrize("name,lmax,N,C,batch,path,mode", [
    ("fused_roomy", 2, 8, 8, 203, cg.PATH_FUSED_ONSITE, 0),
    ("fused_tight", 6, 64, 64, 333, 0, 0),
    ("fused_mid", 4, 32, 32, 1001, cg.PATH_FUSED_ONSITE, 0),
    ("proj_fast+onsite_fast", 6, 64, 64, 333, cg.PATH_UNFUSED_ONSITE | cg.PATH_SMEM_CORE, 0),
    ("proj_fast+onsite_reg", 6, 64, 64, 333, cg.PATH_UNFUSED_ONSITE, 0),
    ("onsite_reg_lb4", 4, 32, 32, 1001, cg.PATH_UNFUSED_ONSITE, 0),
    ("onsite_reg_lb2", 2, 8, 24, 517, cg.PATH_UNFUSED_ONSITE, 0),
    ("onsite_fast_rowblocks", 12, 8, 8, 75, cg.PATH_UNFUSED_ONSITE, 0),
    ("generic", 5, 12, 20, 99, cg.PATH_UNFUSED_ONSITE | cg.PATH_GENERIC_CORE | cg.PATH_GENERIC_PROJ, 0),
    ("proj_tc_3xtf32", 4, 24, 40, 170, cg.PATH_UNFUSED_ONSITE, cg.MATH_3XTF32),
])
def test_onsite_families_repeatable_and_in_bounds(name, lmax, N, C, batch, path, mode):
    inp = synthetic.make_onsite(lmax, lmax, N, C, batch, seed=41)
    T = [cuda(x) for x in (inp.A, inp.B, inp.W_a, inp.W_b, inp.W_out)]
    cg.cgtp_set_kernel_path(path)
    cg.cgtp_set_math_mode(mode)
    ws = cg.cgtp_onsite_workspace_bytes(lmax, lmax, N, C, batch)
    _stress(lambda out, w: cg.cgtp_onsite(*T, lmax, lmax, N, C, inp.parity_mask, out=out, workspace=w),
            (batch, 2, N, (lmax + 1) ** 2), ws)


@pytest.mark.parametrize("name,lmax,N,C,nodes,path", [
    ("edge_ring_small", 4, 8, 16, 97, 0),
    ("edge_ring_lb8", 8, 16, 32, 61, 0),
    ("generic_edge_synth", 6, 8, 16, 55, cg.PATH_GENERIC_EDGE | cg.PATH_GENERIC_SYNTH),
])
def test_message_families_repeatable_and_in_bounds(name, lmax, N, C, nodes, path):
    deg = np.random.default_rng(lmax).integers(0, 40, nodes)
    deg[0] = 0
    m = synthetic.make_message(lmax, lmax, N, C, nodes, deg, seed=43)
    T = [cuda(x) for x in (m.node_feats, m.edge_index, m.edge_vec, m.edge_radial, m.W_node, m.W_out)]
    cg.cgtp_set_kernel_path(path)
    ws = cg.cgtp_message_workspace_bytes(lmax, lmax, N, C, m.parity_mask, nodes, m.E)
    _stress(lambda out, w: cg.cgtp_message(*T, lmax, lmax, N, C, m.parity_mask, out=out, workspace=w),
            (nodes, 2, N, (lmax + 1) ** 2), ws)


def test_edge_lr_nbody_and_field_families_repeatable_and_in_bounds():
    lmax, N, C, nodes = 4, 8, 8, 40
    m = synthetic.make_message(lmax, lmax, N, C, nodes, np.random.default_rng(2).integers(0, 15, nodes), seed=45)
    (Wn,), Wo = synthetic.lw_weights(lmax, lmax, N, C, seed=45, n_in=1)
    rad = np.ascontiguousarray(np.repeat(m.edge_radial[:, :, None], lmax + 1, axis=2))
    T = [cuda(x) for x in (m.node_feats, m.edge_index, m.edge_vec, rad, Wn, Wo)]
    ws = cg.cgtp_message_workspace_bytes(lmax, lmax, N, C, m.parity_mask, nodes, m.E)
    _stress(lambda out, w: cg.cgtp_message_lwr(*T, lmax, lmax, N, C, m.parity_mask, out=out, workspace=w),
            (nodes, 2, N, (lmax + 1) ** 2), ws)
    XE, We = synthetic.make_edge_field(m, 4, seed=45)
    F = [cuda(x) for x in (m.node_feats, m.edge_index, XE, We, m.W_node, m.W_out)]
    ws = cg.cgtp_message_field_workspace_bytes(lmax, lmax, N, 4, C, nodes, m.E)
    _stress(lambda out, w: cg.cgtp_message_field(*F, lmax, lmax, N, 4, C, m.parity_mask, out=out, workspace=w),
            (nodes, 2, N, (lmax + 1) ** 2), ws)
    m32 = synthetic.make_message(lmax, lmax, N, 32, nodes, np.random.default_rng(3).integers(0, 15, nodes), seed=46)
    XE, We = synthetic.make_edge_field(m32, 4, seed=46)  # 16 channels per parity: the pooled core (field_pool_core_kernel)
    F = [cuda(x) for x in (m32.node_feats, m32.edge_index, XE, We, m32.W_node, m32.W_out)]
    ws = cg.cgtp_message_field_workspace_bytes(lmax, lmax, N, 4, 32, nodes, m32.E)
    _stress(lambda out, w: cg.cgtp_message_field(*F, lmax, lmax, N, 4, 32, m32.parity_mask, out=out, workspace=w),
            (nodes, 2, N, (lmax + 1) ** 2), ws)
    nb = synthetic.make_nbody(3, 3, 3, 8, 8, 130, seed=47)
    Xn = [cuda(x) for x in (nb.X, nb.W_in, nb.W_out)]
    ws = cg.cgtp_onsite_nbody_workspace_bytes(3, 3, 3, 8, 8, 130)
    _stress(lambda out, w: cg.cgtp_onsite_nbody(*Xn, 3, 3, 3, 8, 8, out=out, workspace=w), (130, 8, 16), ws)


def test_chained_launches_across_entry_points_share_one_workspace():
    """The kernels of the on-site step, of message passing and of the nu-body product are chained by programmatic dependent
    launch: a kernel may start while its predecessor in the stream still runs and waits before its first
    access to anything a predecessor produced.  Different entry points issued back to back on one stream, all carving ONE
    workspace buffer (so the H / T / G regions of one call are rewritten by the next): a missed wait is a write-after-read or
    read-after-write race between kernels of different calls.  Every output must equal, bit for bit, the one obtained with
    plain launches (CGTP_PATH_PLAIN_LAUNCH: the same kernels in the usual stream order), over several repetitions with
    unrelated traffic on a second stream."""
    o1 = synthetic.make_onsite(6, 6, 64, 64, 600, seed=71)          # four launches, register core for the odd channels
    o2 = synthetic.make_onsite(2, 2, 32, 32, 3000, seed=72)         # short kernels: the boundaries overlap most
    deg = np.random.default_rng(7).integers(0, 24, 300)
    m = synthetic.make_message(4, 4, 16, 32, 300, deg, seed=73)
    nb = synthetic.make_nbody(3, 3, 3, 16, 16, 700, seed=74)
    To1 = [cuda(x) for x in (o1.A, o1.B, o1.W_a, o1.W_b, o1.W_out)]
    To2 = [cuda(x) for x in (o2.A, o2.B, o2.W_a, o2.W_b, o2.W_out)]
    Tm = [cuda(x) for x in (m.node_feats, m.edge_index, m.edge_vec, m.edge_radial, m.W_node, m.W_out)]
    Tn = [cuda(x) for x in (nb.X, nb.W_in, nb.W_out)]
    ws_bytes = max(cg.cgtp_onsite_workspace_bytes(6, 6, 64, 64, 600), cg.cgtp_onsite_workspace_bytes(2, 2, 32, 32, 3000),
                   cg.cgtp_message_workspace_bytes(4, 4, 16, 32, m.parity_mask, 300, m.E),
                   cg.cgtp_onsite_nbody_workspace_bytes(3, 3, 3, 16, 16, 700))
    g_ws = Guarded(int(ws_bytes))
    outs = [torch.empty((600, 2, 64, 49), device="cuda"), torch.empty((3000, 2, 32, 9), device="cuda"),
            torch.empty((300, 2, 16, 25), device="cuda"), torch.empty((700, 16, 16), device="cuda")]

    def sequence():
        for o in outs:
            o.fill_(float("nan"))
        w = g_ws.view
        cg.cgtp_onsite(*To1, 6, 6, 64, 64, o1.parity_mask, out=outs[0], workspace=w)
        cg.cgtp_message(*Tm, 4, 4, 16, 32, m.parity_mask, out=outs[2], workspace=w)
        cg.cgtp_onsite(*To2, 2, 2, 32, 32, o2.parity_mask, out=outs[1], workspace=w)
        cg.cgtp_onsite_nbody(*Tn, 3, 3, 3, 16, 16, out=outs[3], workspace=w)
        cg.cgtp_onsite(*To1, 6, 6, 64, 64, o1.parity_mask, out=outs[0], workspace=w)
        torch.cuda.synchronize()
        assert all(torch.isfinite(o).all() for o in outs)
        assert g_ws.intact()
        return [o.clone() for o in outs]

    cg.cgtp_set_kernel_path(cg.PATH_PLAIN_LAUNCH)
    ref = sequence()
    cg.cgtp_set_kernel_path(0)
    side = torch.cuda.Stream()
    noise = torch.empty(1 << 24, device="cuda")
    for r in range(8):
        if r % 2:
            with torch.cuda.stream(side):
                noise.normal_()
        got = sequence()
        for k, (a, b) in enumerate(zip(got, ref)):
            assert torch.equal(a, b), f"repetition {r}, output {k}: chained launches differ from plain launches"

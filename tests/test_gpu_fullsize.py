"""Parity and equivariance at BASELINE.json's full sizes, in the launch configuration bench.py times.

SURVEY.md 8(c): at configs[3] (lmax >= 12) and configs[4] the oracle evaluates a deterministic sample of >= 256 atoms /
>= 128 receiver segments; the rest of the batch is covered element by element by running the whole batch a second time
through the *generic* kernels of every stage (cgtp_set_kernel_path: a different mapping of the same arithmetic to the
machine -- other tiles, no TMA ring, no lane = column layout), so a wrong tile, a ring-stage race or a ragged-tail bug
in either family shows up as a disagreement somewhere in the batch, while the sampled oracle anchors both.
north_star: "all five configs ... stay equivariant to 1e-5 under random rotations" -- rotated on the device, whole batch.
"""
import numpy as np
import pytest
import torch

from oracle import cgtp_oracle as orc
from paper_2605_15073_b200 import binding as cg
from paper_2605_15073_b200 import synthetic
from tests import shref
from tests.parity_util import TOL, cuda, degree_signs, rotate_feats, sample_rows, sector_errs, sector_errs_torch

pytestmark = pytest.mark.gpu

GENERIC_ALL = cg.PATH_GENERIC_CORE | cg.PATH_GENERIC_EDGE | cg.PATH_GENERIC_PROJ | cg.PATH_GENERIC_SYNTH | cg.PATH_UNFUSED_ONSITE


@pytest.fixture(autouse=True)
def default_path_after():
    yield
    cg.cgtp_set_kernel_path(0)


def onsite_dev(inp, A, B, **kw):
    return cg.cgtp_onsite(A, B, cuda(inp.W_a), cuda(inp.W_b), cuda(inp.W_out), inp.lmax, inp.lmax_out, inp.N, inp.C,
                          inp.parity_mask, **kw)


def message_dev(m, X, ev, **kw):
    return cg.cgtp_message(X, cuda(m.edge_index), ev, cuda(m.edge_radial), cuda(m.W_node), cuda(m.W_out), m.lmax,
                           m.lmax_out, m.N, m.C, m.parity_mask, **kw)


# ------------------------------------------------------------------------------------------------ on-site
@pytest.mark.parametrize("lmax", [2, 4, 8, 12, 16, 20])
def test_onsite_config3_sweep_sampled_oracle_and_full_batch_cross_check(lmax):
    """BASELINE.json configs[3]: N = C = 32, batch = 16384.  >= 256 atoms (512 at lmax <= 4) against the oracle; every
    element of the batch against the generic kernels."""
    inp = synthetic.config(3, lmax=lmax)
    A, B = cuda(inp.A), cuda(inp.B)
    got = onsite_dev(inp, A, B).clone()
    idx = sample_rows(inp.batch, 512 if lmax <= 4 else 256, seed=lmax, extra=(31, 32, 255, 256, 8191, 8192))
    assert idx.size >= 256
    ref = orc.onsite(inp.A[idx], inp.B[idx], inp.W_a, inp.W_b, inp.W_out, inp.lmax, inp.lmax_out, inp.parity_mask)
    e = sector_errs(got[torch.from_numpy(idx).cuda()].cpu().numpy(), ref)
    assert max(e) < TOL, e
    cg.cgtp_set_kernel_path(GENERIC_ALL)
    alt = onsite_dev(inp, A, B)
    cg.cgtp_set_kernel_path(0)
    e = sector_errs_torch(got, alt)
    assert max(e) < TOL, e
    assert torch.isfinite(got).all()


@pytest.mark.parametrize("lmax", [2, 4, 8])
def test_onsite_config3_fused_kernel_whole_batch(lmax):
    """configs[3] at the band limits the single-kernel step supports, forced (the library's own choice for N = C = 32 is
    the four-launch step): every element against the default path."""
    inp = synthetic.config(3, lmax=lmax)
    A, B = cuda(inp.A), cuda(inp.B)
    got = onsite_dev(inp, A, B).clone()
    cg.cgtp_set_kernel_path(cg.PATH_FUSED_ONSITE)
    alt = onsite_dev(inp, A, B)
    e = sector_errs_torch(got, alt)
    assert max(e) < TOL, e


@pytest.mark.parametrize("lmax", [2, 4])
def test_onsite_config3_both_cores_whole_batch(lmax):
    """configs[3] at small band limits: the one-thread-per-column register core (onsite_reg.cu, the library's choice) and
    the warp-scheduled shared-memory core (onsite_core.cu, CGTP_PATH_SMEM_CORE) on the whole batch, element by element."""
    inp = synthetic.config(3, lmax=lmax)
    A, B = cuda(inp.A), cuda(inp.B)
    cg.cgtp_set_kernel_path(cg.PATH_UNFUSED_ONSITE)
    got = onsite_dev(inp, A, B).clone()
    cg.cgtp_set_kernel_path(cg.PATH_UNFUSED_ONSITE | cg.PATH_SMEM_CORE)
    alt = onsite_dev(inp, A, B)
    e = sector_errs_torch(got, alt)
    assert max(e) < TOL, e


def test_onsite_config1_every_kernel_path_agrees():
    """configs[1] (the bench workload; the oracle checks every output in test_gpu_parity.py): fused step, four-launch
    step and the generic kernels agree element by element."""
    inp = synthetic.config(1)
    A, B = cuda(inp.A), cuda(inp.B)
    got = onsite_dev(inp, A, B).clone()
    for flags in (cg.PATH_UNFUSED_ONSITE, cg.PATH_UNFUSED_ONSITE | cg.PATH_SMEM_CORE,
                  cg.PATH_UNFUSED_ONSITE | cg.PATH_GENERIC_CORE, cg.PATH_UNFUSED_ONSITE | cg.PATH_GENERIC_PROJ, GENERIC_ALL,
                  cg.PATH_PLAIN_LAUNCH):
        cg.cgtp_set_kernel_path(flags)
        assert cg.cgtp_get_kernel_path() == flags
        alt = onsite_dev(inp, A, B)
        e = sector_errs_torch(got, alt)
        assert max(e) < TOL, (flags, e)
        if flags == cg.PATH_PLAIN_LAUNCH:  # the same kernels, launched in plain stream order instead of chained
            assert torch.equal(got, alt)
    with pytest.raises(cg.CgtpError):
        cg.cgtp_set_kernel_path(1 << 10)


@pytest.mark.parametrize("cfg,lmax", [(0, None), (1, None), (3, 2), (3, 4), (3, 8), (3, 12), (3, 16), (3, 20)])
def test_onsite_equivariance_and_inversion_on_baseline_configs(cfg, lmax):
    """R15 on configs[0], [1] and every point of configs[3], whole batch on the device: rotate A, B with the real
    Wigner-D of a random rotation -> both sectors rotate with D; invert -> sector 0 picks (-1)^l, sector 1 -(-1)^l
    (App. B test 5 PAPER.md:633; Table I :86-:93)."""
    inp = synthetic.config(cfg) if lmax is None else synthetic.config(cfg, lmax=lmax)
    A, B = cuda(inp.A), cuda(inp.B)
    base = onsite_dev(inp, A, B).clone()
    R = shref.random_rotation(np.random.default_rng(1000 + cfg * 31 + inp.lmax))
    D = shref.wigner_D_real(inp.lmax, R)
    rot = onsite_dev(inp, rotate_feats(A, D), rotate_feats(B, D))
    Do = D[: (inp.lmax_out + 1) ** 2, : (inp.lmax_out + 1) ** 2]
    want = base.double() @ torch.from_numpy(Do).cuda().T
    e = sector_errs_torch(rot, want)
    assert max(e) < TOL, e
    sg = torch.from_numpy(degree_signs(inp.lmax)).cuda()
    so = sg[: (inp.lmax_out + 1) ** 2]
    inv = onsite_dev(inp, (A.double() * sg).float(), (B.double() * sg).float())
    want = torch.stack([base[:, 0].double() * so, -base[:, 1].double() * so], dim=1)
    e = sector_errs_torch(inv, want)
    assert max(e) < TOL, e


# ---------------------------------------------------------------------------------------- message passing
def test_message_config4_sampled_oracle_and_full_batch_cross_check():
    """BASELINE.json configs[4]: 16384 nodes x 32 in-edges, lmax = 8, N = C = 128, half odd channels.  >= 128 receiver
    segments against the oracle; every element against the generic kernels (direct-load edge kernel, generic node
    synthesis, SIMT projections)."""
    m = synthetic.config(4)
    X, ev = cuda(m.node_feats), cuda(m.edge_vec)
    got = message_dev(m, X, ev, check=True).clone()
    recv = sample_rows(m.nodes, 128, seed=4, extra=(147, 148, 295, 296, 8191, 8192))
    assert recv.size >= 128
    ref = orc.message(m.node_feats, m.edge_index, m.edge_vec, m.edge_radial, m.W_node, m.W_out, m.lmax, m.lmax_out,
                      m.parity_mask, recv)
    e = sector_errs(got[torch.from_numpy(recv).cuda()].cpu().numpy(), ref)
    assert max(e) < TOL, e
    cg.cgtp_set_kernel_path(GENERIC_ALL)
    alt = message_dev(m, X, ev, check=True)
    cg.cgtp_set_kernel_path(0)
    e = sector_errs_torch(got, alt)
    assert max(e) < TOL, e
    assert torch.isfinite(got).all()


def test_message_config2_every_kernel_path_agrees():
    m = synthetic.config(2)
    m.parity_mask = synthetic.half_mask(m.C)
    X, ev = cuda(m.node_feats), cuda(m.edge_vec)
    got = message_dev(m, X, ev, check=True).clone()
    for flags in (cg.PATH_GENERIC_EDGE, cg.PATH_GENERIC_SYNTH, cg.PATH_GENERIC_PROJ, GENERIC_ALL):
        cg.cgtp_set_kernel_path(flags)
        alt = message_dev(m, X, ev, check=True)
        e = sector_errs_torch(got, alt)
        assert max(e) < TOL, (flags, e)


@pytest.mark.parametrize("cfg,half", [(2, False), (2, True), (4, True)])
def test_message_equivariance_and_inversion_on_baseline_configs(cfg, half):
    """R15 on configs[2] (all-even as stated, and half odd) and configs[4], whole output on the device: node features
    rotate with D, edge vectors with R; inversion flips the edge vectors and multiplies h_lm by (-1)^l."""
    m = synthetic.config(cfg)
    if half:
        m.parity_mask = synthetic.half_mask(m.C)
    X, ev = cuda(m.node_feats), cuda(m.edge_vec)
    base = message_dev(m, X, ev).clone()
    R = shref.random_rotation(np.random.default_rng(2000 + cfg))
    D = shref.wigner_D_real(m.lmax, R)
    ev_rot = (ev.double() @ torch.from_numpy(R).cuda().T).float().contiguous()
    rot = message_dev(m, rotate_feats(X, D), ev_rot)
    Do = D[: (m.lmax_out + 1) ** 2, : (m.lmax_out + 1) ** 2]
    want = base.double() @ torch.from_numpy(Do).cuda().T
    e = sector_errs_torch(rot, want)
    assert max(e) < TOL, e
    sg = torch.from_numpy(degree_signs(m.lmax)).cuda()
    so = sg[: (m.lmax_out + 1) ** 2]
    inv = message_dev(m, (X.double() * sg).float(), (-ev).contiguous())
    want = torch.stack([base[:, 0].double() * so, -base[:, 1].double() * so], dim=1)
    e = sector_errs_torch(inv, want)
    assert max(e) < TOL, e

"""Parity of cgtp_onsite_nbody (nu-body pointwise product) against the FP64
oracle, through the C ABI.  Bar as for the bilinear path: max|out - ref| / max|ref| <= 1e-5 (FP32)."""
import numpy as np
import pytest
import torch

from oracle import cgtp_oracle as orc
from paper_2605_15073_b200 import binding as cg
from paper_2605_15073_b200 import synthetic
from tests import shref

pytestmark = pytest.mark.gpu

TOL = 1e-5


def _cuda(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_nbody(inp, **kw):
    out = cg.cgtp_onsite_nbody(_cuda(inp.X), _cuda(inp.W_in), _cuda(inp.W_out), inp.nu, inp.lmax, inp.lmax_out, inp.N,
                               inp.C, **kw)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def rel_err(got, ref):
    return np.abs(np.asarray(got, np.float64) - ref).max() / np.abs(ref).max()


# sizes span several CTAs (NC columns each) and a ragged last CTA; band limits that are / are not compiled bands (7 -> 8)
@pytest.mark.parametrize("nu,lmax,lmax_out,N,C,batch", [
    (3, 2, 2, 8, 8, 64), (3, 2, 6, 6, 5, 37), (4, 2, 2, 8, 8, 50), (4, 2, 8, 4, 6, 21), (3, 4, 4, 16, 12, 133),
    (2, 3, 5, 8, 8, 40), (1, 3, 2, 8, 4, 17), (3, 6, 6, 16, 16, 67), (4, 3, 3, 12, 10, 91), (3, 7, 7, 8, 8, 19),
    (3, 1, 3, 2, 2, 3), (4, 8, 8, 8, 4, 9), (3, 3, 0, 8, 8, 33),
    # band limits above 8 (round 2): row counts U up to 41, one CTA per SM
    (3, 12, 12, 8, 8, 21), (2, 16, 16, 4, 8, 13), (4, 10, 6, 4, 4, 9), (3, 9, 14, 4, 4, 7), (2, 20, 20, 4, 4, 6), (3, 16, 8, 4, 4, 5),
])
def test_nbody_vs_oracle(nu, lmax, lmax_out, N, C, batch):
    inp = synthetic.make_nbody(nu, lmax, lmax_out, N, C, batch, seed=1000 * nu + 10 * lmax + lmax_out)
    got = run_nbody(inp)
    ref = orc.onsite_nbody(inp.X, inp.W_in, inp.W_out, lmax, lmax_out)
    assert got.shape == ref.shape
    assert rel_err(got, ref) <= TOL, rel_err(got, ref)
    again = run_nbody(inp)
    assert np.array_equal(got, again)  # bitwise reproducible


@pytest.mark.parametrize("nu,lmax,lmax_out,N,C,batch", [
    (3, 2, 2, 8, 8, 64), (4, 2, 2, 8, 8, 50), (3, 4, 4, 16, 12, 133), (4, 3, 3, 12, 10, 91), (3, 1, 3, 2, 2, 3),
    (3, 3, 0, 8, 8, 33), (4, 1, 4, 8, 8, 70), (3, 3, 3, 32, 32, 257), (4, 4, 2, 8, 16, 45), (3, 6, 6, 16, 16, 67),
    (4, 5, 5, 8, 8, 21), (3, 2, 6, 6, 5, 37),
])
def test_nbody_register_and_shared_memory_cores(nu, lmax, lmax_out, N, C, batch):
    """nu >= 3 at band limits <= 6 runs with one thread per column on registers (nbody_reg.cu); CGTP_PATH_SMEM_CORE keeps
    the CTA-tiled kernel of nbody.cu.  Both against the oracle."""
    inp = synthetic.make_nbody(nu, lmax, lmax_out, N, C, batch, seed=500 + 100 * nu + 10 * lmax + lmax_out)
    ref = orc.onsite_nbody(inp.X, inp.W_in, inp.W_out, lmax, lmax_out)
    outs = []
    try:
        for flags in (0, cg.PATH_SMEM_CORE):
            cg.cgtp_set_kernel_path(flags)
            got = run_nbody(inp)
            assert rel_err(got, ref) <= TOL, (flags, rel_err(got, ref))
            assert np.array_equal(got, run_nbody(inp))
            outs.append(got)
    finally:
        cg.cgtp_set_kernel_path(0)
    assert not np.array_equal(outs[0], outs[1])  # two different kernels did run


@pytest.mark.parametrize("lmax,lmax_out,N,C,batch", [(3, 5, 8, 8, 40), (6, 6, 16, 16, 67), (2, 4, 8, 4, 33), (16, 16, 4, 8, 13)])
def test_nbody_nu2_both_cores_vs_oracle(lmax, lmax_out, N, C, batch):
    """nu = 2 runs on the bilinear core (the pointwise product of Eq.(38) with every channel even); under
    CGTP_PATH_GENERIC_CORE the nu-body kernel takes it.  Both against the oracle."""
    inp = synthetic.make_nbody(2, lmax, lmax_out, N, C, batch, seed=77 + lmax)
    ref = orc.onsite_nbody(inp.X, inp.W_in, inp.W_out, lmax, lmax_out)
    outs = []
    try:
        for flags in (0, cg.PATH_GENERIC_CORE):
            cg.cgtp_set_kernel_path(flags)
            got = run_nbody(inp)
            assert rel_err(got, ref) <= TOL, (flags, rel_err(got, ref))
            outs.append(got)
    finally:
        cg.cgtp_set_kernel_path(0)
    assert not np.array_equal(outs[0], outs[1])  # two different kernels did run


def test_nbody_nu2_matches_bilinear_entry_point():
    lmax, lmax_out, N, C, batch = 4, 4, 16, 16, 100
    o = synthetic.make_onsite(lmax, lmax_out, N, C, batch, seed=5, parity_mask=np.zeros(C, np.uint8))
    bil = cg.cgtp_onsite(_cuda(o.A), _cuda(o.B), _cuda(o.W_a), _cuda(o.W_b), _cuda(o.W_out), lmax, lmax_out, N, C,
                         o.parity_mask).cpu().numpy()[:, 0]
    nb = cg.cgtp_onsite_nbody(_cuda(np.stack([o.A, o.B])), _cuda(np.stack([o.W_a, o.W_b])), _cuda(o.W_out), 2, lmax,
                              lmax_out, N, C).cpu().numpy()
    assert np.abs(nb - bil).max() <= 2e-6 * np.abs(bil).max()


def test_nbody_rotation_equivariance_on_device():
    nu, lmax, lmax_out, N, C, batch = 3, 3, 5, 6, 8, 24
    inp = synthetic.make_nbody(nu, lmax, lmax_out, N, C, batch, seed=77)
    base = run_nbody(inp).astype(np.float64)
    D = shref.wigner_D_real(lmax_out, shref.random_rotation(np.random.default_rng(2)))
    L2 = (lmax + 1) ** 2
    rot = synthetic.NbodyInputs(nu, lmax, lmax_out, N, C, batch,
                                np.einsum("ab,...b->...a", D[:L2, :L2], inp.X.astype(np.float64)).astype(np.float32),
                                inp.W_in, inp.W_out)
    got = run_nbody(rot).astype(np.float64)
    want = np.einsum("ab,...b->...a", D, base)
    assert np.abs(got - want).max() <= TOL * np.abs(base).max()


def test_nbody_grid_shape_and_errors():
    assert cg.cgtp_grid_shape_nu(2, 2, 3) == (5, 9)    # ceil((3*2+2+1)/2), 3*2+2+1
    assert cg.cgtp_grid_shape_nu(4, 4, 2) == cg.cgtp_grid_shape(4, 4)
    inp = synthetic.make_nbody(3, 2, 2, 4, 4, 0, seed=1)
    assert run_nbody(inp).shape == (0, 4, 9)  # empty batch
    with pytest.raises(cg.CgtpError) as e:
        run_nbody(synthetic.make_nbody(3, 2, 7, 4, 4, 2))  # lmax_out > nu * lmax
    assert e.value.code == cg.ERR_INVALID
    with pytest.raises(cg.CgtpError) as e:
        run_nbody(synthetic.make_nbody(5, 2, 2, 4, 4, 2))  # body order above the compiled limit
    assert e.value.code == cg.ERR_UNSUPPORTED
    with pytest.raises(cg.CgtpError) as e:
        run_nbody(synthetic.make_nbody(4, 20, 20, 4, 4, 2))  # four fields of band 20 do not fit the shared memory of an SM
    assert e.value.code == cg.ERR_UNSUPPORTED

"""cgtp_onsite_static (include/cgtp.h): the on-site contraction with its scratch in a file-scope device array, for callers
that cannot allocate device memory.  Checked against the existing path (cgtp_onsite with a workspace) on calls in a row that
share the array.  Named test_zz_* so that pytest collects it last: a failure here hides no other test under `pytest -x`."""
import numpy as np
import pytest
import torch

from paper_2605_15073_b200 import binding as cg
from paper_2605_15073_b200 import synthetic
from tests.parity_util import TOL, cuda, sector_errs_torch

pytestmark = pytest.mark.gpu


def _inputs(lmax, lmax_out, N, C, batch, seed, mask=None):
    inp = synthetic.make_onsite(lmax, lmax_out, N, C, batch, seed=seed, parity_mask=mask)
    T = [cuda(x) for x in (inp.A, inp.B, inp.W_a, inp.W_b, inp.W_out)]
    return inp, T


def _existing(inp, T):
    return cg.cgtp_onsite(*T, inp.lmax, inp.lmax_out, inp.N, inp.C, inp.parity_mask)


def _static(inp, T, out=None):
    if out is None:
        out = torch.full((inp.batch, 2, inp.N, (inp.lmax_out + 1) ** 2), float("nan"), device=T[0].device)
    return cg.cgtp_onsite_static(*T, inp.lmax, inp.lmax_out, inp.N, inp.C, inp.parity_mask, out)


@pytest.fixture(autouse=True)
def default_paths():
    cg.cgtp_set_kernel_path(0)
    cg.cgtp_set_math_mode(cg.MATH_FP32)
    yield
    cg.cgtp_set_kernel_path(0)


def test_static_scratch_entry_matches_existing_path_on_calls_in_a_row():
    # call 1 fills many slots of the array (lmax 4, 32 channels, several tiles per CTA, ragged last tile); call 2 runs a
    # different shape (other row stride, other band limit, lmax_out != lmax) over the contents call 1 left behind; call 3
    # repeats call 1's shape with other inputs and one parity only
    cases = [(4, 4, 32, 32, 2500, 11, None), (2, 3, 8, 24, 301, 12, None), (4, 2, 16, 32, 777, 13, [1] * 32),
             (1, 1, 4, 8, 5, 14, [0] * 8), (3, 3, 12, 256, 9, 15, None)]
    prepared = [_inputs(*c) for c in cases]
    refs = [_existing(inp, T).clone() for inp, T in prepared]
    gots = [_static(inp, T) for inp, T in prepared]  # back to back on one stream: no synchronisation in between
    torch.cuda.synchronize()
    for (inp, _), got, ref in zip(prepared, gots, refs):
        assert not torch.isnan(got).any()  # every output element was written
        e = sector_errs_torch(got, ref)
        assert max(e) < TOL, (inp.lmax, inp.lmax_out, inp.N, inp.C, inp.batch, e)
    # same call again, after the others dirtied the array: bitwise the same result
    inp, T = prepared[0]
    assert torch.equal(_static(inp, T), gots[0])


def test_static_scratch_entry_allocates_nothing_and_rejects_sizes_beyond_its_array():
    inp, T = _inputs(3, 3, 8, 16, 200, 21)
    out = torch.empty((inp.batch, 2, inp.N, 16), device=T[0].device)
    _static(inp, T, out)  # first call of this kernel: the driver may load its code now
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        _static(inp, T, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0  # no device memory was taken by the calls
    e = sector_errs_torch(out, _existing(inp, T))
    assert max(e) < TOL, e
    # beyond the stated maximum: a clear error, nothing launched
    big, Tb = _inputs(5, 5, 4, 4, 3, 22)
    with pytest.raises(cg.CgtpError, match="static scratch"):
        _static(big, Tb)
    wide, Tw = _inputs(1, 1, 4, 260, 2, 23)
    with pytest.raises(cg.CgtpError, match="static scratch"):
        _static(wide, Tw)
    with pytest.raises(ValueError):
        cg.cgtp_onsite_static(*T, 3, 3, 8, 16, inp.parity_mask, None)

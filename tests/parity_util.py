"""Helpers shared by the GPU parity tests: the error norm of the parity bar (R14, R22), deterministic
sub-samples of a batch, and Wigner-D rotation of feature tensors.  No arithmetic of the method lives here."""
import numpy as np
import torch

TOL = 1e-5


def cuda(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def sector_errs(got, ref):
    """[err_0, err_1], err_s = max|got - ref| / max|ref| over parity sector s (R14: never pooled -- odd-sector values
    are ~l^2 larger).  R22: a sector whose reference vanishes identically (no odd channels; the curl pairing at
    lmax_out = 0; self-coupled inputs) is measured against max|ref| of the whole output, and absolutely when the whole
    reference vanishes."""
    got = np.asarray(got, np.float64)
    ref = np.asarray(ref, np.float64)
    whole = np.abs(ref).max() if ref.size else 0.0
    errs = []
    for s in range(ref.shape[1]):
        d = np.abs(got[:, s] - ref[:, s]).max() if got.size else 0.0
        den = np.abs(ref[:, s]).max() if ref.size else 0.0
        if den == 0.0:
            den = whole
        errs.append(d / den if den > 0 else d)
    return errs


def sector_errs_torch(got: torch.Tensor, ref: torch.Tensor):
    """sector_errs for device tensors [batch, 2, ...] (whole batches at BASELINE's full sizes stay on the GPU)."""
    got, ref = got.double(), ref.double()
    whole = ref.abs().max().item() if ref.numel() else 0.0
    errs = []
    for s in range(ref.shape[1]):
        d = (got[:, s] - ref[:, s]).abs().max().item() if got.numel() else 0.0
        den = ref[:, s].abs().max().item() if ref.numel() else 0.0
        if den == 0.0:
            den = whole
        errs.append(d / den if den > 0 else d)
    return errs


def sample_rows(total: int, n: int, seed: int, extra=()):
    """At least n distinct rows of range(total): first and last two, a stride, `extra` (tile / chunk boundaries) and
    seeded random picks (first, last, strided and seeded-random atoms / receiver segments)."""
    rng = np.random.default_rng(seed)
    fixed = [0, 1, total - 2, total - 1, *extra]
    stride = np.arange(0, total, max(1, total // (n // 2)))
    idx = np.unique(np.concatenate([np.asarray(fixed, np.int64) % total, stride, rng.integers(0, total, n // 2)]))
    while idx.size < min(n, total):
        idx = np.unique(np.concatenate([idx, rng.integers(0, total, n - idx.size)]))
    return idx


def rotate_feats(X: torch.Tensor, D: np.ndarray) -> torch.Tensor:
    """X[..., (lmax+1)^2] -> D X in FP64 on the device, rounded to FP32 (h' = D h, tests/shref.wigner_D_real)."""
    Dt = torch.from_numpy(np.ascontiguousarray(D)).to(X.device)
    return (X.double() @ Dt.T).float().contiguous()


def degree_signs(lmax: int) -> np.ndarray:
    """(-1)^l per real-SH coefficient, flat index l^2 + l + m."""
    return np.concatenate([np.full(2 * l + 1, (-1.0) ** l) for l in range(lmax + 1)])

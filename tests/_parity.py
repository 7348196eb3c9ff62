"""Helpers for the GPU parity tests: error measures of BASELINE.json `north_star` and device upload.

fp64 bar: max |sigma_gpu - sigma_oracle| / sum|terms| <= 1e-13; fp32 variant: <= 1e-5 on the same
measure against the fp64 oracle of the original fp64 inputs (reading R18).  The VJP uses
the same measure with D = sum |g FK f| as denominator.
"""
import numpy as np

TOL64 = 1e-13
TOL32 = 1e-5


def rel_err(got: np.ndarray, ref: np.ndarray, scale: np.ndarray) -> float:
    """max |got - ref| / scale, with the convention 0/0 = 0 (exact zeros must be exact)."""
    got = np.asarray(got, dtype=np.float64)
    num = np.abs(got - ref)
    out = np.zeros_like(num)
    nz = scale > 0
    out[nz] = num[nz] / scale[nz]
    if np.any(num[~nz] != 0):
        return float("inf")
    return float(out.max()) if out.size else 0.0


def to_dev(a: np.ndarray, dtype=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()

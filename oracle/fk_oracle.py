"""ctypes wrapper over oracle/fk_oracle.c - TEST INFRASTRUCTURE, not the product.

Builds `libfkoracle.so` with gcc on first use (also built by `__graft_entry__.build()`).
Every function follows the passage cited in fk_oracle.c (Eq. (1); gradient P:47).
Shares no code with the CUDA path; never imports `paper_1909_10547_b200.fkconv`.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fk_oracle.c")
_LIB = os.path.join(_HERE, "libfkoracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        for name in ("fk_oracle_hadronic2", "fk_oracle_hadronic", "fk_oracle_dis",
                     "fk_oracle_hadronic_vjp", "fk_oracle_dis_vjp", "fk_oracle_chi2"):
            getattr(_lib, name).restype = ctypes.c_int
        _lib.fk_oracle_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(_load().fk_oracle_num_threads())


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def hadronic(fk, pairs, f, f2=None, nfl=None):
    """sigma[N][R], scale[N][R] (= sum |terms|) for FK[N][nx][nx][C], pairs[C][2], f[R][nfl][nx]."""
    fk, pairs, f = _d(fk), _i(pairs), _d(f)
    f2 = f if f2 is None else _d(f2)
    N, nx, nx2, C = fk.shape
    R, nfl_, nxf = f.shape
    assert nx == nx2 == nxf and pairs.shape == (C, 2) and f2.shape == f.shape
    sigma = np.empty((N, R)); scale = np.empty((N, R))
    rc = _load().fk_oracle_hadronic2(_p(fk), _p(pairs), _p(f), _p(f2), _p(sigma), _p(scale),
                                     N, nx, nfl_, C, R)
    if rc != 0:
        raise ValueError("fk_oracle_hadronic2: invalid argument")
    return sigma, scale


def dis(fk, flav, f):
    fk, flav, f = _d(fk), _i(flav), _d(f)
    N, nx, nA = fk.shape
    R, nfl_, nxf = f.shape
    assert nx == nxf and flav.shape == (nA,)
    sigma = np.empty((N, R)); scale = np.empty((N, R))
    rc = _load().fk_oracle_dis(_p(fk), _p(flav), _p(f), _p(sigma), _p(scale), N, nx, nfl_, nA, R)
    if rc != 0:
        raise ValueError("fk_oracle_dis: invalid argument")
    return sigma, scale


def hadronic_vjp(fk, pairs, f, g):
    """df[R][nfl][nx], D[R][nfl][nx] (= sum |terms|) for upstream g[N][R]."""
    fk, pairs, f, g = _d(fk), _i(pairs), _d(f), _d(g)
    N, nx, _, C = fk.shape
    R, nfl_, _ = f.shape
    assert g.shape == (N, R)
    df = np.empty_like(f); D = np.empty_like(f)
    rc = _load().fk_oracle_hadronic_vjp(_p(fk), _p(pairs), _p(f), _p(g), _p(df), _p(D), N, nx, nfl_, C, R)
    if rc != 0:
        raise ValueError("fk_oracle_hadronic_vjp: invalid argument")
    return df, D


def dis_vjp(fk, flav, f, g):
    fk, flav, f, g = _d(fk), _i(flav), _d(f), _d(g)
    N, nx, nA = fk.shape
    R, nfl_, _ = f.shape
    assert g.shape == (N, R)
    df = np.empty_like(f); D = np.empty_like(f)
    rc = _load().fk_oracle_dis_vjp(_p(fk), _p(flav), _p(f), _p(g), _p(df), _p(D), N, nx, nfl_, nA, R)
    if rc != 0:
        raise ValueError("fk_oracle_dis_vjp: invalid argument")
    return df, D


def chi2(sigma, data, cinv):
    """chi2[R], cscale[R], g[N][R], gscale[N][R] for sigma[N][R], data[N], symmetric cinv[N][N] (reading R22)."""
    sigma, data, cinv = _d(sigma), _d(data), _d(cinv)
    N, R = sigma.shape
    assert data.shape == (N,) and cinv.shape == (N, N)
    c = np.empty(R); cs = np.empty(R); g = np.empty((N, R)); gs = np.empty((N, R))
    rc = _load().fk_oracle_chi2(_p(sigma), _p(data), _p(cinv), _p(c), _p(cs), _p(g), _p(gs), N, R)
    if rc != 0:
        raise ValueError("fk_oracle_chi2: invalid argument")
    return c, cs, g, gs

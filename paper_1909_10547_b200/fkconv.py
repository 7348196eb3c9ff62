"""Thin ctypes binding over the C-ABI library `libfkconv.so` (include/fkconv.h) - argument
marshalling only: every step of the path runs in the CUDA kernels.  Same names as the C entry points.

Tensors are torch CUDA tensors (PyTorch is used for device memory and streams only); index lists
are host int32 arrays.  Importing this module fails loudly if the library has not been built
(`python -m paper_1909_10547_b200.build`); there is no CPU fallback and nothing here imports `oracle/`.

Eq. (1) of arXiv:1909.10547: sigma[n][r] = sum_{c,i,j} f[r][a_c][i] f[r][b_c][j] FK[n][i][j][c].
"""
from __future__ import annotations

import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfkconv.so")

FK_OK, FK_ERR_INVALID_ARG, FK_ERR_ALLOC, FK_ERR_CUDA, FK_ERR_UNSUPPORTED = 0, -1, -2, -3, -4
FK_KIND_DIS, FK_KIND_HADRONIC = 0, 1
FK_F64, FK_F32, FK_F32S64 = 0, 1, 2
FK_STORE_BORROW, FK_STORE_PACK, FK_STORE_SPARSE = 0, 1, 2
(FK_OPT_GEMM_MIN_R, FK_OPT_WARP_SPEC, FK_OPT_FOLD, FK_OPT_FOLDK, FK_OPT_FUSED, FK_OPT_FEWROWS, FK_OPT_TC32,
 FK_OPT_TC32_MIN_R, FK_OPT_PDL, FK_OPT_FUSE_L2, FK_OPT_DIS_DIRECT) = range(11)

# every symbol include/fkconv.h declares
SYMBOLS = (
    "fk_last_error_string", "fk_version", "fk_compiled_arch", "fk_profile_enable", "fk_profile_read", "fk_profile_report", "fk_set_option", "fk_get_option",
    "fk_conv_dis", "fk_conv_hadronic", "fk_conv_hadronic_vjp", "fk_conv_dis_vjp",
    "fk_conv_dis_f32", "fk_conv_hadronic_f32", "fk_conv_hadronic_vjp_f32",
    "fk_table_create", "fk_table_destroy", "fk_table_info", "fk_table_conv", "fk_table_vjp", "fk_table_conv_vjp", "fk_chi2", "fk_table_fit_step",
    "fk_table_conv_host", "fk_table_vjp_host", "fk_table_last_launches",
    "fk_group_create", "fk_group_destroy", "fk_group_offsets", "fk_conv_grouped",
    "fk_conv_grouped_vjp", "fk_conv_grouped_conv_vjp", "fk_group_last_launches", "fk_conv_hadronic2", "fk_conv_hadronic2_vjp", "fk_probe_launch",
    "fk_conv_hadronic_static", "fk_table_conv_vjp_host",
)
FK_STATIC_SCRATCH_BYTES = 32 << 20   # include/fkconv.h

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python -m paper_1909_10547_b200.build` "
        "(nvcc, sm_100a). The FK convolution has no CPU fallback.")

lib = ctypes.CDLL(LIB_PATH)
for _name in SYMBOLS:
    getattr(lib, _name).restype = ctypes.c_int
lib.fk_last_error_string.restype = ctypes.c_char_p

_vp, _ci = ctypes.c_void_p, ctypes.c_int
for _name in ("fk_conv_dis", "fk_conv_hadronic", "fk_conv_dis_f32", "fk_conv_hadronic_f32", "fk_conv_hadronic_static"):
    getattr(lib, _name).argtypes = [_vp, _vp, _vp, _vp, _ci, _ci, _ci, _ci, _ci, _vp]
for _name in ("fk_conv_hadronic_vjp", "fk_conv_dis_vjp", "fk_conv_hadronic_vjp_f32"):
    getattr(lib, _name).argtypes = [_vp, _vp, _vp, _vp, _vp, _ci, _ci, _ci, _ci, _ci, _vp]
lib.fk_conv_hadronic2.argtypes = [_vp, _vp, _vp, _vp, _vp, _ci, _ci, _ci, _ci, _ci, _vp]
lib.fk_conv_hadronic2_vjp.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _ci, _ci, _ci, _ci, _ci, _vp]
lib.fk_probe_launch.argtypes = [_ci, _vp, ctypes.c_longlong, _vp, _vp]
lib.fk_profile_enable.argtypes = [_ci]
lib.fk_set_option.argtypes = [_ci, _ci]
lib.fk_get_option.argtypes = [_ci, ctypes.POINTER(_ci)]
lib.fk_profile_read.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.POINTER(_ci)]
lib.fk_profile_report.argtypes = [ctypes.c_char_p, _ci]
lib.fk_table_create.argtypes = [ctypes.POINTER(_vp), _ci, _vp, _vp, _ci, _ci, _ci, _ci, _ci, _ci, _ci]
lib.fk_table_destroy.argtypes = [_vp]
lib.fk_table_info.argtypes = [_vp] + [ctypes.POINTER(_ci)] * 4 + [ctypes.POINTER(ctypes.c_int64)] * 3
lib.fk_table_conv.argtypes = [_vp, _vp, _vp, _ci, _vp]
lib.fk_table_vjp.argtypes = [_vp, _vp, _vp, _vp, _ci, _vp]
lib.fk_chi2.argtypes = [_vp, _vp, _vp, _vp, _vp, _ci, _ci, _vp]
lib.fk_table_fit_step.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _ci, _vp]
lib.fk_table_conv_vjp.argtypes = [_vp, _vp, _vp, _vp, _vp, _ci, _vp]
lib.fk_table_conv_host.argtypes = [_vp, _vp, _vp, _ci, _vp]
lib.fk_table_vjp_host.argtypes = [_vp, _vp, _vp, _vp, _ci, _vp]
lib.fk_table_conv_vjp_host.argtypes = [_vp, _vp, _vp, _vp, _vp, _ci, _vp]
lib.fk_table_last_launches.argtypes = [_vp]
lib.fk_group_create.argtypes = [ctypes.POINTER(_vp), ctypes.POINTER(_vp), _ci, _ci]
lib.fk_group_destroy.argtypes = [_vp]
lib.fk_group_offsets.argtypes = [_vp, _ci, _vp, _vp]
lib.fk_conv_grouped.argtypes = [_vp, _vp, _vp, _ci, _vp]
lib.fk_conv_grouped_vjp.argtypes = [_vp, _vp, _vp, _vp, _ci, _vp]
lib.fk_conv_grouped_conv_vjp.argtypes = [_vp, _vp, _vp, _vp, _vp, _ci, _vp]
lib.fk_group_last_launches.argtypes = [_vp]


class FkError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = lib.fk_last_error_string()
        super().__init__(f"{where}: status {code}: {msg.decode() if msg else ''}")


def _check(rc: int, where: str) -> None:
    if rc != FK_OK:
        raise FkError(rc, where)


def _stream(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream)


def _dev(t: torch.Tensor, dtype=None) -> int:
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
        raise TypeError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    return t.data_ptr()


def _shape(t, shape, what: str, device=None) -> None:
    """Marshalling check: the kernels trust the sizes the handle was created with."""
    if tuple(t.shape) != tuple(shape):
        raise ValueError(f"{what}: expected shape {tuple(shape)}, got {tuple(t.shape)}")
    if device is not None and isinstance(t, torch.Tensor) and t.device != device:
        raise ValueError(f"{what}: tensor on {t.device}, table on {device}")


def _host(a, dtype, shape, what: str) -> int:
    if not (isinstance(a, np.ndarray) and a.dtype == dtype and a.flags.c_contiguous):
        raise TypeError(f"{what}: expected a C-contiguous numpy array of dtype {np.dtype(dtype)}")
    if tuple(a.shape) != tuple(shape):
        raise ValueError(f"{what}: expected shape {tuple(shape)}, got {tuple(a.shape)}")
    return a.ctypes.data


def _idx(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def _hostptr(a: np.ndarray) -> int:
    return a.ctypes.data


def set_option(option: int, value: int) -> None:
    _check(lib.fk_set_option(option, value), "fk_set_option")


def get_option(option: int) -> int:
    v = _ci()
    _check(lib.fk_get_option(option, ctypes.byref(v)), "fk_get_option")
    return v.value


def probe_launch(kind: int, buf=None, sink=None, stream=None) -> None:
    """Latency floors: kind 0 = empty kernel, kind 1 = one streaming read of `buf` (any contiguous device tensor)."""
    nbytes = 0 if buf is None else buf.numel() * buf.element_size()
    _check(lib.fk_probe_launch(kind, None if buf is None else _vp(buf.data_ptr()), nbytes,
                               None if sink is None else _vp(sink.data_ptr()), _stream(stream)), "fk_probe_launch")


def profile_enable(on: bool) -> None:
    _check(lib.fk_profile_enable(1 if on else 0), "fk_profile_enable")


def profile_report() -> dict:
    """{kernel name: (launches, total milliseconds)} of the launches recorded since the last report."""
    buf = ctypes.create_string_buffer(1 << 16)
    _check(lib.fk_profile_report(buf, len(buf)), "fk_profile_report")
    out = {}
    for ln in buf.value.decode().splitlines():
        name, n, ms = ln.split("\t")
        out[name] = (int(n), float(ms))
    return out


def version() -> int:
    return lib.fk_version()


def compiled_arch() -> int:
    return lib.fk_compiled_arch()


# ------------------------------------------------------------------ stateless entry points
def fk_conv_hadronic(fk, pairs, f, sigma=None, stream=None):
    """fk[N][nx][nx][C], pairs[C][2] (host), f[R][nfl][nx] -> sigma[N][R] (fp64, or fp32 if fk is)."""
    N, nx, _, C = fk.shape
    R, nfl, _ = f.shape
    pairs = _idx(pairs)
    if sigma is None:
        sigma = torch.empty((N, R), dtype=fk.dtype, device=fk.device)
    _shape(pairs, (C, 2), "pairs"); _shape(f, (R, nfl, nx), "f", fk.device); _shape(sigma, (N, R), "sigma", fk.device)
    fn = lib.fk_conv_hadronic if fk.dtype == torch.float64 else lib.fk_conv_hadronic_f32
    _check(fn(_dev(fk), _hostptr(pairs), _dev(f, fk.dtype), _dev(sigma, fk.dtype), N, nx, nfl, C, R,
              _stream(stream)), "fk_conv_hadronic")
    return sigma


def fk_conv_hadronic_static(fk, pairs, f, sigma, stream=None):
    """fk_conv_hadronic (fp64) without any device allocation inside the library: the scratch is a static device array of
    FK_STATIC_SCRATCH_BYTES (include/fkconv.h).  The caller passes the output; larger problems raise FkError
    (FK_ERR_UNSUPPORTED); calls that overlap on the GPU race on the shared array."""
    N, nx, _, C = fk.shape
    R, nfl, _ = f.shape
    pairs = _idx(pairs)
    if fk.dtype != torch.float64:
        raise TypeError("fk_conv_hadronic_static: fp64 only")
    _shape(pairs, (C, 2), "pairs"); _shape(f, (R, nfl, nx), "f", fk.device); _shape(sigma, (N, R), "sigma", fk.device)
    _check(lib.fk_conv_hadronic_static(_dev(fk), _hostptr(pairs), _dev(f, fk.dtype), _dev(sigma, fk.dtype), N, nx, nfl, C, R,
                                       _stream(stream)), "fk_conv_hadronic_static")
    return sigma


def fk_conv_dis(fk, flav, f, sigma=None, stream=None):
    """fk[N][nx][nA], flav[nA] (host), f[R][nfl][nx] -> sigma[N][R]."""
    N, nx, nA = fk.shape
    R, nfl, _ = f.shape
    flav = _idx(flav)
    if sigma is None:
        sigma = torch.empty((N, R), dtype=fk.dtype, device=fk.device)
    _shape(flav, (nA,), "flav"); _shape(f, (R, nfl, nx), "f", fk.device); _shape(sigma, (N, R), "sigma", fk.device)
    fn = lib.fk_conv_dis if fk.dtype == torch.float64 else lib.fk_conv_dis_f32
    _check(fn(_dev(fk), _hostptr(flav), _dev(f, fk.dtype), _dev(sigma, fk.dtype), N, nx, nfl, nA, R,
              _stream(stream)), "fk_conv_dis")
    return sigma


def fk_conv_hadronic_vjp(fk, pairs, f, g, df=None, stream=None):
    """df[R][nfl][nx] = d(sum_n g[n][r] sigma[n][r]) / d f[r][alpha][i]."""
    N, nx, _, C = fk.shape
    R, nfl, _ = f.shape
    pairs = _idx(pairs)
    if df is None:
        df = torch.empty_like(f)
    _shape(pairs, (C, 2), "pairs"); _shape(f, (R, nfl, nx), "f", fk.device); _shape(g, (N, R), "g", fk.device)
    _shape(df, (R, nfl, nx), "df", fk.device)
    fn = lib.fk_conv_hadronic_vjp if fk.dtype == torch.float64 else lib.fk_conv_hadronic_vjp_f32
    _check(fn(_dev(fk), _hostptr(pairs), _dev(f, fk.dtype), _dev(g, fk.dtype), _dev(df, fk.dtype),
              N, nx, nfl, C, R, _stream(stream)), "fk_conv_hadronic_vjp")
    return df


def fk_conv_hadronic2(fk, pairs, f1, f2, sigma=None, stream=None):
    """Two-PDF (p pbar) form: sigma[n][r] = sum f1[r][a_c][i] f2[r][b_c][j] FK[n][i][j][c] (fp64)."""
    N, nx, _, C = fk.shape
    R, nfl, _ = f1.shape
    pairs = _idx(pairs)
    if sigma is None:
        sigma = torch.empty((N, R), dtype=torch.float64, device=fk.device)
    _shape(pairs, (C, 2), "pairs"); _shape(f1, (R, nfl, nx), "f1", fk.device); _shape(f2, (R, nfl, nx), "f2", fk.device)
    _shape(sigma, (N, R), "sigma", fk.device)
    _check(lib.fk_conv_hadronic2(_dev(fk, torch.float64), _hostptr(pairs), _dev(f1, torch.float64), _dev(f2, torch.float64),
                                 _dev(sigma, torch.float64), N, nx, nfl, C, R, _stream(stream)), "fk_conv_hadronic2")
    return sigma


def fk_conv_hadronic2_vjp(fk, pairs, f1, f2, g, df1=None, df2=None, stream=None):
    """(df1, df2): the derivatives of sum_n g[n][r] sigma[n][r] with respect to f1 and f2."""
    N, nx, _, C = fk.shape
    R, nfl, _ = f1.shape
    pairs = _idx(pairs)
    df1 = torch.empty_like(f1) if df1 is None else df1
    df2 = torch.empty_like(f2) if df2 is None else df2
    _shape(pairs, (C, 2), "pairs"); _shape(f1, (R, nfl, nx), "f1", fk.device); _shape(f2, (R, nfl, nx), "f2", fk.device)
    _shape(g, (N, R), "g", fk.device); _shape(df1, (R, nfl, nx), "df1", fk.device); _shape(df2, (R, nfl, nx), "df2", fk.device)
    t64 = torch.float64
    _check(lib.fk_conv_hadronic2_vjp(_dev(fk, t64), _hostptr(pairs), _dev(f1, t64), _dev(f2, t64), _dev(g, t64), _dev(df1, t64),
                                     _dev(df2, t64), N, nx, nfl, C, R, _stream(stream)), "fk_conv_hadronic2_vjp")
    return df1, df2


def fk_conv_dis_vjp(fk, flav, f, g, df=None, stream=None):
    N, nx, nA = fk.shape
    R, nfl, _ = f.shape
    flav = _idx(flav)
    if df is None:
        df = torch.empty_like(f)
    _shape(flav, (nA,), "flav"); _shape(f, (R, nfl, nx), "f", fk.device); _shape(g, (N, R), "g", fk.device)
    _shape(df, (R, nfl, nx), "df", fk.device)
    _check(lib.fk_conv_dis_vjp(_dev(fk, torch.float64), _hostptr(flav), _dev(f, torch.float64),
                               _dev(g, torch.float64), _dev(df, torch.float64), N, nx, nfl, nA, R,
                               _stream(stream)), "fk_conv_dis_vjp")
    return df


def fk_chi2(sigma, data, cinv, chi2=None, g=None, stream=None):
    """chi2[R], g[N][R] for sigma[N][R], data[N], symmetric cinv[N][N] (fp64, device)."""
    N, R = sigma.shape
    if chi2 is None:
        chi2 = torch.empty(R, dtype=torch.float64, device=sigma.device)
    if g is None:
        g = torch.empty_like(sigma)
    _shape(data, (N,), "data", sigma.device); _shape(cinv, (N, N), "cinv", sigma.device)
    _shape(chi2, (R,), "chi2", sigma.device); _shape(g, (N, R), "g", sigma.device)
    _check(lib.fk_chi2(_dev(sigma, torch.float64), _dev(data, torch.float64), _dev(cinv, torch.float64),
                       _dev(chi2, torch.float64), _dev(g, torch.float64), N, R, _stream(stream)), "fk_chi2")
    return chi2, g


# ------------------------------------------------------------------ resident tables
class FkTable:
    """fk_table handle.  `fk_logical` is the fp64 logical-layout table on the device; with
    store=FK_STORE_BORROW it must stay alive (a reference is kept here)."""

    def __init__(self, kind, fk_logical, index_list, nfl, dtype=FK_F64, store=FK_STORE_PACK, R_hint=1):
        self.kind = kind
        idx = _idx(index_list)
        if kind == FK_KIND_HADRONIC:
            N, nx, _, C = fk_logical.shape
        else:
            N, nx, C = fk_logical.shape
        _shape(idx, (C, 2) if kind == FK_KIND_HADRONIC else (C,), "index_list")
        self.N, self.nx, self.nfl, self.C = N, nx, nfl, C
        self.dtype = dtype
        self.tdtype = torch.float32 if dtype == FK_F32 else torch.float64  # FK_F32S64: fp32 table, fp64 buffers
        self.ndtype = np.float32 if dtype == FK_F32 else np.float64
        self.device = fk_logical.device
        self._keep = fk_logical if store == FK_STORE_BORROW else None
        h = _vp()
        _check(lib.fk_table_create(ctypes.byref(h), kind, _dev(fk_logical, torch.float64), _hostptr(idx),
                                   N, nx, nfl, C, dtype, store, R_hint), "fk_table_create")
        self.handle = h

    def info(self):
        N, nx, nfl, C = _ci(), _ci(), _ci(), _ci()
        K, rs, nb = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
        _check(lib.fk_table_info(self.handle, N, nx, nfl, C, K, rs, nb), "fk_table_info")
        return dict(N=N.value, nx=nx.value, nfl=nfl.value, C=C.value, K=K.value, row_stride=rs.value,
                    device_bytes=nb.value)

    def _chk(self, R, f=None, sigma=None, g=None, df=None):
        for t, shape, what in ((f, (R, self.nfl, self.nx), "f"), (sigma, (self.N, R), "sigma"), (g, (self.N, R), "g"),
                               (df, (R, self.nfl, self.nx), "df")):
            if t is not None:
                _shape(t, shape, what, self.device)

    def conv(self, f, sigma=None, stream=None):
        R = f.shape[0]
        if sigma is None:
            sigma = torch.empty((self.N, R), dtype=self.tdtype, device=self.device)
        self._chk(R, f=f, sigma=sigma)
        _check(lib.fk_table_conv(self.handle, _dev(f, self.tdtype), _dev(sigma, self.tdtype), R,
                                 _stream(stream)), "fk_table_conv")
        return sigma

    def vjp(self, f, g, df=None, stream=None):
        R = f.shape[0]
        if df is None:
            df = torch.empty_like(f)
        self._chk(R, f=f, g=g, df=df)
        _check(lib.fk_table_vjp(self.handle, _dev(f, self.tdtype), _dev(g, self.tdtype), _dev(df, self.tdtype),
                                R, _stream(stream)), "fk_table_vjp")
        return df

    def conv_vjp(self, f, g, sigma=None, df=None, stream=None):
        """sigma and df from ONE read of FK, for an upstream gradient g known before the forward pass."""
        R = f.shape[0]
        if sigma is None:
            sigma = torch.empty((self.N, R), dtype=self.tdtype, device=self.device)
        if df is None:
            df = torch.empty_like(f)
        self._chk(R, f=f, sigma=sigma, g=g, df=df)
        _check(lib.fk_table_conv_vjp(self.handle, _dev(f, self.tdtype), _dev(g, self.tdtype), _dev(sigma, self.tdtype),
                                     _dev(df, self.tdtype), R, _stream(stream)), "fk_table_conv_vjp")
        return sigma, df

    def fit_step(self, f, data, cinv, sigma=None, g=None, chi2=None, df=None, stream=None):
        """One fit iteration: sigma = conv(f), (chi2, g) = fk_chi2(sigma, data, cinv), df = vjp(f, g)."""
        R = f.shape[0]
        sigma = torch.empty((self.N, R), dtype=self.tdtype, device=self.device) if sigma is None else sigma
        g = torch.empty_like(sigma) if g is None else g
        chi2 = torch.empty(R, dtype=torch.float64, device=self.device) if chi2 is None else chi2
        df = torch.empty_like(f) if df is None else df
        self._chk(R, f=f, sigma=sigma, g=g, df=df)
        _shape(data, (self.N,), "data", self.device); _shape(cinv, (self.N, self.N), "cinv", self.device)
        _shape(chi2, (R,), "chi2", self.device)
        _check(lib.fk_table_fit_step(self.handle, _dev(f, torch.float64), _dev(data, torch.float64), _dev(cinv, torch.float64),
                                     _dev(sigma, torch.float64), _dev(g, torch.float64), _dev(chi2, torch.float64),
                                     _dev(df, torch.float64), R, _stream(stream)), "fk_table_fit_step")
        return sigma, chi2, g, df

    def conv_host(self, f_host: np.ndarray, sigma_host: np.ndarray, stream=None):
        R = f_host.shape[0]
        fp = _host(f_host, self.ndtype, (R, self.nfl, self.nx), "f_host")
        sp = _host(sigma_host, self.ndtype, (self.N, R), "sigma_host")
        _check(lib.fk_table_conv_host(self.handle, fp, sp, R, _stream(stream)),
               "fk_table_conv_host")
        return sigma_host

    def vjp_host(self, f_host: np.ndarray, g_host: np.ndarray, df_host: np.ndarray, stream=None):
        R = f_host.shape[0]
        fp = _host(f_host, self.ndtype, (R, self.nfl, self.nx), "f_host")
        gp = _host(g_host, self.ndtype, (self.N, R), "g_host")
        dp = _host(df_host, self.ndtype, (R, self.nfl, self.nx), "df_host")
        _check(lib.fk_table_vjp_host(self.handle, fp, gp, dp, R, _stream(stream)), "fk_table_vjp_host")
        return df_host

    def conv_vjp_host(self, f_host: np.ndarray, g_host: np.ndarray, sigma_host: np.ndarray, df_host: np.ndarray, stream=None):
        R = f_host.shape[0]
        fp = _host(f_host, self.ndtype, (R, self.nfl, self.nx), "f_host")
        gp = _host(g_host, self.ndtype, (self.N, R), "g_host")
        sp = _host(sigma_host, self.ndtype, (self.N, R), "sigma_host")
        dp = _host(df_host, self.ndtype, (R, self.nfl, self.nx), "df_host")
        _check(lib.fk_table_conv_vjp_host(self.handle, fp, gp, sp, dp, R, _stream(stream)), "fk_table_conv_vjp_host")
        return sigma_host, df_host

    def last_launches(self) -> int:
        return lib.fk_table_last_launches(self.handle)

    def destroy(self):
        if getattr(self, "handle", None):
            lib.fk_table_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class FkGroup:
    """fk_group handle: ragged set of tables, one persistent launch per pass."""

    def __init__(self, tables, R_hint=1):
        self.tables = list(tables)
        T = len(self.tables)
        arr = (_vp * T)(*[t.handle for t in self.tables])
        h = _vp()
        _check(lib.fk_group_create(ctypes.byref(h), arr, T, R_hint), "fk_group_create")
        self.handle = h
        self.T = T
        self.tdtype = self.tables[0].tdtype
        self.device = self.tables[0].device

    def offsets(self, R):
        fo = np.zeros(self.T + 1, dtype=np.int64)
        so = np.zeros(self.T + 1, dtype=np.int64)
        _check(lib.fk_group_offsets(self.handle, R, _hostptr(fo), _hostptr(so)), "fk_group_offsets")
        return fo, so

    def _chk(self, R, f_cat=None, sigma_cat=None, g_cat=None, df_cat=None):
        fo, so = self.offsets(R)
        for t, n, what in ((f_cat, fo[-1], "f_cat"), (df_cat, fo[-1], "df_cat"), (sigma_cat, so[-1], "sigma_cat"),
                           (g_cat, so[-1], "g_cat")):
            if t is not None:
                if t.numel() != int(n):
                    raise ValueError(f"{what}: expected {int(n)} elements (fk_group_offsets), got {t.numel()}")
                if t.device != self.device:
                    raise ValueError(f"{what}: tensor on {t.device}, group on {self.device}")

    def conv(self, f_cat, R, sigma_cat=None, stream=None):
        if sigma_cat is None:
            _, so = self.offsets(R)
            sigma_cat = torch.empty(int(so[-1]), dtype=self.tdtype, device=self.device)
        self._chk(R, f_cat=f_cat, sigma_cat=sigma_cat)
        _check(lib.fk_conv_grouped(self.handle, _dev(f_cat, self.tdtype), _dev(sigma_cat, self.tdtype), R,
                                   _stream(stream)), "fk_conv_grouped")
        return sigma_cat

    def vjp(self, f_cat, g_cat, R, df_cat=None, stream=None):
        if df_cat is None:
            df_cat = torch.empty_like(f_cat)
        self._chk(R, f_cat=f_cat, g_cat=g_cat, df_cat=df_cat)
        _check(lib.fk_conv_grouped_vjp(self.handle, _dev(f_cat, self.tdtype), _dev(g_cat, self.tdtype),
                                       _dev(df_cat, self.tdtype), R, _stream(stream)), "fk_conv_grouped_vjp")
        return df_cat

    def conv_vjp(self, f_cat, g_cat, R, sigma_cat=None, df_cat=None, stream=None):
        """Forward and VJP of the whole group from one read of every table (g known before the forward pass)."""
        if sigma_cat is None:
            sigma_cat = torch.empty(int(self.offsets(R)[1][-1]), dtype=self.tdtype, device=f_cat.device)
        if df_cat is None:
            df_cat = torch.empty_like(f_cat)
        self._chk(R, f_cat=f_cat, sigma_cat=sigma_cat, g_cat=g_cat, df_cat=df_cat)
        _check(lib.fk_conv_grouped_conv_vjp(self.handle, _dev(f_cat, self.tdtype), _dev(g_cat, self.tdtype), _dev(sigma_cat, self.tdtype),
                                            _dev(df_cat, self.tdtype), R, _stream(stream)), "fk_conv_grouped_conv_vjp")
        return sigma_cat, df_cat

    def last_launches(self) -> int:
        return lib.fk_group_last_launches(self.handle)

    def destroy(self):
        if getattr(self, "handle", None):
            lib.fk_group_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no convolution, no luminosity, no
gradient): it only draws the inputs that stand in for the NNPDF3.1 FK tables and PDF grids
the paper used (PAPER.md:29, :47 - not available here).  Recipe: BASELINE.json `configs`,
SURVEY.md 8(c).4 / 8(d), restated in DESIGN.md "Input recipe".

* FK entries i.i.d. N(0,1) (config 1: 30% zeroed by an i.i.d. Bernoulli mask, stored dense).
* x-grid log-spaced 1e-5..1, last point exactly 1.0 (reading R12).
* f_a(x) = A_a x^(-p_a) (1-x)^(q_a), A~U[0.1,2], p~U[0,0.5], q~U[1,5] per flavour and replica,
  evaluated once on the host in fp64; the same bytes go to oracle and GPU (reading R13).
* seeds: 190910547 + 1000*config + tensor_id, numpy Philox (counter-based) bit generator.

Logical layouts (BASELINE.json): hadronic FK[N][nx][nx][C] (channel innermost),
DIS FK[N][nx][nA], pairs[C][2] int32, flav[nA] int32, f[R][nfl][nx], g[N][R].
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 190910547
NFL = 14

# tensor ids
T_FK, T_PAIRS, T_PDF, T_G, T_SHAPE, T_MASK = 0, 1, 2, 3, 4, 5


def rng_for(config: int, tensor_id: int, sub: int = 0) -> np.random.Generator:
    """Counter-based generator keyed by (config, tensor, sub-stream)."""
    seed = BASE_SEED + 1000 * config + tensor_id
    return np.random.Generator(np.random.Philox(key=[seed, sub]))


def x_grid(nx: int) -> np.ndarray:
    """x_i = 10^(-5 + 5 i/(nx-1)), i=0..nx-1, with x_{nx-1} = 1.0 exactly."""
    if nx == 1:
        return np.array([1.0])
    x = 10.0 ** (-5.0 + 5.0 * np.arange(nx, dtype=np.float64) / (nx - 1))
    x[-1] = 1.0
    return x


def pdf_params(rng: np.random.Generator, R: int, nfl: int = NFL):
    A = rng.uniform(0.1, 2.0, size=(R, nfl))
    p = rng.uniform(0.0, 0.5, size=(R, nfl))
    q = rng.uniform(1.0, 5.0, size=(R, nfl))
    return A, p, q


def pdf_grid(params, nx: int) -> np.ndarray:
    """f[R][nfl][nx] from per-(replica, flavour) (A, p, q) on the nx-point grid."""
    A, p, q = params
    x = x_grid(nx)[None, None, :]
    f = A[..., None] * x ** (-p[..., None]) * (1.0 - x) ** (q[..., None])
    return np.ascontiguousarray(f, dtype=np.float64)


def draw_pairs(rng: np.random.Generator, C: int, nfl: int = NFL) -> np.ndarray:
    """C distinct ordered flavour pairs out of nfl*nfl, in increasing (a*nfl+b) order.
    All pairs active (C == nfl*nfl) gives the full list in order."""
    if C > nfl * nfl:
        raise ValueError("C > nfl^2")
    idx = np.sort(rng.choice(nfl * nfl, size=C, replace=False))
    return np.stack([idx // nfl, idx % nfl], axis=1).astype(np.int32)


def draw_flavours(rng: np.random.Generator, nA: int, nfl: int = NFL) -> np.ndarray:
    return np.sort(rng.choice(nfl, size=nA, replace=False)).astype(np.int32)


def normal_table(rng: np.random.Generator, shape) -> np.ndarray:
    return rng.standard_normal(size=shape, dtype=np.float64)


@dataclass
class HadronicCase:
    name: str
    fk: np.ndarray          # [N][nx][nx][C]
    pairs: np.ndarray       # [C][2] int32
    f: np.ndarray           # [R][nfl][nx]
    g: np.ndarray | None = None   # [N][R]
    nfl: int = NFL

    @property
    def N(self): return self.fk.shape[0]
    @property
    def nx(self): return self.fk.shape[1]
    @property
    def C(self): return self.fk.shape[3]
    @property
    def R(self): return self.f.shape[0]


@dataclass
class DisCase:
    name: str
    fk: np.ndarray          # [N][nx][nA]
    flav: np.ndarray        # [nA] int32
    f: np.ndarray           # [R][nfl][nx]
    g: np.ndarray | None = None
    nfl: int = NFL

    @property
    def N(self): return self.fk.shape[0]
    @property
    def nx(self): return self.fk.shape[1]
    @property
    def nA(self): return self.fk.shape[2]
    @property
    def R(self): return self.f.shape[0]


def hadronic_case(config: int, N: int, nx: int, C: int, R: int, nfl: int = NFL,
                  name: str = "", sub: int = 0, with_g: bool = True) -> HadronicCase:
    pairs = draw_pairs(rng_for(config, T_PAIRS, sub), C, nfl)
    fk = normal_table(rng_for(config, T_FK, sub), (N, nx, nx, C))
    f = pdf_grid(pdf_params(rng_for(config, T_PDF, 0), R, nfl), nx)
    g = None
    if with_g:
        w = rng_for(config, T_G, sub).standard_normal(size=(N, 1))
        g = np.ascontiguousarray(np.broadcast_to(w, (N, R)))   # reading R9: g[n][r] = w[n]
    return HadronicCase(name or f"cfg{config}", fk, pairs, f, g, nfl)


def config0(R: int = 1) -> HadronicCase:
    """BASELINE config 0: tiny hadronic, N=16, nx=20, all 196 pairs."""
    return hadronic_case(0, 16, 20, 196, R, name="cfg0-tiny-hadronic")


def config1(R: int = 1, N: int = 2048) -> DisCase:
    """BASELINE config 1: DIS, N=2048, nx=50, 9 of 14 flavours, 30% of entries zeroed."""
    nx, nA = 50, 9
    flav = draw_flavours(rng_for(1, T_PAIRS), nA)
    fk = normal_table(rng_for(1, T_FK), (N, nx, nA))
    mask = rng_for(1, T_MASK).random(size=fk.shape) < 0.3
    fk[mask] = 0.0
    f = pdf_grid(pdf_params(rng_for(1, T_PDF), R), nx)
    w = rng_for(1, T_G).standard_normal(size=(N, 1))
    g = np.ascontiguousarray(np.broadcast_to(w, (N, R)))
    return DisCase("cfg1-dis", fk, flav, f, g)


def config2(R: int = 1, N: int = 512) -> HadronicCase:
    """BASELINE config 2 (R=1) / config 3 (R=128): N=512, nx=50, 100 of 196 pairs, ~1.0 GB.
    Config 3 reuses config 2's table (same seeds) with R per-replica PDFs."""
    return hadronic_case(2, N, 50, 100, R, name="cfg2-hadronic-1GB" if R == 1 else "cfg3-hadronic-R%d" % R)


@dataclass
class RaggedShapes:
    N: np.ndarray
    nx: np.ndarray
    C: np.ndarray

    @property
    def T(self): return len(self.N)
    def fk_elements(self) -> int:
        return int(np.sum(self.N.astype(np.int64) * self.nx.astype(np.int64) ** 2 * self.C))


def config4_shapes(T: int = 60, scale_to_sumN: int | None = None) -> RaggedShapes:
    """BASELINE config 4 shapes: N~U{10..400}, nx~U{30..50}, C~U{20..150} (reading R15: the
    explicit distributions are the config of record; `scale_to_sumN=4000` gives variant B)."""
    rng = rng_for(4, T_SHAPE)
    N = rng.integers(10, 401, size=T)
    nx = rng.integers(30, 51, size=T)
    C = rng.integers(20, 151, size=T)
    if scale_to_sumN is not None:
        N = np.maximum(10, np.round(N * (scale_to_sumN / N.sum())).astype(np.int64))
    return RaggedShapes(N.astype(np.int64), nx.astype(np.int64), C.astype(np.int64))


def config4_table(t: int, shapes: RaggedShapes, R: int, params=None, with_fk: bool = True) -> HadronicCase:
    """Table t of the ragged batch.  One PDF (A,p,q) per replica, sampled on each table's own
    x-grid (reading R14).  with_fk=False: the table is a zero-memory placeholder of the right shape (a rank of a
    sharded run needs f, g and the shapes of the tables it does not own, not their entries)."""
    N, nx, C = int(shapes.N[t]), int(shapes.nx[t]), int(shapes.C[t])
    pairs = draw_pairs(rng_for(4, T_PAIRS, t + 1), C)
    fk = normal_table(rng_for(4, T_FK, t + 1), (N, nx, nx, C)) if with_fk else np.broadcast_to(np.zeros((), dtype=np.float64), (N, nx, nx, C))
    if params is None:
        params = pdf_params(rng_for(4, T_PDF), R)
    f = pdf_grid(params, nx)
    w = rng_for(4, T_G, t + 1).standard_normal(size=(N, 1))
    g = np.ascontiguousarray(np.broadcast_to(w, (N, R)))
    return HadronicCase(f"cfg4-t{t}", fk, pairs, f, g)


def small_ragged_shapes(T: int = 7, seed_sub: int = 99) -> RaggedShapes:
    """Scaled-down ragged batch for parity tests the oracle finishes in seconds (odd nx, N=1,
    C=1 included on purpose)."""
    rng = rng_for(4, T_SHAPE, seed_sub)
    N = rng.integers(1, 40, size=T); nx = rng.integers(5, 24, size=T); C = rng.integers(1, 30, size=T)
    N[0], nx[0], C[0] = 1, 7, 1
    if T > 1:
        N[1], nx[1], C[1] = 37, 23, 29
    return RaggedShapes(N.astype(np.int64), nx.astype(np.int64), C.astype(np.int64))


def integer_hadronic_case(seed_sub: int, N: int, nx: int, C: int, R: int, nfl: int = NFL,
                          lim: int = 8) -> HadronicCase:
    """Exact-integer inputs in [-lim, lim]: every product and partial sum is exact in fp64, so any
    summation order must give bit-identical results."""
    rng = rng_for(7, T_FK, seed_sub)
    pairs = draw_pairs(rng_for(7, T_PAIRS, seed_sub), C, nfl)
    fk = rng.integers(-lim, lim + 1, size=(N, nx, nx, C)).astype(np.float64)
    f = rng.integers(-lim, lim + 1, size=(R, nfl, nx)).astype(np.float64)
    g = rng.integers(-lim, lim + 1, size=(N, R)).astype(np.float64)
    return HadronicCase(f"int-{seed_sub}", fk, pairs, f, g, nfl)

"""GPU-vs-oracle parity through the C-ABI (include/fkconv.h), element by element on seeded inputs.

Small and medium cases here; the BASELINE.json full-size configurations are in test_gpu_fullsize.py.
Tolerances: BASELINE.json north_star (fp64 1e-13, fp32 1e-5 of sum|terms|); exact-integer inputs must
match bit for bit in any summation order.
"""
import numpy as np
import pytest

from oracle import fk_oracle as O
from paper_1909_10547_b200 import synth
from tests._parity import TOL32, TOL64, rel_err, to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def K():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device (no CPU fallback exists)"
    from paper_1909_10547_b200 import fkconv
    return fkconv


def _tables(K, case, kind):
    """The same table through every storage path: stateless (logical), BORROW handle, PACK handle."""
    fk_d = to_dev(case.fk)
    idx = case.pairs if kind == K.FK_KIND_HADRONIC else case.flav
    tb = K.FkTable(kind, fk_d, idx, case.nfl, K.FK_F64, K.FK_STORE_BORROW)
    tp = K.FkTable(kind, fk_d, idx, case.nfl, K.FK_F64, K.FK_STORE_PACK)
    return fk_d, idx, tb, tp


# ------------------------------------------------------------------ config 0 and friends (hadronic)
@pytest.mark.parametrize("R", [1, 2, 3, 6])
def test_config0_forward_and_vjp(K, R):
    case = synth.config0(R=R)
    ref, scale = O.hadronic(case.fk, case.pairs, case.f)
    dref, D = O.hadronic_vjp(case.fk, case.pairs, case.f, case.g)
    fk_d, idx, tb, tp = _tables(K, case, K.FK_KIND_HADRONIC)
    f_d, g_d = to_dev(case.f), to_dev(case.g)
    outs = {
        "stateless": K.fk_conv_hadronic(fk_d, idx, f_d),
        "borrow": tb.conv(f_d),
        "pack": tp.conv(f_d),
    }
    for name, s in outs.items():
        assert rel_err(s.cpu().numpy(), ref, scale) <= TOL64, name
    # same layout, same plan, same partials, same order: the stateless call and the borrowing table give the same bits
    assert np.array_equal(outs["stateless"].cpu().numpy(), outs["borrow"].cpu().numpy())
    douts = {
        "stateless": K.fk_conv_hadronic_vjp(fk_d, idx, f_d, g_d),
        "borrow": tb.vjp(f_d, g_d),
        "pack": tp.vjp(f_d, g_d),
    }
    for name, d in douts.items():
        assert rel_err(d.cpu().numpy(), dref, D) <= TOL64, name


RAGGED = [  # (N, nx, nfl, C)  - odd nx / odd C (64-bit load path), N=1, C=1, K below one chunk, several chunks
    (1, 7, 14, 1), (37, 23, 14, 29), (5, 3, 3, 9), (130, 9, 5, 13), (33, 31, 14, 21), (64, 16, 14, 40),
    (3, 50, 14, 2), (300, 5, 2, 4),
]


@pytest.mark.parametrize("shape", RAGGED)
@pytest.mark.parametrize("R", [1, 5])
def test_ragged_shapes_hadronic(K, shape, R):
    N, nx, nfl, C = shape
    case = synth.hadronic_case(5, N, nx, C, R, nfl=nfl, sub=N * 1000 + nx)
    ref, scale = O.hadronic(case.fk, case.pairs, case.f)
    dref, D = O.hadronic_vjp(case.fk, case.pairs, case.f, case.g)
    fk_d, idx, tb, tp = _tables(K, case, K.FK_KIND_HADRONIC)
    f_d, g_d = to_dev(case.f), to_dev(case.g)
    for name, s in (("stateless", K.fk_conv_hadronic(fk_d, idx, f_d)), ("borrow", tb.conv(f_d)), ("pack", tp.conv(f_d))):
        assert rel_err(s.cpu().numpy(), ref, scale) <= TOL64, (name, shape)
    for name, d in (("stateless", K.fk_conv_hadronic_vjp(fk_d, idx, f_d, g_d)), ("borrow", tb.vjp(f_d, g_d)),
                    ("pack", tp.vjp(f_d, g_d))):
        assert rel_err(d.cpu().numpy(), dref, D) <= TOL64, (name, shape)
    # a flavour that appears in no pair gets exactly zero
    used = set(case.pairs[:, 0]) | set(case.pairs[:, 1])
    dn = tp.vjp(f_d, g_d).cpu().numpy()
    for a in range(nfl):
        if a not in used:
            assert np.all(dn[:, a, :] == 0.0)


# R >> 1 path: every fragment count of the warp-specialised DMMA kernels (replica passes are padded to 16),
# datapoint tiles of 128 / 64 / 32 rows (k sub-splits 1 / 2 / 4), K ranges that end inside a channel block
@pytest.mark.parametrize("R", [8, 17, 33, 49, 70, 81, 100, 113, 128, 150])
@pytest.mark.parametrize("shape", [(70, 13, 14, 17), (200, 30, 14, 9), (20, 21, 6, 5)])
def test_dense_path_replica_counts(K, shape, R):
    N, nx, nfl, C = shape
    case = synth.hadronic_case(6, N, nx, C, R, nfl=nfl, sub=N * 1000 + nx + R)
    # a general upstream gradient g[n][r] (reading R8), not the broadcast weights of config 4
    g = synth.rng_for(6, synth.T_G, 7 + R).standard_normal(size=(N, R))
    ref, scale = O.hadronic(case.fk, case.pairs, case.f)
    dref, D = O.hadronic_vjp(case.fk, case.pairs, case.f, g)
    fk_d, idx, tb, tp = _tables(K, case, K.FK_KIND_HADRONIC)
    f_d, g_d = to_dev(case.f), to_dev(g)
    for name, t in (("borrow", tb), ("pack", tp)):
        assert rel_err(t.conv(f_d).cpu().numpy(), ref, scale) <= TOL64, (name, shape, R)
        assert rel_err(t.vjp(f_d, g_d).cpu().numpy(), dref, D) <= TOL64, (name, shape, R)
    assert np.array_equal(tp.conv(f_d).cpu().numpy(), tp.conv(f_d).cpu().numpy())
    assert np.array_equal(tp.vjp(f_d, g_d).cpu().numpy(), tp.vjp(f_d, g_d).cpu().numpy())


@pytest.mark.parametrize("c", [0.3, 1.1])
def test_dense_vjp_same_sign_many_datapoints(K, c):
    """f = c, FK = 1, g = 1 with N = 10 000 datapoints at R = 8: the dense VJP contraction sums over ALL datapoints,
    and with one sign nothing cancels -- an unbounded register chain of N/4 DMMA steps misses 1e-13 here
    (the kernels flush every 512 datapoints).  Closed form: df[a][i] = N c nx (#{a_c = a} + #{b_c = a})."""
    from fractions import Fraction
    import torch
    N, nx, nfl, C, R = 10000, 8, 3, 4, 8
    pairs = np.array([(0, 1), (1, 1), (2, 0), (0, 0)], dtype=np.int32)
    fk_d = torch.ones((N, nx, nx, C), dtype=torch.float64, device="cuda")
    f = np.full((R, nfl, nx), c); g = np.ones((N, R))
    exact = np.zeros((R, nfl, nx))
    for a in range(nfl):
        cnt = int(np.sum(pairs[:, 0] == a) + np.sum(pairs[:, 1] == a))
        exact[:, a, :] = float(Fraction(c) * N * nx * cnt)
    for store in (K.FK_STORE_PACK, K.FK_STORE_BORROW):
        t = K.FkTable(K.FK_KIND_HADRONIC, fk_d, pairs, nfl, K.FK_F64, store, R_hint=R)
        df = t.vjp(to_dev(f), to_dev(g)).cpu().numpy()
        err = float(np.max(np.abs(df - exact) / exact))
        print(f"dense VJP same sign c={c} store={store}: {err:.2e}")
        assert err <= TOL64, (c, store, err)
        sig = t.conv(to_dev(f)).cpu().numpy()
        assert float(np.max(np.abs(sig - float(Fraction(c) ** 2 * nx * nx * C)) / float(Fraction(c) ** 2 * nx * nx * C))) <= TOL64
        t.destroy()


# x-grids beyond what the single-pass VJP folds hold (nx > 64 at R >> 1, nx > 128 at small R): gather fallbacks
@pytest.mark.parametrize("shape_R", [((12, 70, 3, 4), 6), ((12, 70, 3, 4), 1), ((6, 131, 2, 2), 1), ((6, 131, 2, 2), 5)])
def test_large_x_grids(K, shape_R):
    (N, nx, nfl, C), R = shape_R
    case = synth.hadronic_case(7, N, nx, C, R, nfl=nfl, sub=nx)
    ref, scale = O.hadronic(case.fk, case.pairs, case.f)
    dref, D = O.hadronic_vjp(case.fk, case.pairs, case.f, case.g)
    fk_d, idx, tb, tp = _tables(K, case, K.FK_KIND_HADRONIC)
    f_d, g_d = to_dev(case.f), to_dev(case.g)
    for name, t in (("borrow", tb), ("pack", tp)):
        assert rel_err(t.conv(f_d).cpu().numpy(), ref, scale) <= TOL64, (name, shape_R)
        assert rel_err(t.vjp(f_d, g_d).cpu().numpy(), dref, D) <= TOL64, (name, shape_R)


# forward + VJP from one read of FK (fk_table_conv_vjp)
@pytest.mark.parametrize("shape", RAGGED + [(512, 20, 14, 60)])
@pytest.mark.parametrize("R", [1, 2, 3, 4, 6])
def test_conv_vjp_one_read(K, shape, R):
    N, nx, nfl, C = shape
    case = synth.hadronic_case(8, N, nx, C, R, nfl=nfl, sub=N * 1000 + nx)
    g = synth.rng_for(8, synth.T_G, 11 + R).standard_normal(size=(N, R))
    ref, scale = O.hadronic(case.fk, case.pairs, case.f)
    dref, D = O.hadronic_vjp(case.fk, case.pairs, case.f, g)
    fk_d, idx, tb, tp = _tables(K, case, K.FK_KIND_HADRONIC)
    f_d, g_d = to_dev(case.f), to_dev(g)
    for name, t in (("borrow", tb), ("pack", tp)):
        sig, df = t.conv_vjp(f_d, g_d)
        assert rel_err(sig.cpu().numpy(), ref, scale) <= TOL64, (name, shape, R)
        assert rel_err(df.cpu().numpy(), dref, D) <= TOL64, (name, shape, R)
        sig2, df2 = t.conv_vjp(f_d, g_d)
        assert np.array_equal(sig.cpu().numpy(), sig2.cpu().numpy()) and np.array_equal(df.cpu().numpy(), df2.cpu().numpy())
    # the forward half is the same arithmetic as fk_table_conv: bit for bit
    assert np.array_equal(tp.conv_vjp(f_d, g_d)[0].cpu().numpy(), tp.conv(f_d).cpu().numpy())


def test_conv_vjp_one_read_dis_and_fp32(K):
    dis = synth.config1(R=2, N=300)
    rd, sd = O.dis(dis.fk, dis.flav, dis.f)
    g = synth.rng_for(8, synth.T_G, 3).standard_normal(size=(dis.N, 2))
    dref, D = O.dis_vjp(dis.fk, dis.flav, dis.f, g)
    t = K.FkTable(K.FK_KIND_DIS, to_dev(dis.fk), dis.flav, dis.nfl)
    sig, df = t.conv_vjp(to_dev(dis.f), to_dev(g))
    assert rel_err(sig.cpu().numpy(), rd, sd) <= TOL64 and rel_err(df.cpu().numpy(), dref, D) <= TOL64
    import torch
    case = synth.hadronic_case(8, 96, 24, 30, 2, sub=5)
    ref, scale = O.hadronic(case.fk, case.pairs, case.f)
    dref, D = O.hadronic_vjp(case.fk, case.pairs, case.f, case.g)
    t32 = K.FkTable(K.FK_KIND_HADRONIC, to_dev(case.fk), case.pairs, case.nfl, K.FK_F32)
    sig, df = t32.conv_vjp(to_dev(case.f, torch.float32), to_dev(case.g, torch.float32))
    assert rel_err(sig.cpu().numpy(), ref, scale) <= TOL32 and rel_err(df.cpu().numpy(), dref, D) <= TOL32


# ------------------------------------------------------------------ element-sparse storage
@pytest.mark.parametrize("zero_frac", [0.0, 0.3, 0.9, 1.0])
@pytest.mark.parametrize("shape_R", [((37, 23, 14, 29), 1), ((64, 50, 14, 9), 3), ((33, 8, 6, 5), 6), ((300, 30, 14, 40), 2)])
def test_sparse_storage_hadronic(K, shape_R, zero_frac):
    """FK_STORE_SPARSE: only the nonzero entries are stored (bit masks + packed values).  Same gates as the
    dense table against the oracle of the same (zero-riddled) table; a zero fraction of 1.0 is the empty table (sigma = 0,
    df = 0 exactly); the stored bytes follow the nonzero count; forward + VJP, one-read entry point, bitwise repeatable."""
    import torch
    (N, nx, nfl, C), R = shape_R
    case = synth.hadronic_case(8, N, nx, C, R, nfl=nfl, sub=N + 31 * nx)
    rng = synth.rng_for(8, synth.T_FK, 9000 + N + int(100 * zero_frac))
    fk = case.fk * (rng.random(size=case.fk.shape) >= zero_frac)
    if zero_frac == 0.3:   # structured zeros as well: a whole channel, a whole datapoint, a band of x-rows
        fk[..., 0] = 0.0; fk[N // 2] = 0.0; fk[:, nx // 2:, : nx // 3, :] = 0.0
    g = synth.rng_for(8, synth.T_G, 40 + N).standard_normal(size=(N, R))
    ref, scale = O.hadronic(fk, case.pairs, case.f)
    dref, D = O.hadronic_vjp(fk, case.pairs, case.f, g)
    ts = K.FkTable(K.FK_KIND_HADRONIC, to_dev(fk), case.pairs, case.nfl, K.FK_F64, K.FK_STORE_SPARSE, R_hint=R)
    f_d, g_d = to_dev(case.f), to_dev(g)
    sig, df = ts.conv(f_d), ts.vjp(f_d, g_d)
    assert rel_err(sig.cpu().numpy(), ref, scale) <= TOL64 and rel_err(df.cpu().numpy(), dref, D) <= TOL64
    assert torch.equal(sig, ts.conv(f_d)) and torch.equal(df, ts.vjp(f_d, g_d))
    s2, d2 = ts.conv_vjp(f_d, g_d)   # two passes on a sparse table, same results
    assert torch.equal(s2, sig) and torch.equal(d2, df)
    nnz = int(np.count_nonzero(fk))
    Kp = C * ((nx * nx + 3) // 4 * 4)
    stored = ts.info()["device_bytes"]
    assert stored >= 8 * nnz + N * ((Kp + 511) // 512) * 80 and stored <= 8 * nnz + N * ((Kp + 511) // 512) * 80 + (1 << 26)
    if zero_frac == 1.0:
        assert not sig.any() and not df.any()
    ts.destroy()


def test_sparse_storage_dis_config1(K):
    """BASELINE config 1 as given (30 % of the entries zeroed): the sparse table against the oracle and bit for bit
    repeatable; exact-integer inputs equal the oracle bit for bit in any order."""
    import torch
    for R in (1, 5):
        case = synth.config1(R=R)
        ref, scale = O.dis(case.fk, case.flav, case.f)
        dref, D = O.dis_vjp(case.fk, case.flav, case.f, case.g)
        ts = K.FkTable(K.FK_KIND_DIS, to_dev(case.fk), case.flav, case.nfl, K.FK_F64, K.FK_STORE_SPARSE, R_hint=R)
        f_d, g_d = to_dev(case.f), to_dev(case.g)
        assert rel_err(ts.conv(f_d).cpu().numpy(), ref, scale) <= TOL64
        assert rel_err(ts.vjp(f_d, g_d).cpu().numpy(), dref, D) <= TOL64
        stored = 8 * int(np.count_nonzero(case.fk)) + case.N * ((case.nx * case.nA + 511) // 512) * 80   # values + masks + headers
        frac = stored / case.fk.nbytes
        print(f"config 1 sparse R={R}: stored / dense bytes = {frac:.3f}")
        assert frac < 0.75 and stored <= ts.info()["device_bytes"] <= stored + (1 << 24)   # + scratch and staging
        ts.destroy()
    ic = synth.integer_hadronic_case(11, N=40, nx=17, C=12, R=2)
    fk = ic.fk * (synth.rng_for(7, synth.T_FK, 123).random(size=ic.fk.shape) >= 0.4)
    ref, _ = O.hadronic(fk, ic.pairs, ic.f)
    dref, _ = O.hadronic_vjp(fk, ic.pairs, ic.f, ic.g)
    ts = K.FkTable(K.FK_KIND_HADRONIC, to_dev(fk), ic.pairs, ic.nfl, K.FK_F64, K.FK_STORE_SPARSE)
    assert np.array_equal(ts.conv(to_dev(ic.f)).cpu().numpy(), ref)
    assert np.array_equal(ts.vjp(to_dev(ic.f), to_dev(ic.g)).cpu().numpy(), dref)
    with pytest.raises(RuntimeError):
        K.FkGroup([ts])
    ts.destroy()


# ------------------------------------------------------------------ two-PDF (p pbar) form
@pytest.mark.parametrize("shape_R", [((5, 6, 4, 7), 1), ((40, 17, 14, 30), 3), ((70, 30, 14, 60), 9)])
def test_two_pdf_form_against_the_oracle(K, shape_R):
    """fk_conv_hadronic2 / _vjp (Eq. (1), with distinct PDFs on the two legs) against the
    oracle's two-PDF loop.  The VJP is checked without any two-PDF derivative code on the oracle side: sigma is linear in
    f1 for fixed f2, so df1[r][alpha][i] = sum_n g[n][r] sigma(e_{alpha,i}, f2)[n][r] exactly (e = unit grid), and the same
    with the roles swapped for df2; the unit-grid sigmas come from the oracle.  R = 9 takes the dense contraction."""
    (N, nx, nfl, C), R = shape_R
    case = synth.hadronic_case(8, N, nx, C, R, nfl=nfl, sub=77 + N)
    rng = synth.rng_for(8, synth.T_PDF, 500 + N)
    f2 = case.f * rng.uniform(0.5, 1.5, size=case.f.shape) + 0.01 * rng.standard_normal(size=case.f.shape)
    g = synth.rng_for(8, synth.T_G, 600 + N).standard_normal(size=(N, R))
    ref, scale = O.hadronic(case.fk, case.pairs, case.f, f2=f2)
    fk_d, f1_d, f2_d, g_d = to_dev(case.fk), to_dev(case.f), to_dev(f2), to_dev(g)
    sig = K.fk_conv_hadronic2(fk_d, case.pairs, f1_d, f2_d).cpu().numpy()
    assert rel_err(sig, ref, scale) <= TOL64
    # swapping the legs is a different observable unless FK is symmetric: the entry point must not symmetrise
    swapped, _ = O.hadronic(case.fk, case.pairs, f2, f2=case.f)
    assert np.max(np.abs(swapped - ref)) > 1e-6 * np.max(np.abs(ref))
    df1, df2 = (t.cpu().numpy() for t in K.fk_conv_hadronic2_vjp(fk_d, case.pairs, f1_d, f2_d, g_d))
    used_a, used_b = sorted(set(int(a) for a in case.pairs[:, 0])), sorted(set(int(b) for b in case.pairs[:, 1]))
    for alpha in range(nfl):
        if alpha not in used_a:
            assert np.all(df1[:, alpha] == 0.0)
        if alpha not in used_b:
            assert np.all(df2[:, alpha] == 0.0)
    picks = [(used_a[0], 0), (used_a[-1], nx - 1), (used_a[len(used_a) // 2], nx // 2)]
    for (alpha, i) in picks:
        e = np.zeros_like(case.f); e[:, alpha, i] = 1.0
        s_e, sc_e = O.hadronic(case.fk, case.pairs, e, f2=f2)
        want, D = np.sum(g * s_e, axis=0), np.sum(np.abs(g) * sc_e, axis=0)
        assert np.max(np.abs(df1[:, alpha, i] - want) / np.maximum(D, 1e-300)) <= TOL64, (alpha, i)
    picks = [(used_b[0], 0), (used_b[-1], nx - 1), (used_b[len(used_b) // 2], nx // 3)]
    for (beta, j) in picks:
        e = np.zeros_like(case.f); e[:, beta, j] = 1.0
        s_e, sc_e = O.hadronic(case.fk, case.pairs, case.f, f2=e)
        want, D = np.sum(g * s_e, axis=0), np.sum(np.abs(g) * sc_e, axis=0)
        assert np.max(np.abs(df2[:, beta, j] - want) / np.maximum(D, 1e-300)) <= TOL64, (beta, j)
    # f1 = f2 = f reduces to the single-PDF entry points: forward bit for bit (same kernel, same order), df = df1 + df2
    s1 = K.fk_conv_hadronic2(fk_d, case.pairs, f1_d, f1_d).cpu().numpy()
    r1, sc1 = O.hadronic(case.fk, case.pairs, case.f)
    assert rel_err(s1, r1, sc1) <= TOL64
    d1, d2 = (t.cpu().numpy() for t in K.fk_conv_hadronic2_vjp(fk_d, case.pairs, f1_d, f1_d, g_d))
    dref, D = O.hadronic_vjp(case.fk, case.pairs, case.f, g)
    assert rel_err(d1 + d2, dref, np.maximum(D, 1e-300)) <= 2 * TOL64


# ------------------------------------------------------------------ config 1 (DIS)
@pytest.mark.parametrize("R", [1, 100])
def test_config1_dis(K, R):
    case = synth.config1(R=R)
    ref, scale = O.dis(case.fk, case.flav, case.f)
    dref, D = O.dis_vjp(case.fk, case.flav, case.f, case.g)
    fk_d, idx, tb, tp = _tables(K, case, K.FK_KIND_DIS)
    f_d, g_d = to_dev(case.f), to_dev(case.g)
    for name, s in (("stateless", K.fk_conv_dis(fk_d, idx, f_d)), ("borrow", tb.conv(f_d)), ("pack", tp.conv(f_d))):
        assert rel_err(s.cpu().numpy(), ref, scale) <= TOL64, name
    for name, d in (("stateless", K.fk_conv_dis_vjp(fk_d, idx, f_d, g_d)), ("borrow", tb.vjp(f_d, g_d)),
                    ("pack", tp.vjp(f_d, g_d))):
        assert rel_err(d.cpu().numpy(), dref, D) <= TOL64, name


@pytest.mark.parametrize("shape", [(1, 2, 1, 13), (63, 20, 3, 16), (64, 50, 9, 17), (65, 36, 14, 40), (200, 50, 9, 100),
                                   (130, 50, 10, 130), (2048, 50, 9, 100), (77, 8, 5, 300)])
def test_dis_direct_small_tables(K, shape):
    """Small packed DIS tables at R >= 13 (config 1 at R = 100) run in ONE launch (fk_dis_direct_kernel: both operands by bulk
    copies, no transposed f, no split-K partials).  Against the oracle, and against the general R >> 1 path that
    FK_OPT_DIS_DIRECT = 0 selects: ragged datapoint tiles, replica counts that are not multiples of 8 or 32, partial last
    k-stage, K up to 500."""
    N, nx, nA, R = shape
    rng = synth.rng_for(11, synth.T_FK, N * 1000 + R)
    fk = rng.standard_normal(size=(N, nx, nA))
    flav = synth.draw_flavours(synth.rng_for(11, synth.T_PAIRS, nA), nA)
    f = synth.pdf_grid(synth.pdf_params(synth.rng_for(11, synth.T_PDF, R), R), nx)
    ref, scale = O.dis(fk, flav, f)
    t = K.FkTable(K.FK_KIND_DIS, to_dev(fk), flav, synth.NFL, K.FK_F64, K.FK_STORE_PACK, R_hint=R)
    f_d = to_dev(f)
    default = K.get_option(K.FK_OPT_DIS_DIRECT)   # smallest R that takes the path (80: where it starts to win)
    try:
        K.set_option(K.FK_OPT_DIS_DIRECT, 13)
        s1 = t.conv(f_d).cpu().numpy()
        assert t.last_launches() == 1
        assert np.array_equal(s1, t.conv(f_d).cpu().numpy())   # repeatable bit for bit
        K.set_option(K.FK_OPT_DIS_DIRECT, 0)
        s0 = t.conv(f_d).cpu().numpy()
        assert t.last_launches() > 1
    finally:
        K.set_option(K.FK_OPT_DIS_DIRECT, default)
    assert rel_err(s1, ref, scale) <= TOL64
    assert rel_err(s0, ref, scale) <= TOL64
    t.conv(f_d)
    assert (t.last_launches() == 1) == (R >= default)
    t.destroy()


@pytest.mark.parametrize("shape_R", [((8, 3571, 1), 1), ((8, 3571, 1), 7), ((100, 1021, 1), 3), ((33, 2048, 1), 40),
                                     ((8, 5_000_000, 1), 1), ((5, 4_900_001, 1), 3)])  # the last two: fk_fwd_fewrows_kernel
def test_flat_matrix_view_of_table3(K, shape_R):
    """The paper's Table-3 operation: flat FK[N x K] . PDF[K x R] with a pre-built PDF matrix =
    the DIS convolution with one pseudo-flavour and nx = K (f = PDF^T)."""
    (N, Kc, nA), R = shape_R
    rng = synth.rng_for(9, synth.T_FK, Kc + R)
    fk = rng.standard_normal(size=(N, Kc, nA))
    f = rng.standard_normal(size=(R, 1, Kc))
    flav = np.zeros(1, dtype=np.int32)
    ref, scale = O.dis(fk, flav, f)
    t = K.FkTable(K.FK_KIND_DIS, to_dev(fk), flav, 1, K.FK_F64, K.FK_STORE_BORROW)
    assert rel_err(t.conv(to_dev(f)).cpu().numpy(), ref, scale) <= TOL64
    assert rel_err(K.fk_conv_dis(to_dev(fk), flav, to_dev(f)).cpu().numpy(), ref, scale) <= TOL64
    flat = fk.reshape(N, Kc) @ f.reshape(R, Kc).T  # library GEMM of the same flat view
    assert rel_err(t.conv(to_dev(f)).cpu().numpy(), flat, scale) <= 1e-12


def test_dis_small_unsorted_flavours(K):
    rng = np.random.default_rng(3)
    N, nx, nfl = 19, 11, 6
    flav = np.array([4, 0, 2], dtype=np.int32)
    fk = rng.standard_normal((N, nx, 3))
    f = rng.uniform(0.1, 2.0, (2, nfl, nx))
    ref, scale = O.dis(fk, flav, f)
    s = K.fk_conv_dis(to_dev(fk), flav, to_dev(f))
    assert rel_err(s.cpu().numpy(), ref, scale) <= TOL64


def test_dis_equals_hadronic_with_delta_flavour_on_gpu(K):
    """DIS = hadronic with a pseudo-flavour delta_j0 on the second leg; ties the two
    GPU kernels to each other end to end."""
    rng = np.random.default_rng(8)
    N, nx, nfl, nA = 40, 12, 5, 3
    flav = np.array([3, 1, 4], dtype=np.int32)
    fk_dis = rng.standard_normal((N, nx, nA))
    f = rng.uniform(0.1, 2.0, (2, nfl, nx))
    f_ext = np.zeros((2, nfl + 1, nx)); f_ext[:, :nfl] = f; f_ext[:, nfl, 0] = 1.0
    pairs = np.stack([flav, np.full(nA, nfl)], axis=1).astype(np.int32)
    fk_h = rng.standard_normal((N, nx, nx, nA)); fk_h[:, :, 0, :] = fk_dis
    s_dis = K.fk_conv_dis(to_dev(fk_dis), flav, to_dev(f)).cpu().numpy()
    s_had = K.fk_conv_hadronic(to_dev(fk_h), pairs, to_dev(f_ext)).cpu().numpy()
    _, scale = O.dis(fk_dis, flav, f)
    assert rel_err(s_had, s_dis, scale) <= TOL64


# ------------------------------------------------------------------ exact arithmetic and determinism
@pytest.mark.parametrize("shape", [(40, 12, 30, 1), (17, 25, 50, 3), (200, 9, 11, 5)])
def test_exact_integer_inputs_are_bitwise_equal(K, shape):
    N, nx, C, R = shape
    case = synth.integer_hadronic_case(N, N, nx, C, R)
    ref, _ = O.hadronic(case.fk, case.pairs, case.f)
    dref, _ = O.hadronic_vjp(case.fk, case.pairs, case.f, case.g)
    fk_d, idx, tb, tp = _tables(K, case, K.FK_KIND_HADRONIC)
    f_d, g_d = to_dev(case.f), to_dev(case.g)
    for s in (K.fk_conv_hadronic(fk_d, idx, f_d), tb.conv(f_d), tp.conv(f_d)):
        assert np.array_equal(s.cpu().numpy(), ref)
    for d in (K.fk_conv_hadronic_vjp(fk_d, idx, f_d, g_d), tb.vjp(f_d, g_d), tp.vjp(f_d, g_d)):
        assert np.array_equal(d.cpu().numpy(), dref)


def test_bitwise_repeatable_runs(K):
    case = synth.hadronic_case(6, 96, 30, 37, 2, sub=1)
    fk_d, idx, tb, tp = _tables(K, case, K.FK_KIND_HADRONIC)
    f_d, g_d = to_dev(case.f), to_dev(case.g)
    s0 = tp.conv(f_d).cpu().numpy(); d0 = tp.vjp(f_d, g_d).cpu().numpy()
    for _ in range(10):
        assert np.array_equal(tp.conv(f_d).cpu().numpy(), s0)
        assert np.array_equal(tp.vjp(f_d, g_d).cpu().numpy(), d0)


def test_replica_independence(K):
    """Column r of a batched call equals the R=1 call on replica r (within tolerance)."""
    case = synth.hadronic_case(6, 50, 20, 25, 7, sub=2)
    ref, scale = O.hadronic(case.fk, case.pairs, case.f)
    fk_d = to_dev(case.fk)
    batched = K.fk_conv_hadronic(fk_d, case.pairs, to_dev(case.f)).cpu().numpy()
    for r in range(case.R):
        one = K.fk_conv_hadronic(fk_d, case.pairs, to_dev(case.f[r:r + 1])).cpu().numpy()
        assert rel_err(one[:, 0], batched[:, r], scale[:, r]) <= 2 * TOL64


# ------------------------------------------------------------------ fp32 variant
@pytest.mark.parametrize("R", [1, 4])
def test_fp32_variant(K, R):
    import torch
    case = synth.hadronic_case(3, 64, 30, 40, R, sub=4)
    ref, scale = O.hadronic(case.fk, case.pairs, case.f)       # fp64 oracle of the fp64 inputs
    dref, D = O.hadronic_vjp(case.fk, case.pairs, case.f, case.g)
    f32 = torch.float32
    fk_d = to_dev(case.fk)
    s = K.fk_conv_hadronic(fk_d.to(f32), case.pairs, to_dev(case.f, f32))
    assert s.dtype == f32 and rel_err(s.cpu().numpy(), ref, scale) <= TOL32
    d = K.fk_conv_hadronic_vjp(fk_d.to(f32), case.pairs, to_dev(case.f, f32), to_dev(case.g, f32))
    assert rel_err(d.cpu().numpy(), dref, D) <= TOL32
    tp = K.FkTable(K.FK_KIND_HADRONIC, fk_d, case.pairs, case.nfl, K.FK_F32, K.FK_STORE_PACK)
    s2 = tp.conv(to_dev(case.f, f32))
    assert s2.dtype == f32 and rel_err(s2.cpu().numpy(), ref, scale) <= TOL32
    d2 = tp.vjp(to_dev(case.f, f32), to_dev(case.g, f32))
    assert rel_err(d2.cpu().numpy(), dref, D) <= TOL32


# fp32 variant at R >> 1: the tcgen05 (3xTF32) contraction.  Every padded replica count (multiples of 16), partial
# datapoint tiles (N % 128 != 0), K ranges that end inside a channel, x-grids from 8 to 50, a pass boundary at
# R > 128.  Gate: 1e-5 of sum|terms| against the fp64 oracle of the fp64 inputs (reading R18); printed next to the
# error of the fp32 column kernels on the same inputs.
@pytest.mark.parametrize("R", [9, 16, 33, 48, 70, 81, 100, 113, 128, 150])
@pytest.mark.parametrize("shape", [(70, 13, 14, 17), (200, 30, 14, 9), (300, 8, 6, 5), (129, 50, 14, 3)])
def test_tc32_dense_path_fp32_variant(K, shape, R):
    import torch
    N, nx, nfl, C = shape
    case = synth.hadronic_case(8, N, nx, C, R, nfl=nfl, sub=N * 1000 + nx + R)
    ref, scale = O.hadronic(case.fk, case.pairs, case.f)
    f32 = torch.float32
    tp = K.FkTable(K.FK_KIND_HADRONIC, to_dev(case.fk), case.pairs, case.nfl, K.FK_F32, K.FK_STORE_PACK, R_hint=R)
    f_d = to_dev(case.f, f32)
    s = tp.conv(f_d)
    nl = tp.last_launches()
    e_tc = rel_err(s.cpu().numpy(), ref, scale)
    K.set_option(K.FK_OPT_TC32, 0)
    try:
        s_col = tp.conv(f_d)
        nl_col = tp.last_launches()
    finally:
        K.set_option(K.FK_OPT_TC32, 1)
    e_col = rel_err(s_col.cpu().numpy(), ref, scale)
    print(f"tc32 {shape} R={R}: tcgen05 {e_tc:.2e} ({nl} launches)  column kernels {e_col:.2e} ({nl_col} launches)")
    assert nl == 3 * ((R + 127) // 128) and nl_col >= nl         # the tensor-core path really ran (transpose, contraction, reduce per pass)
    assert s.dtype == f32 and e_tc <= TOL32 and e_col <= TOL32
    assert torch.equal(s, tp.conv(f_d))                           # bitwise repeatable
    tp.destroy()


def test_tc32_same_sign_and_exact_small_integers(K):
    """Two pins of the 3xTF32 split itself.  (1) Integers in [-2, 2] are exact in TF32 and every partial sum is exact
    in fp32 (|sum| <= 2^24): the result must equal the oracle bit for bit.  (2) f = c, FK = 1 (closed form
    c^2 nx^2 C): all terms have one sign, so the truncation of the split and of the tensor core's
    accumulation cannot cancel -- the bounded TMEM chains keep it inside 1e-5."""
    from fractions import Fraction
    import torch
    f32 = torch.float32
    case = synth.integer_hadronic_case(9, N=150, nx=20, C=7, R=40, lim=2)
    ref, _ = O.hadronic(case.fk, case.pairs, case.f)
    tp = K.FkTable(K.FK_KIND_HADRONIC, to_dev(case.fk), case.pairs, case.nfl, K.FK_F32, K.FK_STORE_PACK, R_hint=40)
    s = tp.conv(to_dev(case.f, f32)).cpu().numpy()
    assert tp.last_launches() == 3 and np.array_equal(s.astype(np.float64), ref)
    tp.destroy()
    N, nx, C, nfl, R = 256, 50, 100, 14, 64
    pairs = synth.draw_pairs(synth.rng_for(2, synth.T_PAIRS, 0), C)
    fk_d = torch.ones((N, nx, nx, C), dtype=torch.float64, device="cuda")
    tp = K.FkTable(K.FK_KIND_HADRONIC, fk_d, pairs, nfl, K.FK_F32, K.FK_STORE_PACK, R_hint=R)
    for c in (0.3, 1.1):
        c32 = float(np.float32(c))                       # the fp32 variant demotes f (reading R18)
        exact = float(Fraction(c32) ** 2 * nx * nx * C)
        s = tp.conv(torch.full((R, nfl, nx), c32, dtype=f32, device="cuda")).cpu().numpy().astype(np.float64)
        err = float(np.max(np.abs(s - exact) / exact))
        print(f"tc32 same sign c={c}: {err:.2e}")
        assert tp.last_launches() == 3 and err <= TOL32
    tp.destroy()


# ------------------------------------------------------------------ launch-mode options change timing, never bits
def test_launch_options_do_not_change_results(K):
    """FK_OPT_PDL (programmatic dependent launch of the later kernels of a call) and FK_OPT_FUSE_L2 (small tables: the
    forward kernel's last CTA per datapoint range runs the level-2 reduction, one launch instead of two) only move
    work in time: every result must be bit for bit the same with the option off."""
    import torch
    c0 = synth.config0(R=2)
    big = synth.hadronic_case(8, 200, 30, 9, 2, nfl=14, sub=4)       # several k-blocks and several datapoint ranges
    c32 = synth.hadronic_case(8, 129, 50, 3, 40, nfl=14, sub=9)
    tabs = [(K.FkTable(K.FK_KIND_HADRONIC, to_dev(c.fk), c.pairs, c.nfl, K.FK_F64, K.FK_STORE_PACK, R_hint=2), c) for c in (c0, big)]
    t32 = K.FkTable(K.FK_KIND_HADRONIC, to_dev(c32.fk), c32.pairs, c32.nfl, K.FK_F32, K.FK_STORE_PACK, R_hint=40)
    grp = K.FkGroup([t for t, _ in tabs], R_hint=2)
    f_cat = torch.cat([to_dev(c.f).reshape(-1) for _, c in tabs])

    def run():
        out = []
        for t, c in tabs:
            out.append(t.conv(to_dev(c.f)))
            out.append(t.vjp(to_dev(c.f), to_dev(c.g)))
            out.append(torch.tensor([t.last_launches()]))
        out.append(grp.conv(f_cat, 2))
        out.append(t32.conv(to_dev(c32.f, torch.float32)))
        torch.cuda.synchronize()
        return out

    base = run()
    ref, scale = O.hadronic(c0.fk, c0.pairs, c0.f)
    assert rel_err(base[0].cpu().numpy(), ref, scale) <= TOL64
    for option in (K.FK_OPT_PDL, K.FK_OPT_FUSE_L2):
        K.set_option(option, 0)
        try:
            other = run()
        finally:
            K.set_option(option, 1)
        for i, (a, b) in enumerate(zip(base, other)):
            if a.numel() == 1 and a.dtype == torch.int64:
                continue   # launch counts differ by design
            assert torch.equal(a, b), (option, i)
    # config 0 (one wave of CTAs) really is a single forward launch with the in-kernel reduction, and two without it
    t0, c = tabs[0]
    t0.conv(to_dev(c.f)); n_fused = t0.last_launches()
    K.set_option(K.FK_OPT_FUSE_L2, 0)
    try:
        t0.conv(to_dev(c.f)); n_split = t0.last_launches()
    finally:
        K.set_option(K.FK_OPT_FUSE_L2, 1)
    assert (n_fused, n_split) == (1, 2)
    grp.destroy()


# ------------------------------------------------------------------ CUDA graphs
def test_calls_capture_into_a_cuda_graph(K):
    """Every compute call is asynchronous on the caller's stream, allocates nothing once its scratch is sized and
    synchronises nothing (include/fkconv.h): a fit iteration (forward, VJP, one-read step, grouped forward) must
    therefore capture into a CUDA graph -- programmatic dependent launches included -- and every replay must give
    the eager result bit for bit, also after the inputs changed in place."""
    import torch
    case = synth.hadronic_case(8, 96, 24, 30, 2, sub=77)
    dis = synth.config1(R=2, N=300)
    tp = K.FkTable(K.FK_KIND_HADRONIC, to_dev(case.fk), case.pairs, case.nfl, K.FK_F64, K.FK_STORE_PACK, R_hint=2)
    td = K.FkTable(K.FK_KIND_DIS, to_dev(dis.fk), dis.flav, dis.nfl, R_hint=2)
    t32 = K.FkTable(K.FK_KIND_HADRONIC, to_dev(case.fk), case.pairs, case.nfl, K.FK_F32, K.FK_STORE_PACK, R_hint=40)
    grp = K.FkGroup([tp, td], R_hint=2)
    f_d, g_d = to_dev(case.f), to_dev(case.g)
    fd_d = to_dev(dis.f)
    f40 = to_dev(np.ascontiguousarray(np.broadcast_to(case.f[:1], (40,) + case.f.shape[1:])), torch.float32)
    f_cat = torch.cat([f_d.reshape(-1), fd_d.reshape(-1)])
    sig, df = torch.empty((case.N, 2), dtype=torch.float64, device="cuda"), torch.empty_like(f_d)
    sig1, df1 = torch.empty_like(sig), torch.empty_like(df)
    sig_cat = torch.empty(int(grp.offsets(2)[1][-1]), dtype=torch.float64, device="cuda")
    sig40 = torch.empty((case.N, 40), dtype=torch.float32, device="cuda")

    def step():
        tp.conv(f_d, sig)
        tp.vjp(f_d, g_d, df)
        tp.conv_vjp(f_d, g_d, sig1, df1)
        grp.conv(f_cat, 2, sig_cat)
        t32.conv(f40, sig40)      # the tcgen05 contraction (TMA, tensor memory) inside the graph as well

    step()                        # sizes every scratch buffer outside the capture
    torch.cuda.synchronize()
    want = [t.clone() for t in (sig, df, sig1, df1, sig_cat, sig40)]
    graph = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    with torch.cuda.graph(graph, stream=side):
        step()
    for t in (sig, df, sig1, df1, sig_cat, sig40):
        t.zero_()
    graph.replay()
    torch.cuda.synchronize()
    for got, ref in zip((sig, df, sig1, df1, sig_cat, sig40), want):
        assert torch.equal(got, ref)
    f_d.mul_(1.25)                # new inputs in place: the graph reads the same buffers
    f_cat[: f_d.numel()] = f_d.reshape(-1)
    graph.replay()
    torch.cuda.synchronize()
    ref, scale = O.hadronic(case.fk, case.pairs, case.f * 1.25)
    assert rel_err(sig.cpu().numpy(), ref, scale) <= TOL64
    assert torch.equal(sig, sig1) and torch.equal(sig_cat[: sig.numel()].reshape(sig.shape), sig)
    # a handle refuses to grow its scratch inside a capture instead of allocating there
    g2 = torch.cuda.CUDAGraph()
    big = to_dev(np.ascontiguousarray(np.broadcast_to(case.f[:1], (64,) + case.f.shape[1:])))
    with pytest.raises(RuntimeError):
        with torch.cuda.graph(g2, stream=side):
            tp.conv(big)
    grp.destroy()


# ------------------------------------------------------------------ host-buffer calls
def test_host_buffer_calls(K):
    case = synth.hadronic_case(6, 48, 20, 30, 2, sub=5)
    ref, scale = O.hadronic(case.fk, case.pairs, case.f)
    dref, D = O.hadronic_vjp(case.fk, case.pairs, case.f, case.g)
    tp = K.FkTable(K.FK_KIND_HADRONIC, to_dev(case.fk), case.pairs, case.nfl)
    sig = np.empty((case.N, case.R)); df = np.empty_like(case.f)
    tp.conv_host(case.f, sig)
    tp.vjp_host(case.f, case.g, df)
    assert rel_err(sig, ref, scale) <= TOL64
    assert rel_err(df, dref, D) <= TOL64
    assert tp.last_launches() >= 2
    # forward + VJP in one host call (one copy in, one copy out, one wait): the one-read path, then the two passes
    for fused in (1, 0):
        K.set_option(K.FK_OPT_FUSED, fused)
        try:
            sig2 = np.full((case.N, case.R), np.nan); df2 = np.full_like(case.f, np.nan)
            tp.conv_vjp_host(case.f, case.g, sig2, df2)
        finally:
            K.set_option(K.FK_OPT_FUSED, 1)
        assert rel_err(sig2, ref, scale) <= TOL64 and rel_err(df2, dref, D) <= TOL64
        if not fused:
            assert np.array_equal(sig2, sig) and np.array_equal(df2, df)    # the same kernels as the two calls
    t32 = K.FkTable(K.FK_KIND_HADRONIC, to_dev(case.fk), case.pairs, case.nfl, K.FK_F32, K.FK_STORE_PACK)
    sig3 = np.empty((case.N, case.R), dtype=np.float32); df3 = np.empty(case.f.shape, dtype=np.float32)
    t32.conv_vjp_host(case.f.astype(np.float32), case.g.astype(np.float32), sig3, df3)
    assert rel_err(sig3, ref, scale) <= TOL32 and rel_err(df3, dref, D) <= TOL32


# ------------------------------------------------------------------ grouped ragged launch
@pytest.mark.parametrize("R", [1, 3, 6, 130])
@pytest.mark.parametrize("store", ["pack", "borrow"])
def test_grouped_small_ragged(K, R, store):
    import torch
    shapes = synth.small_ragged_shapes(T=7)
    params = synth.pdf_params(synth.rng_for(4, synth.T_PDF), R)
    cases = [synth.config4_table(t, shapes, R, params) for t in range(shapes.T)]
    st = K.FK_STORE_PACK if store == "pack" else K.FK_STORE_BORROW
    keep = [to_dev(c.fk) for c in cases]
    tabs = [K.FkTable(K.FK_KIND_HADRONIC, keep[t], cases[t].pairs, cases[t].nfl, K.FK_F64, st) for t in range(shapes.T)]
    grp = K.FkGroup(tabs, R_hint=R)
    fo, so = grp.offsets(R)
    f_cat = torch.cat([to_dev(c.f).reshape(-1) for c in cases])
    g_cat = torch.cat([to_dev(c.g).reshape(-1) for c in cases])
    assert f_cat.numel() == fo[-1] and g_cat.numel() == so[-1]
    sig = grp.conv(f_cat, R).cpu().numpy()
    df = grp.vjp(f_cat, g_cat, R).cpu().numpy()
    for t, c in enumerate(cases):
        ref, scale = O.hadronic(c.fk, c.pairs, c.f)
        dref, D = O.hadronic_vjp(c.fk, c.pairs, c.f, c.g)
        assert rel_err(sig[so[t]:so[t + 1]].reshape(c.N, R), ref, scale) <= TOL64, t
        assert rel_err(df[fo[t]:fo[t + 1]].reshape(R, c.nfl, c.nx), dref, D) <= TOL64, t
    # repeatable
    assert np.array_equal(grp.conv(f_cat, R).cpu().numpy(), sig)
    assert np.array_equal(grp.vjp(f_cat, g_cat, R).cpu().numpy(), df)
    assert grp.last_launches() >= 2


@pytest.mark.parametrize("R", [1, 2, 4, 6])
@pytest.mark.parametrize("store", ["pack", "borrow"])
def test_grouped_conv_vjp_one_read(K, R, store):
    """fk_conv_grouped_conv_vjp: forward and VJP of a ragged group from one read of every table when g
    is known before the forward pass (config 4's seeded weights).  R <= 4: the fused column kernel over the group's
    static CTA list (3 launches + 1 per extra replica tile); R = 6: the two passes.  sigma is bit for bit the
    grouped forward's; df meets the same 1e-13 gate against the oracle."""
    import torch
    shapes = synth.small_ragged_shapes(T=7)
    params = synth.pdf_params(synth.rng_for(4, synth.T_PDF), R)
    cases = [synth.config4_table(t, shapes, R, params) for t in range(shapes.T)]
    st = K.FK_STORE_PACK if store == "pack" else K.FK_STORE_BORROW
    keep = [to_dev(c.fk) for c in cases]
    tabs = [K.FkTable(K.FK_KIND_HADRONIC, keep[t], cases[t].pairs, cases[t].nfl, K.FK_F64, st) for t in range(shapes.T)]
    grp = K.FkGroup(tabs, R_hint=R)
    fo, so = grp.offsets(R)
    f_cat = torch.cat([to_dev(c.f).reshape(-1) for c in cases])
    rng = synth.rng_for(8, synth.T_G, 50 + R)
    gs = [rng.standard_normal(size=(c.N, R)) for c in cases]     # a general g[n][r], not the broadcast weights
    g_cat = torch.cat([to_dev(g).reshape(-1) for g in gs])
    sig_d, df_d = grp.conv_vjp(f_cat, g_cat, R)
    nl = grp.last_launches()
    assert nl == (4 if R <= 4 else nl) and (R > 4 or nl == 4)   # fused column + reduce + fold + final
    sig, df = sig_d.cpu().numpy(), df_d.cpu().numpy()
    for t, c in enumerate(cases):
        ref, scale = O.hadronic(c.fk, c.pairs, c.f)
        dref, D = O.hadronic_vjp(c.fk, c.pairs, c.f, gs[t])
        assert rel_err(sig[so[t]:so[t + 1]].reshape(c.N, R), ref, scale) <= TOL64, t
        assert rel_err(df[fo[t]:fo[t + 1]].reshape(R, c.nfl, c.nx), dref, np.maximum(D, 1e-300)) <= TOL64, t
    assert np.array_equal(sig, grp.conv(f_cat, R).cpu().numpy())
    sig2, df2 = grp.conv_vjp(f_cat, g_cat, R)
    assert torch.equal(sig2, sig_d) and torch.equal(df2, df_d)   # bitwise repeatable
    grp.destroy()


@pytest.mark.parametrize("R", [2, 9])
def test_grouped_mixed_dis_and_hadronic(K, R):
    """A 'global' group: DIS and hadronic tables in one launch; R=9 takes the
    grouped R >> 1 contraction."""
    import torch
    h = synth.hadronic_case(6, 30, 12, 17, R, sub=7)
    d = synth.config1(R=R, N=200)
    th = K.FkTable(K.FK_KIND_HADRONIC, to_dev(h.fk), h.pairs, h.nfl)
    td = K.FkTable(K.FK_KIND_DIS, to_dev(d.fk), d.flav, d.nfl)
    grp = K.FkGroup([th, td], R_hint=R)
    fo, so = grp.offsets(R)
    f_cat = torch.cat([to_dev(h.f).reshape(-1), to_dev(d.f).reshape(-1)])
    g_cat = torch.cat([to_dev(h.g).reshape(-1), to_dev(d.g).reshape(-1)])
    sig = grp.conv(f_cat, R).cpu().numpy()
    df = grp.vjp(f_cat, g_cat, R).cpu().numpy()
    ref_h, sc_h = O.hadronic(h.fk, h.pairs, h.f); ref_d, sc_d = O.dis(d.fk, d.flav, d.f)
    assert rel_err(sig[so[0]:so[1]].reshape(h.N, R), ref_h, sc_h) <= TOL64
    assert rel_err(sig[so[1]:so[2]].reshape(d.N, R), ref_d, sc_d) <= TOL64
    dref_h, D_h = O.hadronic_vjp(h.fk, h.pairs, h.f, h.g); dref_d, D_d = O.dis_vjp(d.fk, d.flav, d.f, d.g)
    assert rel_err(df[fo[0]:fo[1]].reshape(R, h.nfl, h.nx), dref_h, D_h) <= TOL64
    assert rel_err(df[fo[1]:fo[2]].reshape(R, d.nfl, d.nx), dref_d, D_d) <= TOL64


# ------------------------------------------------------------------ error paths on a live device
def test_error_paths_on_device(K):
    case = synth.hadronic_case(6, 4, 5, 3, 1, sub=9)
    fk_d, f_d = to_dev(case.fk), to_dev(case.f)
    bad = case.pairs.copy(); bad[1, 0] = case.nfl
    with pytest.raises(K.FkError) as e:
        K.fk_conv_hadronic(fk_d, bad, f_d)
    assert e.value.code == K.FK_ERR_INVALID_ARG
    with pytest.raises(K.FkError):
        K.FkTable(K.FK_KIND_HADRONIC, fk_d, bad, case.nfl)
    with pytest.raises(K.FkError):
        K.FkTable(K.FK_KIND_HADRONIC, fk_d, case.pairs, case.nfl, K.FK_F32, K.FK_STORE_BORROW)


# ------------------------------------------------------------------ chi2 and the fit step (reading R22)
def _spd(rng, N):
    a = rng.standard_normal(size=(N, N))
    return a @ a.T / N + np.eye(N)


@pytest.mark.parametrize("N_R", [(1, 1), (7, 3), (100, 1), (257, 9), (512, 128)])
def test_chi2_against_oracle(K, N_R):
    N, R = N_R
    rng = synth.rng_for(10, synth.T_G, N + R)
    sigma, data, cinv = rng.standard_normal(size=(N, R)), rng.standard_normal(size=N), _spd(rng, N)
    c, cs, g, gs = O.chi2(sigma, data, cinv)
    cd, gd = K.fk_chi2(to_dev(sigma), to_dev(data), to_dev(cinv))
    assert rel_err(cd.cpu().numpy(), c, cs) <= TOL64
    assert rel_err(gd.cpu().numpy(), g, gs) <= TOL64
    # exact integers: bit for bit
    si = rng.integers(-8, 9, size=(N, R)).astype(np.float64); di = rng.integers(-8, 9, size=N).astype(np.float64)
    ci = rng.integers(-3, 4, size=(N, N)).astype(np.float64); ci = ci + ci.T
    c, _, g, _ = O.chi2(si, di, ci)
    cd, gd = K.fk_chi2(to_dev(si), to_dev(di), to_dev(ci))
    assert np.array_equal(cd.cpu().numpy(), c) and np.array_equal(gd.cpu().numpy(), g)


@pytest.mark.parametrize("R", [1, 3, 20])
def test_fit_step_is_the_three_calls(K, R):
    case = synth.hadronic_case(11, 70, 16, 25, R, sub=R)
    rng = synth.rng_for(11, synth.T_G, 99)
    data, cinv = rng.standard_normal(size=case.N) * 10, _spd(rng, case.N)
    t = K.FkTable(K.FK_KIND_HADRONIC, to_dev(case.fk), case.pairs, case.nfl)
    f_d, data_d, cinv_d = to_dev(case.f), to_dev(data), to_dev(cinv)
    sig, chi2, g, df = t.fit_step(f_d, data_d, cinv_d)
    s2 = t.conv(f_d); c2, g2 = K.fk_chi2(s2, data_d, cinv_d); d2 = t.vjp(f_d, g2)
    for a, b in ((sig, s2), (chi2, c2), (g, g2), (df, d2)):
        assert np.array_equal(a.cpu().numpy(), b.cpu().numpy())
    # every stage against the oracle on the inputs that stage saw
    ref, scale = O.hadronic(case.fk, case.pairs, case.f)
    assert rel_err(sig.cpu().numpy(), ref, scale) <= TOL64
    c, cs, go, gs = O.chi2(sig.cpu().numpy(), data, cinv)
    assert rel_err(chi2.cpu().numpy(), c, cs) <= TOL64 and rel_err(g.cpu().numpy(), go, gs) <= TOL64
    dref, D = O.hadronic_vjp(case.fk, case.pairs, case.f, g.cpu().numpy())
    assert rel_err(df.cpu().numpy(), dref, D) <= TOL64


def test_sharded_table_single_rank(K):
    """ShardedFkTable at world size 1 (the only size one GPU allows; world size 2 runs on CPU with gloo,
    tests/test_sharded_cpu.py): the rank's slice is the whole table, no collective is issued."""
    from paper_1909_10547_b200 import sharded
    case = synth.hadronic_case(12, 37, 9, 11, 3, sub=4)
    ref, scale = O.hadronic(case.fk, case.pairs, case.f)
    dref, D = O.hadronic_vjp(case.fk, case.pairs, case.f, case.g)
    t = sharded.ShardedFkTable(K.FK_KIND_HADRONIC, case.fk, case.pairs, case.nfl)
    assert (t.n0, t.n1) == (0, case.N)
    assert rel_err(t.conv_all(to_dev(case.f)).cpu().numpy(), ref, scale) <= TOL64
    assert rel_err(t.vjp(to_dev(case.f), to_dev(case.g)).cpu().numpy(), dref, D) <= TOL64


# ------------------------------------------------------------------ fp32-stored table, fp64 everything else
TOL32S = 1e-7  # each FK value carries one fp32 rounding (2^-24 = 6e-8 of its term); f, g and all sums are fp64


@pytest.mark.parametrize("shape", [(37, 23, 14, 29), (130, 9, 5, 13), (3, 50, 14, 2), (512, 20, 14, 60)])
@pytest.mark.parametrize("R", [1, 3, 6, 20])
def test_fp32_storage_fp64_arithmetic(K, shape, R):
    N, nx, nfl, C = shape
    case = synth.hadronic_case(13, N, nx, C, R, nfl=nfl, sub=N + nx)
    g = synth.rng_for(13, synth.T_G, R).standard_normal(size=(N, R))
    ref, scale = O.hadronic(case.fk, case.pairs, case.f)
    dref, D = O.hadronic_vjp(case.fk, case.pairs, case.f, g)
    t = K.FkTable(K.FK_KIND_HADRONIC, to_dev(case.fk), case.pairs, case.nfl, K.FK_F32S64)
    assert t.info()["device_bytes"] < 0.6 * case.fk.nbytes + (1 << 20)
    f_d, g_d = to_dev(case.f), to_dev(g)
    sig, df = t.conv(f_d), t.vjp(f_d, g_d)
    assert sig.dtype == df.dtype and str(sig.dtype) == "torch.float64"
    e1, e2 = rel_err(sig.cpu().numpy(), ref, scale), rel_err(df.cpu().numpy(), dref, D)
    assert e1 <= TOL32S and e2 <= TOL32S, (e1, e2)
    s2, d2 = t.conv_vjp(f_d, g_d)
    assert rel_err(s2.cpu().numpy(), ref, scale) <= TOL32S and rel_err(d2.cpu().numpy(), dref, D) <= TOL32S
    # against the oracle of the DEMOTED table the fp64 bar holds: the only difference is the storage rounding
    fk32 = case.fk.astype(np.float32).astype(np.float64)
    ref32, scale32 = O.hadronic(fk32, case.pairs, case.f)
    dref32, D32 = O.hadronic_vjp(fk32, case.pairs, case.f, g)
    assert rel_err(sig.cpu().numpy(), ref32, scale32) <= TOL64 and rel_err(df.cpu().numpy(), dref32, D32) <= TOL64


# fp32-STORED tables at R >> 1: the VJP is the FP64 tensor-core contraction G = FK^T g over the table as stored (widened
# in the fragment loads) + the fp64 fold; launches: transpose, pad, contraction, fold (+ final) per pass of <= 128
# replicas.  FK_F32S64 (f, g, df fp64) meets the fp64 bar against the oracle of the DEMOTED table; FK_F32 (everything
# fp32 outside the contraction) meets the fp32 bar.  x-grids that need the padded x-row pitch (13), partial tiles,
# a pass boundary (150), DIS tables (gather instead of fold).
@pytest.mark.parametrize("R", [9, 40, 128, 150])
@pytest.mark.parametrize("shape", [(70, 13, 14, 17), (200, 30, 14, 9), (33, 50, 14, 3), (129, 8, 6, 5)])
def test_fp32_stored_tables_dense_vjp(K, shape, R):
    import torch
    N, nx, nfl, C = shape
    case = synth.hadronic_case(21, N, nx, C, R, nfl=nfl, sub=N * 100 + nx + R)
    g = synth.rng_for(21, synth.T_G, R).standard_normal(size=(N, R))
    fk32 = case.fk.astype(np.float32).astype(np.float64)
    dref, D = O.hadronic_vjp(case.fk, case.pairs, case.f, g)
    dref32, D32 = O.hadronic_vjp(fk32, case.pairs, case.f, g)
    passes = (R + 127) // 128
    f32 = torch.float32
    for dtype, ft, tol_paper, tol_stored in ((K.FK_F32S64, torch.float64, TOL32S, TOL64), (K.FK_F32, f32, TOL32, TOL32)):
        t = K.FkTable(K.FK_KIND_HADRONIC, to_dev(case.fk), case.pairs, case.nfl, dtype, K.FK_STORE_PACK, R_hint=R)
        f_d, g_d = to_dev(case.f, ft), to_dev(g, ft)
        df = t.vjp(f_d, g_d)
        nl = t.last_launches()
        assert df.dtype == ft and nl == 5 * passes, nl
        e, es = rel_err(df.cpu().numpy(), dref, D), rel_err(df.cpu().numpy(), dref32, D32)
        K.set_option(K.FK_OPT_GEMM_MIN_R, 1 << 20)
        try:
            dcol = t.vjp(f_d, g_d)
            nl_col = t.last_launches()
        finally:
            K.set_option(K.FK_OPT_GEMM_MIN_R, 0)
        ec = rel_err(dcol.cpu().numpy(), dref, D)
        print(f"stored32 vjp {shape} R={R} dtype={dtype}: dense {e:.2e} / {es:.2e} vs demoted ({nl} launches)  column {ec:.2e} ({nl_col})")
        assert e <= tol_paper and es <= tol_stored and ec <= tol_paper and nl_col >= nl and (R < 40 or nl_col > nl)
        assert torch.equal(df, t.vjp(f_d, g_d))
        if dtype == K.FK_F32S64:   # forward: the warp-specialised FP64 contraction over the fp32 tiles (3 launches per pass)
            ref32, scale32 = O.hadronic(fk32, case.pairs, case.f)
            sig = t.conv(f_d)
            nl = t.last_launches()
            es = rel_err(sig.cpu().numpy(), ref32, scale32)
            print(f"stored32 fwd {shape} R={R}: dense {es:.2e} vs demoted ({nl} launches)")
            assert nl == 3 * passes and es <= TOL64 and torch.equal(sig, t.conv(f_d))
            s2, d2 = t.conv_vjp(f_d, g_d)
            assert torch.equal(s2, sig) and torch.equal(d2, df)
        t.destroy()


def test_fp32_stored_dis_table_dense_vjp(K):
    import torch
    case = synth.config1(R=60, N=300)
    g = synth.rng_for(22, synth.T_G, 60).standard_normal(size=(300, 60))
    fk32 = case.fk.astype(np.float32).astype(np.float64)
    dref32, D32 = O.dis_vjp(fk32, case.flav, case.f, g)
    for dtype, ft, tol in ((K.FK_F32S64, torch.float64, TOL64), (K.FK_F32, torch.float32, TOL32)):
        t = K.FkTable(K.FK_KIND_DIS, to_dev(case.fk), case.flav, case.nfl, dtype, K.FK_STORE_PACK, R_hint=60)
        df = t.vjp(to_dev(case.f, ft), to_dev(g, ft))
        assert t.last_launches() == 4, t.last_launches()
        assert rel_err(df.cpu().numpy(), dref32, D32) <= tol
        t.destroy()


def test_fp32_storage_grouped_and_dis(K):
    import torch
    shapes = synth.small_ragged_shapes(T=5)
    R = 2
    params = synth.pdf_params(synth.rng_for(4, synth.T_PDF), R)
    cases = [synth.config4_table(t, shapes, R, params) for t in range(shapes.T)]
    tabs = [K.FkTable(K.FK_KIND_HADRONIC, to_dev(c.fk), c.pairs, c.nfl, K.FK_F32S64) for c in cases]
    grp = K.FkGroup(tabs, R_hint=R)
    fo, so = grp.offsets(R)
    f_cat = torch.cat([to_dev(c.f).reshape(-1) for c in cases]); g_cat = torch.cat([to_dev(c.g).reshape(-1) for c in cases])
    sig, df = grp.conv(f_cat, R).cpu().numpy(), grp.vjp(f_cat, g_cat, R).cpu().numpy()
    for t, c in enumerate(cases):
        ref, scale = O.hadronic(c.fk, c.pairs, c.f)
        dref, D = O.hadronic_vjp(c.fk, c.pairs, c.f, c.g)
        assert rel_err(sig[so[t]:so[t + 1]].reshape(c.N, R), ref, scale) <= TOL32S
        assert rel_err(df[fo[t]:fo[t + 1]].reshape(R, c.nfl, c.nx), dref, D) <= TOL32S
    dis = synth.config1(R=3, N=200)
    rd, sd = O.dis(dis.fk, dis.flav, dis.f)
    dd, DD = O.dis_vjp(dis.fk, dis.flav, dis.f, dis.g)
    td = K.FkTable(K.FK_KIND_DIS, to_dev(dis.fk), dis.flav, dis.nfl, K.FK_F32S64)
    assert rel_err(td.conv(to_dev(dis.f)).cpu().numpy(), rd, sd) <= TOL32S
    assert rel_err(td.vjp(to_dev(dis.f), to_dev(dis.g)).cpu().numpy(), dd, DD) <= TOL32S


@pytest.mark.parametrize("R", [20, 100])
def test_grouped_dense_tile_heights(K, R):
    """Grouped R >> 1 launch over tables whose last datapoint tile takes every height: 128 (97..128 rows left),
    64 + 32 (65..96), 64 (33..64), 32 (<= 32), and none (N a multiple of 128)."""
    import torch
    shapes = synth.RaggedShapes(np.array([70, 96, 200, 129, 64, 97, 128, 257]), np.array([6, 9, 7, 5, 11, 8, 6, 5]),
                                np.array([5, 3, 7, 9, 4, 6, 8, 10]))
    params = synth.pdf_params(synth.rng_for(4, synth.T_PDF), R)
    cases = [synth.config4_table(t, shapes, R, params) for t in range(shapes.T)]
    gs = [synth.rng_for(4, synth.T_G, 100 + t).standard_normal(size=(c.N, R)) for t, c in enumerate(cases)]
    tabs = [K.FkTable(K.FK_KIND_HADRONIC, to_dev(c.fk), c.pairs, c.nfl) for c in cases]
    grp = K.FkGroup(tabs, R_hint=R)
    fo, so = grp.offsets(R)
    f_cat = torch.cat([to_dev(c.f).reshape(-1) for c in cases]); g_cat = torch.cat([to_dev(g).reshape(-1) for g in gs])
    sig, df = grp.conv(f_cat, R).cpu().numpy(), grp.vjp(f_cat, g_cat, R).cpu().numpy()
    for t, c in enumerate(cases):
        ref, scale = O.hadronic(c.fk, c.pairs, c.f)
        dref, D = O.hadronic_vjp(c.fk, c.pairs, c.f, gs[t])
        assert rel_err(sig[so[t]:so[t + 1]].reshape(c.N, R), ref, scale) <= TOL64, t
        assert rel_err(df[fo[t]:fo[t + 1]].reshape(R, c.nfl, c.nx), dref, D) <= TOL64, t
    assert np.array_equal(grp.conv(f_cat, R).cpu().numpy(), sig)


def test_grouped_fp32_variant(K):
    """The fp32 variant (reading R18) through the grouped launch, against the fp64 oracle of the fp64 inputs."""
    import torch
    shapes = synth.small_ragged_shapes(T=5)
    R = 3
    params = synth.pdf_params(synth.rng_for(4, synth.T_PDF), R)
    cases = [synth.config4_table(t, shapes, R, params) for t in range(shapes.T)]
    tabs = [K.FkTable(K.FK_KIND_HADRONIC, to_dev(c.fk), c.pairs, c.nfl, K.FK_F32) for c in cases]
    grp = K.FkGroup(tabs, R_hint=R)
    fo, so = grp.offsets(R)
    f_cat = torch.cat([to_dev(c.f, torch.float32).reshape(-1) for c in cases])
    g_cat = torch.cat([to_dev(c.g, torch.float32).reshape(-1) for c in cases])
    sig, df = grp.conv(f_cat, R).cpu().numpy(), grp.vjp(f_cat, g_cat, R).cpu().numpy()
    assert sig.dtype == np.float32
    for t, c in enumerate(cases):
        ref, scale = O.hadronic(c.fk, c.pairs, c.f)
        dref, D = O.hadronic_vjp(c.fk, c.pairs, c.f, c.g)
        assert rel_err(sig[so[t]:so[t + 1]].reshape(c.N, R), ref, scale) <= TOL32, t
        assert rel_err(df[fo[t]:fo[t + 1]].reshape(R, c.nfl, c.nx), dref, D) <= TOL32, t
    grp.destroy()


@pytest.mark.parametrize("R", [20, 130])
def test_grouped_fp32_variant_tensor_cores(K, R):
    """The fp32 variant of a ragged group at R >> 1: ONE tcgen05 launch per pass of <= 128 replicas over static items
    (table, 128-datapoint tile, range of (c, i) rows) of about equal cost; tables of 1..400 datapoints and x-grids from 7 to
    50 points (partial tiles, K extents of one and two TMA boxes) against the fp64 oracle at 1e-5; equal to the
    single-table calls bit for bit only where the plans coincide, so compared through the oracle."""
    import torch
    shapes = synth.RaggedShapes(np.array([1, 37, 130, 400, 64, 257], dtype=np.int64), np.array([7, 23, 50, 30, 32, 44], dtype=np.int64),
                                np.array([1, 29, 12, 9, 20, 5], dtype=np.int64))
    params = synth.pdf_params(synth.rng_for(4, synth.T_PDF), R)
    cases = [synth.config4_table(t, shapes, R, params) for t in range(shapes.T)]
    tabs = [K.FkTable(K.FK_KIND_HADRONIC, to_dev(c.fk), c.pairs, c.nfl, K.FK_F32, R_hint=R) for c in cases]
    grp = K.FkGroup(tabs, R_hint=R)
    fo, so = grp.offsets(R)
    f_cat = torch.cat([to_dev(c.f, torch.float32).reshape(-1) for c in cases])
    sig_d = grp.conv(f_cat, R)
    assert grp.last_launches() == 3 * ((R + 127) // 128)     # transpose, contraction, reduce per pass
    sig = sig_d.cpu().numpy()
    worst = 0.0
    for t, c in enumerate(cases):
        ref, scale = O.hadronic(c.fk, c.pairs, c.f)
        worst = max(worst, rel_err(sig[so[t]:so[t + 1]].reshape(c.N, R), ref, scale))
    print(f"grouped tcgen05 R={R}: {worst:.2e}")
    assert sig.dtype == np.float32 and worst <= TOL32
    assert torch.equal(sig_d, grp.conv(f_cat, R))
    grp.destroy()


@pytest.mark.parametrize("R", [20, 130])
def test_grouped_fp32_stored_tables_dense_paths(K, R):
    """Groups of fp32-STORED tables at R >> 1: FK_F32S64 runs both FP64 contractions over the tables as stored (3 and 5
    launches per pass of <= 128 replicas) and meets the fp64 bar against the oracle of the DEMOTED tables; FK_F32 takes
    the same VJP (fp32 f, g, df) at the fp32 bar.  Ragged: 1..400 datapoints, x-grids 7..50 (padded x-rows for FK_F32)."""
    import torch
    shapes = synth.RaggedShapes(np.array([1, 37, 130, 400, 64, 257], dtype=np.int64), np.array([7, 23, 50, 30, 32, 44], dtype=np.int64),
                                np.array([1, 29, 12, 9, 20, 5], dtype=np.int64))
    params = synth.pdf_params(synth.rng_for(4, synth.T_PDF), R)
    cases = [synth.config4_table(t, shapes, R, params) for t in range(shapes.T)]
    gs = [synth.rng_for(23, synth.T_G, t).standard_normal(size=(c.N, R)) for t, c in enumerate(cases)]
    passes = (R + 127) // 128
    for dtype, ft, tol in ((K.FK_F32S64, torch.float64, TOL64), (K.FK_F32, torch.float32, TOL32)):
        tabs = [K.FkTable(K.FK_KIND_HADRONIC, to_dev(c.fk), c.pairs, c.nfl, dtype, R_hint=R) for c in cases]
        grp = K.FkGroup(tabs, R_hint=R)
        fo, so = grp.offsets(R)
        f_cat = torch.cat([to_dev(c.f, ft).reshape(-1) for c in cases])
        g_cat = torch.cat([to_dev(g, ft).reshape(-1) for g in gs])
        df_d = grp.vjp(f_cat, g_cat, R)
        assert grp.last_launches() == 5 * passes, grp.last_launches()
        df = df_d.cpu().numpy()
        worst = 0.0
        for t, c in enumerate(cases):
            fk32 = c.fk.astype(np.float32).astype(np.float64)
            dref, D = O.hadronic_vjp(fk32, c.pairs, c.f, gs[t])
            worst = max(worst, rel_err(df[fo[t]:fo[t + 1]].reshape(c.f.shape), dref, D))
        print(f"grouped stored32 vjp R={R} dtype={dtype}: {worst:.2e} vs demoted")
        assert worst <= tol and torch.equal(df_d, grp.vjp(f_cat, g_cat, R))
        if dtype == K.FK_F32S64:
            sig_d = grp.conv(f_cat, R)
            assert grp.last_launches() == 3 * passes, grp.last_launches()
            sig = sig_d.cpu().numpy()
            worst = 0.0
            for t, c in enumerate(cases):
                ref, scale = O.hadronic(c.fk.astype(np.float32).astype(np.float64), c.pairs, c.f)
                worst = max(worst, rel_err(sig[so[t]:so[t + 1]].reshape(c.N, R), ref, scale))
            print(f"grouped stored32 fwd R={R}: {worst:.2e} vs demoted")
            assert worst <= TOL64 and torch.equal(sig_d, grp.conv(f_cat, R))
            s2, d2 = grp.conv_vjp(f_cat, g_cat, R)
            assert torch.equal(s2, sig_d) and torch.equal(d2, df_d)
        grp.destroy()

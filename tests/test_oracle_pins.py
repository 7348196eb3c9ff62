"""Pins for the CPU oracle (oracle/fk_oracle.c) against what the paper and the mathematics fix.

The paper prints no worked example with inputs (Table 1, gives outputs only), so
the oracle is pinned by: exact-rational brute force, one-hot / separable tables (index conventions),
closed forms (counting), exact-integer arithmetic, bilinearity, DIS as a hadronic special case, the
numpy GEMM view of Table 3, and for the gradient central differences, Euler's
identity and closed forms.  None of these re-types the oracle's own loop.
"""
from fractions import Fraction

import numpy as np
import pytest

from oracle import fk_oracle as O
from paper_1909_10547_b200 import synth

U = 2.0 ** -53


def _rand_case(seed, N=3, nx=4, nfl=3, C=5, R=2):
    rng = np.random.default_rng(seed)
    pairs = synth.draw_pairs(rng, C, nfl)
    fk = rng.standard_normal((N, nx, nx, C))
    f = rng.uniform(0.1, 2.0, (R, nfl, nx))
    g = rng.standard_normal((N, R))
    return fk, pairs, f, g


# ---------------------------------------------------------------- brute force, exact rationals
def test_brute_force_fraction_hadronic_and_vjp():
    """Eq. (1) enumerated term by term in exact rational arithmetic on a tiny table with
    ALL ordered pairs active (so (a,b) vs (b,a) and a==b are all exercised)."""
    N, nx, nfl, R = 2, 3, 3, 2
    rng = np.random.default_rng(11)
    pairs = np.array([(a, b) for a in range(nfl) for b in range(nfl)], dtype=np.int32)
    C = len(pairs)
    fk = rng.standard_normal((N, nx, nx, C))
    f = rng.uniform(0.1, 2.0, (R, nfl, nx))
    g = rng.standard_normal((N, R))
    sigma, scale = O.hadronic(fk, pairs, f)
    df, D = O.hadronic_vjp(fk, pairs, f, g)
    F = lambda v: Fraction(float(v))
    for r in range(R):
        dref = [[Fraction(0)] * nx for _ in range(nfl)]
        Dref = [[Fraction(0)] * nx for _ in range(nfl)]
        for n in range(N):
            acc = Fraction(0); S = Fraction(0)
            for c, (a, b) in enumerate(pairs):
                for i in range(nx):
                    for j in range(nx):
                        t = F(f[r, a, i]) * F(f[r, b, j]) * F(fk[n, i, j, c])
                        acc += t; S += abs(t)
                        ta = F(g[n, r]) * F(fk[n, i, j, c]) * F(f[r, b, j])
                        tb = F(g[n, r]) * F(fk[n, i, j, c]) * F(f[r, a, i])
                        dref[a][i] += ta; Dref[a][i] += abs(ta)
                        dref[b][j] += tb; Dref[b][j] += abs(tb)
            assert abs(Fraction(float(sigma[n, r])) - acc) <= 2 * U * S
            assert abs(Fraction(float(scale[n, r])) - S) <= 4 * U * S
        for a in range(nfl):
            for i in range(nx):
                assert abs(Fraction(float(df[r, a, i])) - dref[a][i]) <= 2 * U * Dref[a][i]
                # the VJP tolerance denominator itself (reading R21): D = sum |g FK f| over every term of the slot
                assert abs(Fraction(float(D[r, a, i])) - Dref[a][i]) <= 4 * U * Dref[a][i]


def test_brute_force_fraction_dis():
    N, nx, nfl, nA, R = 3, 4, 5, 3, 2
    rng = np.random.default_rng(5)
    flav = np.array([4, 0, 2], dtype=np.int32)          # deliberately unsorted
    fk = rng.standard_normal((N, nx, nA))
    f = rng.uniform(0.1, 2.0, (R, nfl, nx))
    g = rng.standard_normal((N, R))
    sigma, scale = O.dis(fk, flav, f)
    df, D = O.dis_vjp(fk, flav, f, g)
    F = lambda v: Fraction(float(v))
    for r in range(R):
        for n in range(N):
            acc = sum(F(f[r, flav[c], i]) * F(fk[n, i, c]) for c in range(nA) for i in range(nx))
            S = sum(abs(F(f[r, flav[c], i]) * F(fk[n, i, c])) for c in range(nA) for i in range(nx))
            assert abs(F(sigma[n, r]) - acc) <= 2 * U * S
            assert abs(F(scale[n, r]) - S) <= 4 * U * S          # the DIS tolerance denominator
        for a in range(nfl):
            for i in range(nx):
                ref = sum(F(g[n, r]) * F(fk[n, i, c]) for n in range(N) for c in range(nA) if flav[c] == a)
                Dref = sum(abs(F(g[n, r]) * F(fk[n, i, c])) for n in range(N) for c in range(nA) if flav[c] == a)
                assert abs(F(df[r, a, i]) - ref) <= 2 * U * Dref
                assert abs(F(D[r, a, i]) - Dref) <= 4 * U * Dref   # the DIS-VJP tolerance denominator
                if a not in flav:
                    assert df[r, a, i] == 0.0


# ---------------------------------------------------------------- index conventions
def test_one_hot_fk_pins_axes():
    """A single 1 at (n0,i0,j0,c0) => sigma[n0] = f[a_c0][i0] * f[b_c0][j0] (one rounding), all others 0.
    i0 != j0 and a != b, so an i/j transposition or an a/b swap changes the value."""
    N, nx, nfl, C = 4, 6, 5, 7
    rng = np.random.default_rng(3)
    pairs = np.array([(0, 1), (1, 0), (2, 4), (4, 2), (3, 3), (0, 4), (2, 1)], dtype=np.int32)
    f = rng.uniform(0.1, 2.0, (1, nfl, nx))
    for (n0, i0, j0, c0) in [(2, 1, 4, 2), (0, 5, 0, 3), (3, 2, 3, 6)]:
        fk = np.zeros((N, nx, nx, C)); fk[n0, i0, j0, c0] = 1.0
        sigma, _ = O.hadronic(fk, pairs, f)
        a, b = pairs[c0]
        expect = np.zeros((N, 1)); expect[n0, 0] = f[0, a, i0] * f[0, b, j0]
        assert np.array_equal(sigma, expect)
        assert f[0, a, i0] * f[0, b, j0] != f[0, b, i0] * f[0, a, j0]
        assert f[0, a, i0] * f[0, b, j0] != f[0, a, j0] * f[0, b, i0]


def test_separable_fk_closed_form():
    """FK = u_n p_i q_j s_c => sigma_n = u_n sum_c s_c (sum_i p_i f[a_c][i]) (sum_j q_j f[b_c][j])."""
    N, nx, nfl, C = 5, 9, 6, 11
    rng = np.random.default_rng(8)
    pairs = synth.draw_pairs(rng, C, nfl)
    u, p, q, s = rng.standard_normal(N), rng.standard_normal(nx), rng.standard_normal(nx), rng.standard_normal(C)
    fk = np.einsum("n,i,j,c->nijc", u, p, q, s)
    f = rng.uniform(0.1, 2.0, (2, nfl, nx))
    sigma, scale = O.hadronic(fk, pairs, f)
    for r in range(2):
        P = f[r] @ p; Q = f[r] @ q
        ref = u * sum(s[c] * P[pairs[c, 0]] * Q[pairs[c, 1]] for c in range(C))
        assert np.max(np.abs(sigma[:, r] - ref) / scale[:, r]) < 50 * U
    # the transposed reading (i<->b, j<->a) gives a different number
    wrong = u * sum(s[c] * (f[0] @ p)[pairs[c, 1]] * (f[0] @ q)[pairs[c, 0]] for c in range(C))
    assert np.max(np.abs(sigma[:, 0] - wrong) / scale[:, 0]) > 1e-6


# ---------------------------------------------------------------- closed forms / counting
@pytest.mark.parametrize("c", [0.5, 1.5, 0.3])
def test_closed_form_constant_pdf(c):
    """f == c, FK == 1 => sigma_n = c^2 nx^2 C (BASELINE north_star); exact for dyadic c."""
    N, nx, nfl = 3, 20, 14
    pairs = np.array([(a, b) for a in range(nfl) for b in range(nfl)], dtype=np.int32)
    C = len(pairs)
    fk = np.ones((N, nx, nx, C)); f = np.full((1, nfl, nx), c)
    sigma, scale = O.hadronic(fk, pairs, f)
    expect = c * c * nx * nx * C
    if c in (0.5, 1.5):
        assert np.all(sigma == expect) and np.all(scale == expect)
    else:   # K = 78400 same-sign terms: the long-double accumulator keeps this at the ulp level
        # accumulator bound: K additions rounded to 64 bits, then one rounding to double; far below 1e-13
        exact = Fraction(c) ** 2 * nx * nx * C
        bound = nx * nx * C * 2.0 ** -64 + 2 * U
        assert bound < 1e-14
        assert all(abs(Fraction(float(v)) - exact) / exact < bound for v in sigma.ravel())
    # DIS: c * nx * nA
    s2, _ = O.dis(np.ones((N, nx, 9)), np.arange(9, dtype=np.int32), f)
    exact = Fraction(c) * nx * 9
    assert all(abs(Fraction(float(v)) - exact) / exact < 2 * U for v in s2.ravel())


def test_closed_form_large_K_same_sign():
    """K = 250 000 same-sign terms (config-2 row shape): sequential fp64 misses 1e-13 here
    (SURVEY 8(c).5); the oracle must not."""
    nx, nfl, C = 50, 14, 100
    pairs = synth.draw_pairs(np.random.default_rng(0), C, nfl)
    fk = np.ones((1, nx, nx, C)); f = np.full((1, nfl, nx), 0.7)
    sigma, _ = O.hadronic(fk, pairs, f)
    expect = Fraction(0.7) ** 2 * nx * nx * C
    bound = nx * nx * C * 2.0 ** -64 + 2 * U          # 1.4e-14: 7x below the 1e-13 parity gate
    assert abs(Fraction(float(sigma[0, 0])) - expect) / expect < bound < 1.5e-14


def test_vjp_closed_form_and_diagonal():
    """f==c, FK==1, g==1 => df[a][i] = N c nx (#{c: a_c=a} + #{c: b_c=a}); (a,a) one-hot at i==j gives 2 g f."""
    N, nx, nfl, c = 4, 7, 5, 1.5
    pairs = np.array([(0, 1), (1, 1), (2, 0), (0, 0), (3, 1)], dtype=np.int32)   # flavour 4 in no pair
    C = len(pairs)
    df, _ = O.hadronic_vjp(np.ones((N, nx, nx, C)), pairs, np.full((1, nfl, nx), c), np.ones((N, 1)))
    for a in range(nfl):
        cnt = int(np.sum(pairs[:, 0] == a) + np.sum(pairs[:, 1] == a))
        assert np.all(df[0, a] == N * c * nx * cnt)
    assert np.all(df[0, 4] == 0.0)
    f = np.random.default_rng(2).uniform(0.1, 2, (1, nfl, nx))
    fk = np.zeros((1, nx, nx, 1)); fk[0, 3, 3, 0] = 1.0
    df, _ = O.hadronic_vjp(fk, np.array([(2, 2)], dtype=np.int32), f, np.array([[0.75]]))
    expect = np.zeros_like(f); expect[0, 2, 3] = 2 * 0.75 * f[0, 2, 3]
    assert np.array_equal(df, expect)


# ---------------------------------------------------------------- exact integers
def test_exact_integer_inputs_match_int64():
    """Integers in [-8,8]: all products and sums exact => oracle equals int64 einsum bit for bit."""
    case = synth.integer_hadronic_case(1, N=5, nx=8, C=12, R=3, nfl=6)
    sigma, scale = O.hadronic(case.fk, case.pairs, case.f)
    fi, ki = case.f.astype(np.int64), case.fk.astype(np.int64)
    A = fi[:, case.pairs[:, 0], :]; B = fi[:, case.pairs[:, 1], :]
    ref = np.einsum("rci,rcj,nijc->nr", A, B, ki)
    assert np.array_equal(sigma, ref.astype(np.float64))
    refabs = np.einsum("rci,rcj,nijc->nr", np.abs(A), np.abs(B), np.abs(ki))
    assert np.array_equal(scale, refabs.astype(np.float64))


def test_exact_integer_denominators_match_int64():
    """The tolerance denominators every GPU gate divides by (reading R21) are exact sums of
    integers here, so they must equal an int64 abs-einsum bit for bit: D of the hadronic VJP (scatter of
    |g FK f| onto both legs), D of the DIS VJP and scale of the DIS forward.  A denominator inflated or deflated
    by any factor fails this."""
    case = synth.integer_hadronic_case(2, N=5, nx=8, C=12, R=3, nfl=6)
    fi, ki, gi = np.abs(case.f.astype(np.int64)), np.abs(case.fk.astype(np.int64)), np.abs(case.g.astype(np.int64))
    df, D = O.hadronic_vjp(case.fk, case.pairs, case.f, case.g)
    Gabs = np.einsum("nr,nijc->rijc", gi, ki)                     # |g| |FK| summed over datapoints
    Dref = np.zeros(case.f.shape, dtype=np.int64)
    dref = np.zeros(case.f.shape, dtype=np.int64)
    Gs = np.einsum("nr,nijc->rijc", case.g.astype(np.int64), case.fk.astype(np.int64))
    fs = case.f.astype(np.int64)
    for c, (a, b) in enumerate(case.pairs):
        Dref[:, a, :] += np.einsum("rij,rj->ri", Gabs[..., c], fi[:, b, :])
        Dref[:, b, :] += np.einsum("rij,ri->rj", Gabs[..., c], fi[:, a, :])
        dref[:, a, :] += np.einsum("rij,rj->ri", Gs[..., c], fs[:, b, :])
        dref[:, b, :] += np.einsum("rij,ri->rj", Gs[..., c], fs[:, a, :])
    assert np.array_equal(D, Dref.astype(np.float64)) and np.array_equal(df, dref.astype(np.float64))
    assert Dref.max() > 0 and np.any(Dref != np.abs(dref))        # cancellation: D is not |df|
    # DIS: forward scale and VJP denominator
    rng = synth.rng_for(7, synth.T_FK, 5)
    N, nx, nfl, nA, R = 6, 9, 7, 4, 3
    flav = np.array([5, 1, 6, 2], dtype=np.int32)
    fkd = rng.integers(-8, 9, size=(N, nx, nA)).astype(np.float64)
    f = rng.integers(-8, 9, size=(R, nfl, nx)).astype(np.float64)
    g = rng.integers(-8, 9, size=(N, R)).astype(np.float64)
    s, sc = O.dis(fkd, flav, f)
    ka, fa, ga = np.abs(fkd.astype(np.int64)), np.abs(f.astype(np.int64)), np.abs(g.astype(np.int64))
    assert np.array_equal(sc, np.einsum("nic,rci->nr", ka, fa[:, flav, :]).astype(np.float64))
    assert np.array_equal(s, np.einsum("nic,rci->nr", fkd.astype(np.int64), f.astype(np.int64)[:, flav, :]).astype(np.float64))
    dfd, Dd = O.dis_vjp(fkd, flav, f, g)
    Dref = np.zeros((R, nfl, nx), dtype=np.int64); dref = np.zeros((R, nfl, nx), dtype=np.int64)
    for c, a in enumerate(flav):
        Dref[:, a, :] += np.einsum("nr,ni->ri", ga, ka[:, :, c])
        dref[:, a, :] += np.einsum("nr,ni->ri", g.astype(np.int64), fkd.astype(np.int64)[:, :, c])
    assert np.array_equal(Dd, Dref.astype(np.float64)) and np.array_equal(dfd, dref.astype(np.float64))


# ---------------------------------------------------------------- algebraic structure
def test_bilinearity_and_fk_linearity():
    fk, pairs, f, _ = _rand_case(21, N=4, nx=6, nfl=5, C=9, R=2)
    h = np.random.default_rng(22).uniform(-1, 1, f.shape)
    lam = 0.375
    s_ff, sc = O.hadronic(fk, pairs, f)
    s_hh, _ = O.hadronic(fk, pairs, h)
    s_fh, _ = O.hadronic(fk, pairs, f, h)
    s_hf, _ = O.hadronic(fk, pairs, h, f)
    s_mix, sc2 = O.hadronic(fk, pairs, f + lam * h)
    ref = s_ff + lam * (s_fh + s_hf) + lam * lam * s_hh
    assert np.max(np.abs(s_mix - ref) / sc2) < 100 * U
    assert np.max(np.abs(s_fh - s_hf) / sc) > 1e-6          # pairs are ordered: not symmetric
    fk2 = np.random.default_rng(23).standard_normal(fk.shape)
    s2, sc3 = O.hadronic(fk2, pairs, f)
    s12, _ = O.hadronic(fk + 2.0 * fk2, pairs, f)
    assert np.max(np.abs(s12 - (s_ff + 2.0 * s2)) / (sc + 2 * sc3)) < 100 * U


def test_channel_permutation_and_replica_independence():
    fk, pairs, f, _ = _rand_case(31, N=3, nx=5, nfl=4, C=8, R=3)
    perm = np.random.default_rng(32).permutation(8)
    s, sc = O.hadronic(fk, pairs, f)
    s_p, _ = O.hadronic(fk[..., perm], pairs[perm], f)
    assert np.max(np.abs(s - s_p) / sc) < 8 * U
    for r in range(3):
        s_r, _ = O.hadronic(fk, pairs, f[r:r + 1])
        assert np.array_equal(s_r[:, 0], s[:, r])


def test_duplicate_pair_counts_twice():
    """Reading R4: the channel list is taken literally."""
    fk, pairs, f, _ = _rand_case(41, C=3)
    fk[..., 2] = fk[..., 0]; pairs[2] = pairs[0]
    s, sc = O.hadronic(fk, pairs, f)
    fk2 = fk[..., :2].copy(); fk2[..., 0] *= 2
    s2, _ = O.hadronic(fk2, pairs[:2], f)
    assert np.max(np.abs(s - s2) / sc) < 8 * U


# ---------------------------------------------------------------- DIS
def test_dis_is_hadronic_special_case():
    """Add a pseudo-flavour delta with f_delta[j] = [j == 0]; channels (flav_c, delta);
    FK_h[n][i][0][c] = FK_dis[n][i][c], arbitrary values at j != 0 => sigma_h == sigma_dis."""
    N, nx, nfl, nA, R = 6, 7, 5, 3, 2
    rng = np.random.default_rng(51)
    flav = synth.draw_flavours(rng, nA, nfl)
    fkd = rng.standard_normal((N, nx, nA))
    f = rng.uniform(0.1, 2.0, (R, nfl, nx))
    fh = np.zeros((R, nfl + 1, nx)); fh[:, :nfl] = f; fh[:, nfl, 0] = 1.0
    fkh = rng.standard_normal((N, nx, nx, nA)); fkh[:, :, 0, :] = fkd
    pairs = np.stack([flav, np.full(nA, nfl)], axis=1).astype(np.int32)
    s_d, sc_d = O.dis(fkd, flav, f)
    s_h, _ = O.hadronic(fkh, pairs, fh)
    assert np.array_equal(s_d, s_h)


def test_dis_is_textbook_gemv():
    c = synth.config1(R=2, N=64)
    L = c.f[:, c.flav, :].transpose(2, 1, 0).reshape(c.nx * c.nA, 2)      # [(i,c)][r]
    ref = c.fk.reshape(c.N, -1) @ L
    s, sc = O.dis(c.fk, c.flav, c.f)
    assert np.max(np.abs(s - ref) / sc) < 100 * U


# ---------------------------------------------------------------- flat GEMM view (Table 3)
def test_flat_gemm_view_matches_numpy():
    c = synth.hadronic_case(0, N=8, nx=20, C=49, R=3, name="table3-like")
    A = c.f[:, c.pairs[:, 0], :]; B = c.f[:, c.pairs[:, 1], :]
    L = np.einsum("rci,rcj->ijcr", A, B).reshape(-1, 3)                     # K x R, K = nx*nx*C
    ref = c.fk.reshape(c.N, -1) @ L
    s, sc = O.hadronic(c.fk, c.pairs, c.f)
    assert np.max(np.abs(s - ref) / sc) < 200 * U


# ---------------------------------------------------------------- gradient
def test_vjp_central_difference_is_exact_for_bilinear_form():
    fk, pairs, f, g = _rand_case(61, N=4, nx=5, nfl=4, C=7, R=1)
    df, D = O.hadronic_vjp(fk, pairs, f, g)

    def J(fx):
        s, _ = O.hadronic(fk, pairs, fx)
        return float(np.sum(g * s))
    h = 1e-3
    s0, sc0 = O.hadronic(fk, pairs, f)
    for (a, i) in [(0, 0), (1, 3), (3, 4), (2, 2)]:
        e = np.zeros_like(f); e[0, a, i] = h
        fd = (J(f + e) - J(f - e)) / (2 * h)
        assert abs(fd - df[0, a, i]) <= 1e-11 * max(D[0, a, i], 1.0)


def test_vjp_euler_identity():
    """sigma is homogeneous of degree 2 in f: sum f df = 2 sum g sigma (DIS: degree 1)."""
    c = synth.hadronic_case(0, N=6, nx=12, C=30, R=3)
    g = np.random.default_rng(71).standard_normal((c.N, c.R))
    s, sc = O.hadronic(c.fk, c.pairs, c.f)
    df, D = O.hadronic_vjp(c.fk, c.pairs, c.f, g)
    for r in range(c.R):
        lhs = np.sum(c.f[r] * df[r]); rhs = 2 * np.sum(g[:, r] * s[:, r])
        assert abs(lhs - rhs) <= 1e-13 * np.sum(np.abs(c.f[r]) * D[r])
    d = synth.config1(R=2, N=32)
    sd, _ = O.dis(d.fk, d.flav, d.f)
    dfd, Dd = O.dis_vjp(d.fk, d.flav, d.f, d.g)
    for r in range(2):
        assert abs(np.sum(d.f[r] * dfd[r]) - np.sum(d.g[:, r] * sd[:, r])) <= 1e-13 * np.sum(np.abs(d.f[r]) * Dd[r])


def test_vjp_matches_einsum():
    fk, pairs, f, g = _rand_case(81, N=5, nx=6, nfl=5, C=10, R=2)
    df, D = O.hadronic_vjp(fk, pairs, f, g)
    ref = np.zeros_like(f)
    G = np.einsum("nr,nijc->rijc", g, fk)
    for c, (a, b) in enumerate(pairs):
        ref[:, a, :] += np.einsum("rij,rj->ri", G[..., c], f[:, b, :])
        ref[:, b, :] += np.einsum("rij,ri->rj", G[..., c], f[:, a, :])
    assert np.max(np.abs(df - ref) / np.maximum(D, 1e-300)) < 200 * U


# ---------------------------------------------------------------- error behaviour
def test_invalid_arguments_rejected():
    fk, pairs, f, g = _rand_case(91)
    bad = pairs.copy(); bad[0, 1] = 3
    with pytest.raises(ValueError):
        O.hadronic(fk, bad, f)
    with pytest.raises(ValueError):
        O.hadronic_vjp(fk, bad, f, g)
    with pytest.raises(ValueError):
        O.dis(np.ones((2, 4, 2)), np.array([0, -1], dtype=np.int32), f)


# ------------------------------------------------------------------ chi2 of the fit step (reading R22)
def _spd(rng, N):
    a = rng.standard_normal(size=(N, N))
    return a @ a.T / N + np.eye(N)


def test_chi2_identity_covariance_exact_integers():
    """Cinv = 1: chi2 = sum d^2 and g = 2 d, exact for integer inputs."""
    rng = np.random.default_rng(7)
    N, R = 23, 3
    sigma = rng.integers(-8, 9, size=(N, R)).astype(np.float64)
    data = rng.integers(-8, 9, size=N).astype(np.float64)
    c, cs, g, gs = O.chi2(sigma, data, np.eye(N))
    d = sigma - data[:, None]
    assert np.array_equal(c, (d * d).sum(axis=0)) and np.array_equal(g, 2 * d)
    assert np.array_equal(cs, c) and np.array_equal(gs, 2 * np.abs(d))


def test_chi2_brute_force_fractions():
    rng = np.random.default_rng(8)
    N, R = 3, 2
    sigma = rng.integers(-5, 6, size=(N, R)) / 4.0
    data = rng.integers(-5, 6, size=N) / 8.0
    cinv = rng.integers(-4, 5, size=(N, N)) / 2.0
    cinv = cinv + cinv.T
    c, _, g, _ = O.chi2(sigma, data, cinv)
    F = Fraction
    for r in range(R):
        d = [F(sigma[n, r]) - F(data[n]) for n in range(N)]
        tot = sum(d[n] * F(cinv[n, m]) * d[m] for n in range(N) for m in range(N))
        assert c[r] == float(tot)
        for n in range(N):
            assert g[n, r] == float(2 * sum(F(cinv[n, m]) * d[m] for m in range(N)))


def test_chi2_matches_numpy_quadratic_form_and_euler_identity():
    rng = np.random.default_rng(9)
    N, R = 61, 4
    sigma, data, cinv = rng.standard_normal(size=(N, R)), rng.standard_normal(size=N), _spd(rng, N)
    c, cs, g, gs = O.chi2(sigma, data, cinv)
    d = sigma - data[:, None]
    ref = np.einsum("nr,nm,mr->r", d, cinv, d)
    assert np.all(np.abs(c - ref) <= 1e-14 * cs)
    assert np.all(np.abs(g - 2 * cinv @ d) <= 1e-14 * gs)
    # chi2 is homogeneous of degree 2 in d: sum_n g_n d_n = 2 chi2
    assert np.all(np.abs((g * d).sum(axis=0) - 2 * c) <= 1e-13 * cs)


def test_chi2_gradient_is_the_central_difference():
    """A quadratic form has no third derivative: the central difference is exact up to rounding for any h."""
    rng = np.random.default_rng(10)
    N = 17
    sigma, data, cinv = rng.standard_normal(size=(N, 1)), rng.standard_normal(size=N), _spd(rng, N)
    _, cs, g, _ = O.chi2(sigma, data, cinv)
    h = 1e-3
    for n in (0, 5, 16):
        e = np.zeros((N, 1)); e[n] = h
        cp = O.chi2(sigma + e, data, cinv)[0][0]; cm = O.chi2(sigma - e, data, cinv)[0][0]
        assert abs((cp - cm) / (2 * h) - g[n, 0]) <= 1e-15 * cs[0] / h + 1e-12 * abs(g[n, 0])  # rounding of chi2 / h


def test_oracle_matches_its_committed_golden_file():
    """tests/golden/oracle_tiny.json is written by tests/golden/make_golden.py (oracle only): guards against silent
    drift of the oracle or of the seeded generators."""
    import importlib.util
    import json
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(here, "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    with open(os.path.join(here, "oracle_tiny.json")) as fh:
        stored = json.load(fh)
    assert mod.build() == stored


# ------------------------------------------------------------------ property tests on random small shapes
def test_random_shapes_algebraic_properties():
    """Seeded sweep over small random shapes: linearity in FK, degree-2 homogeneity in f, invariance under a
    permutation of the channel list together with FK's channel axis, replica independence, and the numpy einsum
    of the flat view -- a wrong index, stride or bound in the oracle breaks one of them at some shape."""
    rng = np.random.default_rng(20260001)
    for _ in range(25):
        N, nx, nfl = int(rng.integers(1, 6)), int(rng.integers(1, 8)), int(rng.integers(1, 6))
        C = int(rng.integers(1, nfl * nfl + 1))
        R = int(rng.integers(1, 4))
        pairs = synth.draw_pairs(rng, C, nfl)
        fk, fk2 = rng.standard_normal((N, nx, nx, C)), rng.standard_normal((N, nx, nx, C))
        f = rng.standard_normal((R, nfl, nx))
        s1, sc1 = O.hadronic(fk, pairs, f)
        s2, sc2 = O.hadronic(fk2, pairs, f)
        s12, _ = O.hadronic(fk + 2.0 * fk2, pairs, f)
        tol = 4e-16 * (sc1 + 2 * sc2)
        assert np.all(np.abs(s12 - (s1 + 2.0 * s2)) <= tol + 1e-300)
        s3, _ = O.hadronic(fk, pairs, 3.0 * f)
        assert np.all(np.abs(s3 - 9.0 * s1) <= 4e-15 * sc1 + 1e-300)
        perm = rng.permutation(C)
        sp, _ = O.hadronic(np.ascontiguousarray(fk[..., perm]), pairs[perm], f)
        assert np.all(np.abs(sp - s1) <= 4e-16 * sc1 + 1e-300)
        for r in range(R):
            sr, _ = O.hadronic(fk, pairs, f[r:r + 1])
            assert np.array_equal(sr[:, 0], s1[:, r])
        L = np.einsum("rci,rcj->rcij", f[:, pairs[:, 0], :], f[:, pairs[:, 1], :])   # [R][C][i][j]
        flat = np.einsum("nijc,rcij->nr", fk, L)
        assert np.all(np.abs(flat - s1) <= 1e-14 * sc1 + 1e-300)
        g = rng.standard_normal((N, R))
        df, D = O.hadronic_vjp(fk, pairs, f, g)
        assert np.all(np.abs((f * df).sum(axis=(1, 2)) - 2.0 * (g * s1).sum(axis=0)) <= 1e-13 * (np.abs(f) * D).sum(axis=(1, 2)) + 1e-300)

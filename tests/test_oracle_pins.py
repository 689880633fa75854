"""Pins for the CPU oracle (oracle/agnvar_oracle.cpp): every oracle function is checked against
something other than itself -- values the paper prints (tests/golden/), closed forms, invariants,
numpy/scipy library routines on special cases, brute force on tiny inputs.  CPU only.
"""
import math
import os

import numpy as np
import pytest
from scipy import integrate, special, stats

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _paper_numbers():
    out = {}
    for line in open(os.path.join(GOLD, "paper_numbers.txt")):
        line = line.split("#")[0].strip()
        if line:
            k, v, tol = line.split()
            out[k] = (float(v), float(tol))
    return out


# ------------------------------------------------------------------------------------------------
# O1 Philox4x32-10, u53, Box-Muller
# ------------------------------------------------------------------------------------------------
def test_philox_known_answer_vectors(orc):
    n = 0
    for line in open(os.path.join(GOLD, "philox_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(t, 16) for t in line.split()]
        got = orc.philox4x32_10(w[0:4], w[4:6])
        assert [int(v) for v in got] == w[6:10]
        n += 1
    assert n == 3


def test_philox_stream_layout(orc):
    # key = (seed lo, seed hi); counter = (i lo, i hi, b, tag)
    seed, i, b, tag = 0x1122334455667788, 0x0000000900000007, 5, 1
    a = orc.philox_stream(seed, i, b, tag)
    c = orc.philox4x32_10([7, 9, 5, 1], [0x55667788, 0x11223344])
    assert np.array_equal(a, c)


def test_u53_exact_dyadic(orc):
    assert orc.u53(0, 0) == 2.0 ** -53
    assert orc.u53(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53
    assert orc.u53(0x80000000, 0) == 0.5 + 2.0 ** -53
    # low 12 bits of the second word are dropped
    assert orc.u53(123, 0x00000FFF) == orc.u53(123, 0)
    assert orc.u53(1, 0) == (2 * (1 << 20) + 1) * 2.0 ** -53


def test_normals_are_standard_normal(orc):
    g = np.array([orc.tk_normal_pair(3, j, 2) for j in range(1, 20001)])
    for col in (0, 1):
        assert stats.kstest(g[:, col], "norm").pvalue > 0.01
    assert abs(np.mean(g[:, 0] * g[:, 1])) < 0.03           # re and im uncorrelated
    r2 = g[:, 0] ** 2 + g[:, 1] ** 2                          # chi^2 with 2 dof = Exp(1/2)
    assert stats.kstest(r2, "expon", args=(0, 2)).pvalue > 0.01
    # Box-Muller by hand from the words
    w = orc.philox_stream(3, 17, 2, 0)
    u1, u2 = orc.u53(w[0], w[1]), orc.u53(w[2], w[3])
    gr, gi = orc.tk_normal_pair(3, 17, 2)
    assert gr == pytest.approx(math.sqrt(-2 * math.log(u1)) * math.cos(2 * math.pi * u2), rel=1e-14)
    assert gi == pytest.approx(math.sqrt(-2 * math.log(u1)) * math.sin(2 * math.pi * u2), rel=1e-14)


# ------------------------------------------------------------------------------------------------
# DFT (Eq. A1) and FFT
# ------------------------------------------------------------------------------------------------
def test_dft_naive_closed_forms(orc):
    n = 12
    d = np.zeros(n); d[3] = 1.0
    k = np.arange(n)
    assert np.allclose(orc.dft_naive(d, -1), np.exp(-2j * np.pi * 3 * k / n), atol=1e-14)
    assert np.allclose(orc.dft_naive(d, +1), np.exp(+2j * np.pi * 3 * k / n), atol=1e-14)
    c = np.ones(n)
    e = np.zeros(n); e[0] = n
    assert np.allclose(orc.dft_naive(c, -1), e, atol=1e-13)
    tone = np.exp(2j * np.pi * 5 * k / n)                      # single tone -> one bin
    e = np.zeros(n, dtype=complex); e[5] = n
    assert np.allclose(orc.dft_naive(tone, -1), e, atol=1e-12)
    rng = np.random.default_rng(1)
    a = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    b = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    assert np.allclose(orc.dft_naive(2 * a - 3j * b), 2 * orc.dft_naive(a) - 3j * orc.dft_naive(b), atol=1e-12)


@pytest.mark.parametrize("n", [2, 4, 8, 16, 20, 40, 64, 80, 160, 256])
def test_fft_recursive_vs_naive(orc, n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    for sign in (-1, +1):
        a, b = orc.fft(x, sign), orc.dft_naive(x, sign)
        assert np.linalg.norm(a - b) <= 1e-13 * np.linalg.norm(b)


@pytest.mark.parametrize("n", [512, 4096, 5 * 2 ** 10, 40960])
def test_fft_parseval_roundtrip_and_library(orc, n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n)
    X = orc.rfft(x)
    full = np.concatenate([X, np.conj(X[-2:0:-1])])
    assert np.sum(np.abs(full) ** 2) == pytest.approx(n * np.sum(x ** 2), rel=1e-12)   # Parseval
    assert np.max(np.abs(orc.irfft(X, n) - x)) < 1e-13 * np.max(np.abs(x)) * math.log2(n)
    Xl = np.fft.rfft(x)                                        # independent library routine
    assert np.linalg.norm(X - Xl) <= 1e-13 * np.linalg.norm(Xl)


def test_rfft_small_uses_definition_and_matches(orc):
    rng = np.random.default_rng(0)
    x = rng.standard_normal(128)
    assert np.linalg.norm(orc.rfft(x) - orc.dft_naive(x)[:65]) == 0.0
    assert np.linalg.norm(orc.rfft(x) - orc.fft(x)[:65]) < 1e-12


# ------------------------------------------------------------------------------------------------
# O2 PSD (Eq. 3)
# ------------------------------------------------------------------------------------------------
def test_psd_bpl_shape(orc):
    A, fb, al, ah = 3.0, 1 / 300.0, 1.0, 2.5
    assert orc.psd_bpl([fb], A, fb, al, ah)[0] == pytest.approx(A / 2, rel=1e-15)     # value at the break
    f = np.array([1e-9 * fb, 2e-9 * fb])
    s = orc.psd_bpl(f, A, fb, al, ah)
    assert math.log(s[1] / s[0]) / math.log(2) == pytest.approx(-al, abs=1e-6)         # low-f slope
    f = np.array([1e9 * fb, 2e9 * fb])
    s = orc.psd_bpl(f, A, fb, al, ah)
    assert math.log(s[1] / s[0]) / math.log(2) == pytest.approx(-ah, abs=1e-6)         # high-f slope
    f = np.geomspace(1e-5, 1, 50)
    assert np.array_equal(orc.psd_bpl(f, A, fb, al, ah), orc.psd_bpl(f, A, fb, ah, al))  # symmetric in slopes
    # BASELINE C1 writes the same law as A' f^-1 / (1 + f/f_b): Eq. 3 with slopes (1, 2) and A' = A f_b
    assert np.allclose(orc.psd_bpl(f, A, fb, 1, 2), A * fb / f / (1 + f / fb), rtol=1e-14)


def test_unit_variance_normalisation(orc):
    N, dt, fb = 512, 1.0, 1 / 50.0
    v = [np.var(orc.tk_generate(-1, fb, 1, 2, N, dt, 1, 11, b, want_full=True)["x_full"]) for b in range(3000)]
    assert np.mean(v) == pytest.approx(1.0, abs=0.03)
    # closed form: expected variance = (2 sum_{j<M/2} S_j + S_{M/2}) / M^2
    A = orc.psd_unit_variance_A(N, dt, fb, 1, 2)
    S = orc.psd_bpl(np.arange(1, N // 2 + 1) / (N * dt), A, fb, 1, 2)
    assert (2 * S[:-1].sum() + S[-1]) / N ** 2 == pytest.approx(1.0, rel=1e-12)


# ------------------------------------------------------------------------------------------------
# O3 TK95
# ------------------------------------------------------------------------------------------------
def test_tk_ensemble_periodogram_matches_psd(orc):
    """North-star pin: ensemble-mean periodogram over 1e4 realisations within 5% of the PSD
    (oversample 1; per-bin standard error is 1%)."""
    N, dt, fb, A = 1024, 1.0, 1 / 100.0, 7.0
    acc = np.zeros(N // 2 + 1)
    nreal = 10000
    for b in range(nreal):
        acc += orc.tk_generate(A, fb, 1.0, 2.0, N, dt, 1, 5, b)["A_norm"] ** 2
    acc /= nreal
    S = orc.psd_bpl(np.arange(1, N // 2 + 1) / (N * dt), A, fb, 1.0, 2.0)
    assert acc[0] < 1e-20 * S.max()                       # X_0 = 0
    assert np.max(np.abs(acc[1:] / S - 1.0)) < 0.05


def test_tk_structure(orc):
    N, os_ = 256, 10
    r = orc.tk_generate(2.0, 1 / 30.0, 1.0, 2.0, N, 1.0, os_, 9, 4, want_full=True)
    M = N * os_
    X, x = r["X"], r["x_full"]
    assert X[0] == 0 and X[-1].imag == 0.0
    assert abs(x.mean()) < 1e-12 * np.abs(x).max()        # zero mean because X_0 = 0
    assert np.allclose(x, np.fft.irfft(X, M), atol=1e-12 * np.abs(x).max())   # library inverse, 1/M
    assert np.array_equal(r["x_norm"], x[(M - N) // 2:(M - N) // 2 + N])     # central N kept (BASELINE C1)
    assert np.allclose(r["A_norm"], np.abs(np.fft.rfft(r["x_norm"])), rtol=1e-10, atol=1e-12)
    # spectrum by hand from the normals for one bin, and the Nyquist bin
    S = orc.psd_bpl(np.arange(0, M // 2 + 1) / (M * 1.0), 2.0, 1 / 30.0, 1.0, 2.0)
    gr, gi = orc.tk_normal_pair(9, 37, 4)
    assert X[37] == pytest.approx(math.sqrt(S[37] / 2) * complex(gr, gi), rel=1e-13)
    gr, _ = orc.tk_normal_pair(9, M // 2, 4)
    assert X[M // 2].real == pytest.approx(math.sqrt(S[M // 2]) * gr, rel=1e-13)


# ------------------------------------------------------------------------------------------------
# O4 ERDF (Eq. 1-2; sampled density is dN/dlambda)
# ------------------------------------------------------------------------------------------------
def _draws(orc, erdf, n, G=4096, seed=1, dtype=1):
    lam, U = orc.erdf_draw(erdf, G, n, seed, 0, dtype)
    return lam, U


def test_erdf_bpl_closed_form_ks(orc):
    d = 0.6
    e = dict(kind=0, lam_star=0.03, delta1=d, delta2=2 * d, lam_min=1e-4, lam_max=1.0)
    lam, _ = _draws(orc, e, 200000)
    assert lam.min() >= e["lam_min"] and lam.max() <= e["lam_max"]

    def Gf(l):
        t = (l / e["lam_star"]) ** d
        return (-1.0 / t - np.log(t) + np.log1p(t)) / d

    def cdf(l):
        return (Gf(l) - Gf(e["lam_min"])) / (Gf(e["lam_max"]) - Gf(e["lam_min"]))

    assert stats.kstest(lam, cdf).pvalue > 0.01


def test_erdf_bpl_quadrature_ks(orc):
    e = dict(kind=0, lam_star=10 ** -1.5, delta1=0.45, delta2=2.5, lam_min=1e-5, lam_max=1.0)   # C2's ERDF
    lam, _ = _draws(orc, e, 100000, seed=2)
    xi = lambda u: 1.0 / ((10 ** u / e["lam_star"]) ** e["delta1"] + (10 ** u / e["lam_star"]) ** e["delta2"])
    tot = integrate.quad(xi, -5, 0, epsabs=1e-13, epsrel=1e-12, limit=200)[0]
    us = np.linspace(-5, 0, 2001)
    cd = np.array([integrate.quad(xi, -5, u, epsabs=1e-13, epsrel=1e-12, limit=200)[0] for u in us]) / tot
    cdf = lambda l: np.interp(np.log10(l), us, cd)
    assert stats.kstest(lam, cdf).pvalue > 0.01


def test_erdf_lognormal_ks(orc):
    e = dict(kind=1, mu_log10=-2.0, sigma_log10=0.7, lam_min=1e-5, lam_max=1.0)       # C3's ERDF
    lam, _ = _draws(orc, e, 200000, seed=3)
    a, b = (-5 + 2) / 0.7, (0 + 2) / 0.7
    Phi = lambda z: 0.5 * (1 + special.erf(z / math.sqrt(2)))
    cdf = lambda l: (Phi((np.log10(l) + 2) / 0.7) - Phi(a)) / (Phi(b) - Phi(a))
    assert stats.kstest(lam, cdf).pvalue > 0.01


def test_erdf_paper_fractions(orc):
    """The only ERDF numbers the paper prints -- they fix reading Q10."""
    gold = _paper_numbers()
    e = dict(kind=0, lam_star=0.11, delta1=0.47, delta2=2.53, lam_min=10 ** -3.75, lam_max=10 ** 0.5)
    lam, _ = _draws(orc, e, 400000, seed=4)
    v, tol = gold["active_fraction_above_0p01"]
    assert abs(np.mean(lam > 0.01) - v) < tol
    v, tol = gold["fraction_above_logl_m1p2"]
    assert abs(np.mean(lam > 10 ** -1.2) - v) < tol


def test_erdf_table_and_draw_mechanics(orc):
    e = dict(kind=0, lam_star=0.1, delta1=0.4, delta2=2.4, lam_min=1e-4, lam_max=1.0)          # C1's ERDF
    G = 4096
    u, p, Cc = orc.erdf_table(e, G)
    assert u[0] == pytest.approx(-4.0) and u[-1] == pytest.approx(0.0, abs=1e-12)
    assert Cc[0] == 0.0 and Cc[-1] == 1.0 and np.all(np.diff(Cc) > 0)
    assert p[100] == pytest.approx(1 / ((10 ** u[100] / 0.1) ** 0.4 + (10 ** u[100] / 0.1) ** 2.4), rel=1e-13)
    trap = np.concatenate([[0], np.cumsum(0.5 * (p[1:] + p[:-1]) * np.diff(u))])
    assert np.allclose(Cc, trap / trap[-1], rtol=1e-12, atol=1e-15)
    lam, U = orc.erdf_draw(e, G, 1001, 8, 3, 1)
    # uniforms: sample n uses words (0,1) of Philox call n>>1 if n even else (2,3); stream tag 1
    w = orc.philox_stream(8, 250, 3, 1)
    assert U[500] == orc.u53(w[0], w[1]) and U[501] == orc.u53(w[2], w[3])
    # inverse CDF by library interpolation: C(log10 lam) == U
    assert np.allclose(np.interp(np.log10(lam), u, Cc), U, rtol=0, atol=1e-12)
    lam32, _ = orc.erdf_draw(e, G, 1001, 8, 3, 0)
    assert np.array_equal(lam32, lam.astype(np.float32).astype(np.float64))


def test_table1_arithmetic():
    """Table 1: N_steps * t_bin <-> T; fixes the unit convention f = j/(N t_bin)."""
    gold = _paper_numbers()
    yr = 365.25
    for key, n, days in [("table1_T_2p23_100d", 2 ** 23, 100), ("table1_T_2p27_100d", 2 ** 27, 100),
                         ("table1_T_2p23_25d", 2 ** 23, 25), ("table1_T_2p23_400d", 2 ** 23, 400)]:
        v, tol = gold[key]
        assert abs(n * days / yr / 1e6 - v) < tol


# ------------------------------------------------------------------------------------------------
# Stable argsort (O6 step 4)
# ------------------------------------------------------------------------------------------------
def test_stable_argsort_bruteforce(orc):
    rng = np.random.default_rng(0)
    for n in (1, 2, 7, 64):
        x = rng.integers(-3, 4, size=n).astype(np.float64)        # many ties
        if n > 2:
            x[1], x[2] = 0.0, -0.0                                 # -0 == +0: a tie, index order decides
        idx = orc.stable_argsort(x)
        rank = np.array([sum((x[s] < x[t]) or (x[s] == x[t] and s < t) for s in range(n)) for t in range(n)])
        inv = np.empty(n, dtype=np.int64); inv[idx] = np.arange(n)
        assert np.array_equal(inv, rank)
        assert np.array_equal(orc.rank_bruteforce(x), rank.astype(np.uint32))
        assert np.array_equal(idx, np.argsort(x, kind="stable").astype(np.uint32))


# ------------------------------------------------------------------------------------------------
# O6 E13 step and loop
# ------------------------------------------------------------------------------------------------
def _setup(orc, N=1024, os_=10, seed=0, b=0, dtype=1):
    tk = orc.tk_generate(-1, 1 / 300.0, 1.0, 2.0, N, 1.0, os_, seed, b)
    e = dict(kind=0, lam_star=0.1, delta1=0.4, delta2=2.4, lam_min=1e-4, lam_max=1.0)
    srt, perm0, lam = orc.erdf_sample_sorted(e, 4096, N, seed, b, dtype)
    return tk["A_norm"], srt, perm0, lam


def test_e13_step_against_library_pieces(orc):
    A, srt, perm0, lam = _setup(orc, N=512)
    x_adj, idx_new, x_next, ch = orc.e13_step(A, srt, perm0, lam)
    X0, X1 = np.fft.rfft(lam), np.fft.rfft(x_adj)
    assert np.allclose(np.abs(X1), A, rtol=1e-9, atol=1e-12 * A.max())            # amplitudes replaced
    assert np.allclose(X1 * np.abs(X0), X0 * A, rtol=1e-9, atol=1e-9 * (A.max() * np.abs(X0).max()))  # phases kept
    assert np.array_equal(idx_new, np.argsort(x_adj, kind="stable").astype(np.uint32))
    assert np.array_equal(x_next[idx_new], srt)                                   # rank-order scatter
    assert ch == int(np.sum(idx_new != perm0))
    assert np.all(np.diff(x_adj[idx_new]) >= 0)


def test_e13_zero_amplitude_bin_gets_phase_zero(orc):
    # Q17: |X_j| = 0 -> X'_j = A_j.  The zero series has X_j = 0 exactly for every j.
    N = 16
    x = np.zeros(N)
    A = np.arange(1, N // 2 + 2, dtype=np.float64)
    x_adj, *_ = orc.e13_step(A, np.sort(x), np.arange(N, dtype=np.uint32), x)
    assert np.allclose(np.fft.rfft(x_adj), A, atol=1e-12)


def test_e13_loop_invariants(orc):
    A, srt, perm0, lam = _setup(orc, N=1024)
    out = orc.e13_iterate(A, srt, perm0, 100)
    assert np.array_equal(np.sort(out["x"]), srt)                   # exact permutation of the draw
    assert np.array_equal(out["x"][out["perm"]], srt)
    k = out["iters_used"]
    assert 1 <= k <= 100
    if k < 100:
        assert out["changed_hist"][k - 1] == 0 and np.all(out["changed_hist"][:k - 1] > 0)
    # the loop is the step applied repeatedly
    perm, x = perm0.copy(), lam.copy()
    for it in range(min(k, 5)):
        x_adj, perm_n, x, ch = orc.e13_step(A, srt, perm, x)
        assert ch == out["changed_hist"][it]
        perm = perm_n
    # scale invariance: c = 2^k bit-identical, generic c identical permutation
    o2 = orc.e13_iterate(4.0 * A, srt, perm0, 100)
    assert np.array_equal(o2["perm"], out["perm"]) and o2["iters_used"] == k
    assert np.array_equal(o2["changed_hist"], out["changed_hist"])
    o3 = orc.e13_iterate(3.7 * A, srt, perm0, 100)
    assert np.array_equal(o3["perm"], out["perm"])
    # DC amplitude only shifts x_adj
    A2 = A.copy(); A2[0] += 123.0
    o4 = orc.e13_iterate(A2, srt, perm0, 100)
    assert np.array_equal(o4["perm"], out["perm"])
    # restart from own output reproduces itself (fixed point if converged)
    o5 = orc.e13_iterate(A, srt, out["perm"], 3)
    if k < 100:
        assert o5["iters_used"] == 1 and np.array_equal(o5["perm"], out["perm"])
    # split run == single run
    a = orc.e13_iterate(A, srt, perm0, 4)
    bb = orc.e13_iterate(A, srt, a["perm"], 3)
    c = orc.e13_iterate(A, srt, perm0, 7)
    assert np.array_equal(bb["perm"], c["perm"]) and np.array_equal(bb["x"], c["x"])


def test_e13_improves_periodogram(orc):
    """'Periodogram consistent with the input PSD': after the loop the power-law index
    of x_sim's periodogram is that of the target, while the raw draw is white.  Benign regime
    (slope 1, PAPER.md:315-326 reports the method degrades for slopes >~ 1.5 with wide PDFs)."""
    N = 2048
    A = orc.tk_generate(-1, 10.0, 1.0, 2.0, N, 1.0, 1, 0, 0)["A_norm"]      # f_b above Nyquist: pure f^-1
    e = dict(kind=0, lam_star=0.1, delta1=0.4, delta2=2.4, lam_min=1e-4, lam_max=1.0)
    srt, perm0, lam = orc.erdf_sample_sorted(e, 4096, N, 0, 0, 1)
    out = orc.e13_iterate(A, srt, perm0, 100)
    j = np.arange(1, A.size)

    def slope(amp):                      # power-law index of the periodogram, least squares in log-log
        return np.polyfit(np.log(j), 2 * np.log(amp[1:]), 1)[0]

    s_target, s_out, s_draw = slope(A), slope(np.abs(np.fft.rfft(out["x"]))), slope(np.abs(np.fft.rfft(lam)))
    assert abs(s_draw) < 0.15                     # the raw draw is white
    assert s_target < -0.9                        # red target
    assert abs(s_out - s_target) < 0.1


# ------------------------------------------------------------------------------------------------
# O7 periodogram (Eq. A2, A4, A5)
# ------------------------------------------------------------------------------------------------
def test_periodogram_pins(orc):
    N, dt = 1024, 7.0
    n = np.arange(N)
    a, j0 = 3.0, 37
    P = orc.periodogram(a * np.cos(2 * np.pi * j0 * n / N + 0.3), dt, 0)
    assert P[j0 - 1] == pytest.approx(a * a / 2, rel=1e-12)                   # A2: (2/N^2)|X|^2
    assert np.sum(P) - P[j0 - 1] < 1e-20
    rng = np.random.default_rng(5)
    x = 5.0 + rng.standard_normal(N)
    Pr = orc.periodogram(x, dt, 1)
    df = 1.0 / (N * dt)
    lhs = np.sum(Pr[:-1]) * df + 0.5 * Pr[-1] * df                            # A5: integral = sigma^2/mu^2
    assert lhs == pytest.approx(np.var(x) / np.mean(x) ** 2, rel=1e-11)
    P0 = orc.periodogram(x, dt, 0)
    assert np.allclose(P0, 2.0 / N ** 2 * np.abs(np.fft.rfft(x))[1:] ** 2, rtol=1e-11)
    w = rng.standard_normal(1 << 14)                                          # white noise -> flat, mean 2 sigma^2/N
    Pw = orc.periodogram(w, 1.0, 0)
    assert np.mean(Pw[:-1]) == pytest.approx(2.0 / w.size, rel=0.05)
    h = Pw.size // 2
    assert np.mean(Pw[:h]) / np.mean(Pw[h:-1]) == pytest.approx(1.0, abs=0.08)


def test_periodogram_binned(orc):
    N = 4096
    rng = np.random.default_rng(6)
    x = 2.0 + rng.standard_normal(N)
    edges = np.unique(np.ceil((N / 2) ** (np.arange(65) / 64.0)).astype(np.int64))
    out, cnt = orc.periodogram_binned(x, 1.0, 0, edges)
    P = orc.periodogram(x, 1.0, 0)
    assert cnt.sum() == N // 2                                                # every j = 1..N/2 in exactly one bin
    for e in (0, 5, len(edges) - 2):
        j0 = edges[e]
        j1 = edges[e + 1] if e < len(edges) - 2 else N // 2 + 1
        assert cnt[e] == j1 - j0
        assert out[e] == pytest.approx(np.mean(P[j0 - 1:j1 - 1]), rel=1e-13)

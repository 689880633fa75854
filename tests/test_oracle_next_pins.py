"""Pins (-m "not gpu") of the oracle's NEXT-1 / NEXT-2 functions against what the paper and the mathematics fix:
delta_i (Eq. 4), the structure function (Eq. A6), the representative SF (Eq. 6,
PAPER.md:244-251), magnitude differences and P(|dm| > dm_ref | tau)."""
import numpy as np
import pytest

BPL = dict(kind=0, lam_star=0.1, delta1=0.4, delta2=2.4, lam_min=1e-4, lam_max=1.0)


# ---- NEXT-1 ---------------------------------------------------------------------------------------
def test_delta_closed_forms(orc):
    rng = np.random.default_rng(0)
    x = 10.0 ** rng.uniform(-4, 0, 1000)
    assert orc.delta_rms(x, x) == 0.0                                   # a fixed point
    assert orc.delta_rms(10.0 * x, x) == pytest.approx(1.0, abs=1e-15)  # "log" is log10 (dex), not ln
    assert orc.delta_rms(x, 100.0 * x) == pytest.approx(2.0, abs=1e-15)  # a square: the sign of the log is irrelevant
    # one swapped pair: two samples change by +-log10(a/b), the others not at all
    y = x.copy()
    y[3], y[700] = x[700], x[3]
    want = np.sqrt(2.0 * np.log10(x[3] / x[700]) ** 2 / x.size)
    assert orc.delta_rms(y, x) == pytest.approx(want, rel=1e-13)
    # rms, not mean absolute value and not a sum: scale with a known mix
    z = x.copy()
    z[:250] *= 10.0 ** 0.2
    assert orc.delta_rms(z, x) == pytest.approx(0.2 * np.sqrt(0.25), rel=1e-12)


def test_iterate_delta_matches_plain_loop_and_honours_threshold(orc):
    N = 1024
    srt, perm0, _ = orc.erdf_sample_sorted(BPL, 4096, N, 3, 0, 1)
    an = orc.tk_generate(0.0, 1.0 / 50.0, 1.0, 2.0, N, 1.0, 1, 3, 0)["A_norm"]
    plain = orc.e13_iterate(an, srt, perm0, 40)
    full = orc.e13_iterate_delta(an, srt, perm0, 40, 0.0)
    # threshold off: the same trajectory as the plain loop (the rule only adds a reduction)
    assert full["iters_used"] == plain["iters_used"]
    assert (full["perm"] == plain["perm"]).all() and (full["x"] == plain["x"]).all()
    assert (full["changed_hist"] == plain["changed_hist"]).all()
    k_used = full["iters_used"]
    d = full["delta_hist"]
    assert (d[:k_used - 1] > 0).all() and (d[k_used:] == 0).all()
    # delta_k recomputed by hand from the states the step function returns
    x = np.empty(N)
    x[perm0] = srt
    perm = perm0
    for k in range(3):
        _, idx, xn, _ = orc.e13_step(an, srt, perm, x)
        assert d[k] == pytest.approx(np.sqrt(np.mean(np.log10(xn / x) ** 2)), rel=1e-13)
        x, perm = xn, idx
    # the measure falls as the iteration settles ("until their variability converges")
    assert d[min(10, k_used - 2)] < 0.5 * d[0]
    # a threshold between delta_5 and what came before stops the run at the first k with delta_k <= threshold
    thr = float(d[5]) * (1 + 1e-12)
    first = int(np.argmax(d[:k_used] <= thr)) + 1
    stopped = orc.e13_iterate_delta(an, srt, perm0, 40, thr)
    assert stopped["iters_used"] == first <= 6
    assert (stopped["delta_hist"][:first] == d[:first]).all() and (stopped["delta_hist"][first:] == 0).all()
    ref = orc.e13_iterate(an, srt, perm0, first)                 # the state after `first` plain iterations
    assert (stopped["perm"] == ref["perm"]).all() and (stopped["x"] == ref["x"]).all()


# ---- NEXT-2 ---------------------------------------------------------------------------------------
def test_structure_function_bruteforce_and_closed_forms(orc):
    rng = np.random.default_rng(1)
    N = 97
    x = 10.0 ** rng.uniform(-2, 0, N)
    lags = np.array([1, 2, 5, 17, 96, 97, 200])
    for mag in (False, True):
        v = -2.5 * np.log10(x) if mag else x
        sf2, pairs = orc.structure_function(x, lags, mag)
        for q, l in enumerate(lags):
            # Eq. A6 literally: all pairs i < j with t_j - t_i = tau
            acc = [(v[i] - v[j]) ** 2 for i in range(N) for j in range(i + 1, N) if j - i == l]
            assert pairs[q] == len(acc) == max(0, N - l)
            assert sf2[q] == pytest.approx(np.mean(acc) if acc else 0.0, rel=1e-13)
    # a ramp x = a i: every difference at lag l is a l
    a = 0.37
    sf2, _ = orc.structure_function(5.0 + a * np.arange(1000.0), [1, 7, 300])
    assert np.allclose(sf2, (a * np.array([1, 7, 300])) ** 2, rtol=1e-12)
    # a tone with a whole number of periods inside the N - l pairs: SF^2 = 2 sigma^2 (1 - cos(2 pi l / p)), sigma^2 = 1/2
    p, N = 64, 64 * 40
    t = np.arange(N)
    x = np.sin(2 * np.pi * t / p)
    for l in (p, p // 2, p // 4, 3 * p):
        sf2, _ = orc.structure_function(x[:N - p + l] if l < p else x[:N + 0], [l])
        npairs = (N - p + l if l < p else N) - l
        assert npairs % p == 0
        assert sf2[0] == pytest.approx(1.0 - np.cos(2 * np.pi * l / p), abs=1e-12)


def test_structure_function_random_walk_slope(orc):
    """SF ~ tau^beta with beta = (alpha - 1)/2 for PSD ~ f^-alpha: a random walk (alpha = 2) has
    E[SF^2(l)] = sigma_step^2 l exactly, i.e. beta = 1/2.  Representative SF over 200 realisations (Eq. 6)."""
    rng = np.random.default_rng(2)
    lags = np.array([1, 2, 4, 8, 16, 32, 64])
    all_sf2 = np.stack([orc.structure_function(np.cumsum(rng.standard_normal(20000)), lags)[0] for _ in range(200)])
    mean, se = orc.sf_representative(all_sf2)
    assert np.allclose(mean, all_sf2.mean(axis=0), rtol=1e-13)
    assert np.allclose(se, all_sf2.std(axis=0, ddof=1) / np.sqrt(200), rtol=1e-12)
    assert np.all(np.abs(mean / lags - 1.0) < 5 * se / lags + 0.01)
    beta = np.polyfit(np.log10(lags), 0.5 * np.log10(mean), 1)[0]
    assert beta == pytest.approx(0.5, abs=0.01)


def test_magnitude_units(orc):
    rng = np.random.default_rng(3)
    x = 10.0 ** rng.uniform(-3.75, 0.5, 5000)
    lags = np.array([1, 10, 100])
    sf_m, _ = orc.structure_function(x, lags, True)
    # a constant factor on L/L_Edd (zero point) drops out of magnitude differences
    assert np.allclose(orc.structure_function(37.0 * x, lags, True)[0], sf_m, rtol=1e-10)
    # m2 - m1 = -2.5 log10(x2 / x1): SF_mag^2 is 6.25 x the SF^2 of log10 x
    sf_log, _ = orc.structure_function(np.log10(x), lags, False)
    assert np.allclose(sf_m, 6.25 * sf_log, rtol=1e-12)


def test_delta_m_probability(orc):
    rng = np.random.default_rng(4)
    N = 400
    x = 10.0 ** rng.uniform(-3.75, 0.5, N)              # the paper's 4.25-dex range
    m = -2.5 * np.log10(x)
    lags = np.array([1, 3, 50])
    refs = np.array([0.0, 0.5, 2.5, 10.0, 10.625, 11.0])
    prob, cons = orc.delta_m_prob(x, lags, refs)
    for q, l in enumerate(lags):
        d = np.abs(m[:-l] - m[l:])
        assert cons[q] == N - l
        for r, ref in enumerate(refs):
            assert prob[q, r] == pytest.approx(np.mean(d > ref), abs=1e-15)
    assert (np.diff(prob, axis=1) <= 0).all()            # monotone in dm_ref
    # the largest possible |dm| of a 4.25-dex PDF is 2.5 x 4.25 = 10.6 mag: nothing beyond it
    assert (prob[:, refs >= 10.625] == 0).all()
    # magnitude cut (Fig. 17): points fainter than m_cut become upper limits at m_cut; pairs with no detection drop out
    m_zero, m_cut = 20.0, 22.0
    mm = m_zero + m
    det = mm <= m_cut
    mc = np.minimum(mm, m_cut)
    prob_c, cons_c = orc.delta_m_prob(x, lags, refs, m_zero, m_cut)
    for q, l in enumerate(lags):
        use = det[:-l] | det[l:]
        d = np.abs(mc[:-l] - mc[l:])[use]
        assert cons_c[q] == use.sum()
        for r, ref in enumerate(refs):
            assert prob_c[q, r] == pytest.approx(np.mean(d > ref) if d.size else 0.0, abs=1e-15)
    assert (cons_c < cons).all()


# ---- NEXT-4 ---------------------------------------------------------------------------------------
def test_ensemble_sf_reduces_to_plain_sf_and_bruteforce(orc):
    rng = np.random.default_rng(5)
    B, N = 6, 300
    x = 10.0 ** rng.uniform(-2, 0, (B, N))
    lags = np.array([1, 2, 9, 40, 299, 300])
    # one curve, the whole series, nothing masked: Eq. A6 itself
    for mag in (False, True):
        sf2, pairs, offs = orc.ensemble_sf(x[:1], N, 1.0, 7, 0, lags, mag)
        ref, rp = orc.structure_function(x[0], lags, mag)
        assert offs[0] == 0 and (pairs == rp).all() and np.allclose(sf2, ref, rtol=1e-14)
    # general case rebuilt by hand from the raw Philox words (pinned by the published known-answer vectors)
    n_sub, keep, seed, curve0 = 120, 0.3, 11, 4
    sf2, pairs, offs = orc.ensemble_sf(x, n_sub, keep, seed, curve0, lags[:4])
    acc, cnt = np.zeros(4), np.zeros(4, dtype=np.int64)
    for b in range(B):
        w = orc.philox_stream(seed, 0, curve0 + b, 3)
        off = int(np.floor(orc.u53(w[0], w[1]) * (N - n_sub + 1)))
        assert off == offs[b] and 0 <= off <= N - n_sub
        kept = np.zeros(n_sub, dtype=bool)
        for j in range(n_sub):
            w = orc.philox_stream(seed, j >> 1, curve0 + b, 4)
            kept[j] = (orc.u53(w[2], w[3]) if j & 1 else orc.u53(w[0], w[1])) < keep
        seg = x[b, off:off + n_sub]
        for q, l in enumerate(lags[:4]):
            use = kept[:-l] & kept[l:]
            acc[q] += np.sum((seg[:-l] - seg[l:])[use] ** 2)
            cnt[q] += use.sum()
    assert (pairs == cnt).all() and cnt[0] > 0
    assert np.allclose(sf2, acc / np.maximum(cnt, 1), rtol=1e-13)
    # a different curve0 draws different positions and masks
    assert not np.array_equal(orc.ensemble_sf(x, n_sub, keep, seed, curve0 + 1, lags[:4])[2], offs)


def test_ensemble_sf_is_unbiased_and_pair_counts_scale(orc):
    """Fig. 8's statement: "the ensemble SF always scatters around the representative SF"; for a random walk
    E[SF^2(l)] = l whatever the mask, and the pooled number of pairs is ~ keep^2 (n_sub - l) B."""
    rng = np.random.default_rng(6)
    B, N, n_sub = 400, 5000, 1000
    x = np.cumsum(rng.standard_normal((B, N)), axis=1)
    lags = np.array([1, 3, 10, 30, 100])
    for keep in (0.1, 0.5):
        sf2, pairs, offs = orc.ensemble_sf(x, n_sub, keep, 3, 0, lags)
        expect = keep ** 2 * (n_sub - lags) * B
        assert np.all(np.abs(pairs - expect) < 6 * np.sqrt(expect) + 0.02 * expect)
        # relative scatter of the pooled mean: var of a squared Gaussian difference is 2 l^2, pairs are correlated -> loose
        assert np.all(np.abs(sf2 / lags - 1.0) < 0.25)
        assert offs.min() >= 0 and offs.max() <= N - n_sub and len(set(offs.tolist())) > B // 2


def test_moments(orc):
    scipy_stats = pytest.importorskip("scipy.stats")
    rng = np.random.default_rng(7)
    x = rng.gamma(2.0, 1.5, 20000)
    m = orc.moments(x)
    assert m[0] == pytest.approx(x.mean(), rel=1e-13) and m[1] == pytest.approx(x.var(), rel=1e-12)
    assert m[2] == pytest.approx(scipy_stats.skew(x), rel=1e-11) and m[3] == pytest.approx(scipy_stats.kurtosis(x), rel=1e-11)
    # closed forms: two-point distribution {0 with prob 3/4, 1 with prob 1/4}: skew = (1 - 2p)/sqrt(pq), kurt = (1 - 6pq)/(pq)
    y = np.array([0.0] * 750 + [1.0] * 250)
    p, q = 0.25, 0.75
    m = orc.moments(y)
    assert m[0] == pytest.approx(p) and m[1] == pytest.approx(p * q)
    assert m[2] == pytest.approx((1 - 2 * p) / np.sqrt(p * q)) and m[3] == pytest.approx((1 - 6 * p * q) / (p * q))
    # a Gaussian series has skewness and excess kurtosis ~ 0 (what Fig. 2 tests the TK95 output against)
    g = orc.moments(rng.standard_normal(200000))
    assert abs(g[2]) < 0.03 and abs(g[3]) < 0.06

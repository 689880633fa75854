"""Full-size parity (-m gpu): BASELINE.json's configurations at the sizes bench.py times, in the same launch
configuration.  At these sizes the oracle cannot redo a whole batch, so the tests check

  * C4 (B=4 x N=2^26, fp32), lock-step at iterations k = 2, 25 and 50 (= max_iter) of one run of the product kernels:
    properties that hold at any size and pin the result uniquely, on every curve (computed with torch on the GPU from
    the C-ABI outputs only): the permutation is valid; x_adj read along it is non-decreasing and equal keys appear by
    ascending time index (so it is THE stable argsort of the GPU's own x_adj, SURVEY 8(c) clause ii);
    x_sim,k+1[idx[r]] = sorted[r] bit-exactly (clause iv); the change count equals the number of differing entries of
    the two permutations (clause v); no curve left the distribution sort for the LSD fallback;
    and ONE CURVE AGAINST THE fp64 ORACLE, one whole step from the GPU's own x_sim (P1): relative L2 of
    x_adj <= 1e-5 (clause i) and eps-sortedness of the GPU order on the exact x_adj (clause iii);
  * S2 at C4's own size: one curve of agnvar_tk_generate at N = 2^26 (the three-pass generic FFT with split hi/lo
    twiddle tables) against the oracle's TK95 series and amplitudes;
  * P at C3's size: the periodogram and its 64-bin form at N = 2^20 against the oracle.
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def u32(t):
    return t.cpu().numpy().view(np.uint32)


def rel_l2(a, b):
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def test_c4_tk_generate_full_size(orc):
    import paper_1909_06374_b200 as ag
    from paper_1909_06374_b200 import workloads
    cfg = workloads.config("C4")
    N, p = cfg["N"], cfg["psd"][0]
    assert N == 2 ** 26
    xn, an = ag.agnvar_tk_generate(cfg["psd"], 1, N, cfg["dt"], cfg["oversample"], "f32", cfg["seed"], 1)
    ref = orc.tk_generate(0.0, p["f_b"], p["alpha_low"], p["alpha_high"], N, cfg["dt"], cfg["oversample"], cfg["seed"], 1)
    ex, ea = rel_l2(xn[0].cpu().numpy(), ref["x_norm"]), rel_l2(an[0].cpu().numpy(), ref["A_norm"])
    print(f"S2 at N=2^26: x_norm rel L2 {ex:.2e}, A_norm rel L2 {ea:.2e}")
    assert ex <= 1e-5 and ea <= 1e-5
    ag.free_workspace()


def test_c3_periodogram_full_size(orc):
    import paper_1909_06374_b200 as ag
    from paper_1909_06374_b200 import workloads
    cfg = workloads.config("C3", B=2)
    B, N = cfg["B"], cfg["N"]
    assert N == 2 ** 20 and cfg["nbins"] == 64
    out = ag.generate_light_curves(dict(cfg, max_iter=3))
    x = out["x"].cpu().numpy()
    edges = workloads.log_bin_edges(N, 64)
    P = ag.agnvar_periodogram(out["x"], cfg["dt"], 1).cpu().numpy()
    pb, cnt = out["pbin"].cpu().numpy(), out["counts"].cpu().numpy()
    for b in range(B):
        ref = orc.periodogram(x[b].astype(np.float64), cfg["dt"], 1)
        assert rel_l2(P[b], ref) <= 1e-5
        rb, rc = orc.periodogram_binned(x[b].astype(np.float64), cfg["dt"], 0, edges)
        assert (cnt == rc).all()
        assert np.max(np.abs(pb[b] / rb - 1.0)) <= 1e-5
    ag.free_workspace()


def test_c4_full_size_lockstep(orc):
    import paper_1909_06374_b200 as ag
    from paper_1909_06374_b200 import workloads
    cfg = workloads.config("C4")
    B, N = cfg["B"], cfg["N"]
    assert (B, N, cfg["max_iter"]) == (4, 2 ** 26, 50)
    srt, perm, draw = ag.agnvar_erdf_sample_sorted(cfg["erdf"], B, N, "f32", cfg["seed"], 0, cfg["grid_points"],
                                                   want_draw=True)
    # S1 at full size, every curve: perm0 is a permutation, the sorted draw is the draw read along it and ascending,
    # equal values (tens of per cent of the fp32 keys at 2^26) appear by ascending draw index -> perm0 is THE stable
    # argsort of the GPU's own draw; one curve's draw against the oracle's inverse-CDF draw
    n_tied = 0
    for b in range(B):
        p = perm[b].long()
        seen = torch.zeros(N, dtype=torch.uint8, device="cuda")
        seen[p] = 1
        assert bool(seen.all()), "S1: perm0 is not a permutation"
        del seen
        assert torch.equal(draw[b][p], srt[b]), "S1: sorted != draw[perm0]"
        assert bool((srt[b][1:] >= srt[b][:-1]).all()), "S1: the sorted draw is not ascending"
        tie = srt[b][1:] == srt[b][:-1]
        assert bool((p[1:][tie] > p[:-1][tie]).all()), "S1: equal values are not in draw-index order"
        n_tied += int(tie.sum())
        del p, tie
    lam, _ = orc.erdf_draw(cfg["erdf"][1 if len(cfg["erdf"]) > 1 else 0], cfg["grid_points"], N, cfg["seed"], 1, 0)
    err = float(np.max(np.abs(draw[1].cpu().numpy().astype(np.float64) / lam - 1.0)))
    print(f"S1 at C4: adjacent equal keys {n_tied} of {B * N}; curve 1 draw vs oracle: max relative error {err:.2e}")
    assert err <= 1e-6 and n_tied > 0
    del draw, lam
    _, an = ag.agnvar_tk_generate(cfg["psd"], B, N, cfg["dt"], cfg["oversample"], "f32", cfg["seed"], 0,
                                  want_xnorm=False)
    b_chk = 1
    an_h, srt_h = an[b_chk].cpu().numpy(), srt[b_chk].cpu().numpy()
    done = 0
    for k_check in (2, 25, 50):
        # the product kernels up to iteration k_check - 1, then the step that is checked
        o = ag.agnvar_e13_iterate(an, srt, perm, k_check - 1 - done, want_fallbacks=True)
        assert int(o["sort_fallbacks"].sum()) == 0, "a curve left the distribution sort"
        done = k_check - 1
        perm_prev = perm.clone()
        x_prev = o["x"].clone()
        del o
        out = ag.agnvar_e13_iterate(an, srt, perm, 1, want_hist=True, want_xadj=True, want_fallbacks=True)
        done += 1
        torch.cuda.synchronize()
        xadj, x, hist = out["x_adj"], out["x"], out["changed_hist"]
        assert int(out["sort_fallbacks"].sum()) == 0
        for b in range(B):
            p = perm[b].long()
            seen = torch.zeros(N, dtype=torch.uint8, device="cuda")
            seen[p] = 1
            assert bool(seen.all()), "not a permutation"
            del seen
            xa = (xadj[b] + 0.0)[p]                        # -0 -> +0 (Q13)
            assert bool((xa[1:] >= xa[:-1]).all()), "x_adj is not sorted along the permutation"
            tie = xa[1:] == xa[:-1]
            assert bool((p[1:][tie] > p[:-1][tie]).all()), "equal keys are not in time-index order"
            del xa, tie
            assert torch.equal(x[b][p], srt[b]), "rank scatter"
            assert int(hist[b, 0]) == int((perm[b] != perm_prev[b]).sum()), "change count"
            del p
        # one curve, one whole step, against the fp64 oracle started from the GPU's own x_sim
        xadj64, _, xnext64, _ = orc.e13_step(an_h, srt_h, u32(perm_prev[b_chk]).copy(), x_prev[b_chk].cpu().numpy())
        xg = xadj[b_chk].cpu().numpy().astype(np.float64)
        rel = np.linalg.norm(xg - xadj64) / np.linalg.norm(xadj64)
        assert rel <= 1e-5, rel
        eps = np.max(np.abs(xg - xadj64))
        pn = u32(perm[b_chk])
        assert (np.diff(xadj64[pn]) >= -2.0 * eps).all()
        eq = float(np.mean(x[b_chk].cpu().numpy().astype(np.float64) == xnext64))
        print(f"C4 full size, iteration {k_check}: x_adj rel L2 {rel:.2e}, eps {eps:.2e}, one-step value-equal "
              f"fraction {eq:.4f}, changed {hist[:, 0].tolist()}")
        del xadj, x, out, x_prev, perm_prev, xadj64, xnext64, xg
    ag.free_workspace()


def test_maximum_size_2p27(orc):
    """The largest series the ABI accepts (N = 2^27, the paper's own cap), one curve, fp32: S1, S2 and two
    E13 iterations through the paths only this size takes (two-level distribution sort, three column sub-passes of the
    FFT, two-level rank scatter).  Properties that pin the result at any size, plus one whole oracle step from the GPU's
    own x_sim (x_adj relative L2, eps-sortedness)."""
    import paper_1909_06374_b200 as ag
    from paper_1909_06374_b200 import workloads
    cfg = workloads.config("C4", B=1)
    N = 2 ** 27
    srt, perm, _ = ag.agnvar_erdf_sample_sorted(cfg["erdf"], 1, N, "f32", cfg["seed"], 0, cfg["grid_points"])
    assert bool((srt[:, 1:] >= srt[:, :-1]).all())
    _, an = ag.agnvar_tk_generate(cfg["psd"], 1, N, cfg["dt"], 1, "f32", cfg["seed"], 0, want_xnorm=False)
    assert bool(torch.isfinite(an).all())
    o = ag.agnvar_e13_iterate(an, srt, perm, 1, want_fallbacks=True)
    perm_prev, x_prev = perm.clone(), o["x"].clone()
    del o
    out = ag.agnvar_e13_iterate(an, srt, perm, 1, want_hist=True, want_xadj=True, want_fallbacks=True)
    torch.cuda.synchronize()
    xadj, x, hist = out["x_adj"], out["x"], out["changed_hist"]
    p = perm[0].long()
    seen = torch.zeros(N, dtype=torch.uint8, device="cuda")
    seen[p] = 1
    assert bool(seen.all()), "not a permutation"
    del seen
    xa = (xadj[0] + 0.0)[p]
    assert bool((xa[1:] >= xa[:-1]).all()), "x_adj is not sorted along the permutation"
    tie = xa[1:] == xa[:-1]
    assert bool((p[1:][tie] > p[:-1][tie]).all()), "equal keys are not in time-index order"
    del xa, tie
    assert torch.equal(x[0][p], srt[0]), "rank scatter"
    assert int(hist[0, 0]) == int((perm[0] != perm_prev[0]).sum()), "change count"
    del p
    xadj64, _, xnext64, _ = orc.e13_step(an[0].cpu().numpy(), srt[0].cpu().numpy(), u32(perm_prev[0]).copy(),
                                         x_prev[0].cpu().numpy())
    xg = xadj[0].cpu().numpy().astype(np.float64)
    rel = np.linalg.norm(xg - xadj64) / np.linalg.norm(xadj64)
    eps = np.max(np.abs(xg - xadj64))
    print(f"N=2^27: x_adj rel L2 {rel:.2e}, eps {eps:.2e}, changed {hist[:, 0].tolist()}, "
          f"sort fallbacks {out['sort_fallbacks'].tolist()}")
    assert rel <= 1e-5, rel
    assert (np.diff(xadj64[u32(perm[0])]) >= -2.0 * eps).all()
    ag.free_workspace()


@pytest.mark.parametrize("logn,dtype", [(28, "f32"), (30, "f32"), (27, "f64")])
def test_beyond_the_papers_cap(orc, logn, dtype):
    """N = 2^28 and 2^30 (the largest series the ABI accepts), 2x and 8x the paper's maximum (2^27, "set
    by memory limitations"), one curve, fp32, through the generic three-pass FFT (twiddle levels up to 2^30), the LSD
    sort and the two-level scatter; and fp64 at its own maximum, 2^27.  The oracle cannot redo a step of this size in
    test time, so the checks are: the properties that pin L4-L6 at any size (exact); the FFT / replace / IFFT chain
    against a library FFT in fp64 (torch.fft on the GPU's own arrays): |rfft(x_adj)| = A_norm and the phases of x_adj
    are those of x_sim; S2 by sampled Fourier coefficients of x_norm against the oracle's normals and Eq. 3."""
    import paper_1909_06374_b200 as ag
    from paper_1909_06374_b200 import workloads
    cfg = workloads.config("C4", B=1)
    N, p, seed, dt = 2 ** logn, cfg["psd"][0], cfg["seed"], cfg["dt"]
    # ---- S2
    xn, an = ag.agnvar_tk_generate(cfg["psd"], 1, N, dt, 1, dtype, seed, 0)
    X = torch.fft.rfft(xn[0].double())
    rel_a = float(torch.linalg.norm(X.abs() - an[0].double()) / torch.linalg.norm(an[0].double()))
    A = orc.psd_unit_variance_A(N, dt, p["f_b"], p["alpha_low"], p["alpha_high"])
    rng = np.random.default_rng(0)
    js = np.unique(np.concatenate([[1, 2, 3, N // 2 - 1], rng.integers(1, N // 2, 2000),
                                   np.round(10 ** rng.uniform(0, np.log10(N // 2 - 1), 2000)).astype(np.int64)]))
    S = orc.psd_bpl(js / (N * dt), A, p["f_b"], p["alpha_low"], p["alpha_high"])
    want = np.array([complex(*orc.tk_normal_pair(seed, int(j), 0)) for j in js]) * np.sqrt(0.5 * S)
    got = X[torch.tensor(js, device="cuda")].cpu().numpy()
    rel_x = float(np.linalg.norm(got - want) / np.linalg.norm(want))
    print(f"N=2^{logn} S2: |rfft(x_norm)| vs A_norm rel L2 {rel_a:.2e}; {js.size} sampled coefficients vs the oracle rel L2 {rel_x:.2e}")
    tol = 1e-5 if dtype == "f32" else 1e-12
    assert rel_a <= tol and rel_x <= 10 * tol
    del X, xn
    torch.cuda.empty_cache()
    # ---- S1 + two iterations
    srt, perm, _ = ag.agnvar_erdf_sample_sorted(cfg["erdf"], 1, N, dtype, seed, 0, cfg["grid_points"])
    assert bool((srt[:, 1:] >= srt[:, :-1]).all())
    o = ag.agnvar_e13_iterate(an, srt, perm, 1)
    perm_prev, x_prev = perm.clone(), o["x"].clone()
    del o
    out = ag.agnvar_e13_iterate(an, srt, perm, 1, want_hist=True, want_xadj=True)
    torch.cuda.synchronize()
    xadj, x, hist = out["x_adj"], out["x"], out["changed_hist"]
    pl = perm[0].long()
    seen = torch.zeros(N, dtype=torch.uint8, device="cuda")
    seen[pl] = 1
    assert bool(seen.all()), "not a permutation"
    del seen
    xa = (xadj[0] + 0.0)[pl]
    assert bool((xa[1:] >= xa[:-1]).all()), "x_adj is not sorted along the permutation"
    tie = xa[1:] == xa[:-1]
    assert bool((pl[1:][tie] > pl[:-1][tie]).all()), "equal keys are not in time-index order"
    del xa, tie
    assert torch.equal(x[0][pl], srt[0]), "rank scatter"
    assert int(hist[0, 0]) == int((perm[0] != perm_prev[0]).sum()), "change count"
    del pl, x, out, perm_prev, srt
    torch.cuda.empty_cache()
    Xa = torch.fft.rfft(xadj[0].double())
    rel_amp = float(torch.linalg.norm(Xa.abs() - an[0].double()) / torch.linalg.norm(an[0].double()))
    Xs = torch.fft.rfft(x_prev[0].double())
    # phases kept: X_adj = A_norm X_sim / |X_sim|
    ref = an[0].double() * Xs / Xs.abs().clamp_min(1e-300)
    rel_ph = float(torch.linalg.norm(Xa - ref) / torch.linalg.norm(ref))
    print(f"N=2^{logn} E13 step: amplitudes rel L2 {rel_amp:.2e}, spectrum (amplitude replaced, phase kept) rel L2 {rel_ph:.2e}")
    assert rel_amp <= tol and rel_ph <= tol
    ag.free_workspace()

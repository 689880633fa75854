"""Full-size parity (-m gpu): BASELINE.json's metric configuration C4 (B=4 curves x N=2^26, fp32) in the launch
configuration bench.py times.  At this size the oracle cannot redo the whole batch, so the test checks

  * properties that hold at any size and pin the result uniquely, on every curve (computed with torch on the GPU
    from the C-ABI outputs only): the permutation is valid; x_adj read along it is non-decreasing and equal keys
    appear by ascending time index (so it is THE stable argsort of the GPU's own x_adj, SURVEY 8(c) clause ii);
    x_sim,k+1[idx[r]] = sorted[r] bit-exactly (clause iv); the change count equals the number of differing
    entries of the two permutations (clause v);
  * one curve against the fp64 oracle, one whole step from the GPU's own x_sim (lock-step, P1):
    relative L2 of x_adj <= 1e-5 (clause i) and eps-sortedness of the GPU order on the exact x_adj (clause iii).
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def u32(t):
    return t.cpu().numpy().view(np.uint32)


def test_c4_full_size_step(orc):
    import paper_1909_06374_b200 as ag
    from paper_1909_06374_b200 import workloads
    cfg = workloads.config("C4")
    B, N = cfg["B"], cfg["N"]
    assert (B, N) == (4, 2 ** 26)
    srt, perm, _ = ag.agnvar_erdf_sample_sorted(cfg["erdf"], B, N, "f32", cfg["seed"], 0, cfg["grid_points"])
    _, an = ag.agnvar_tk_generate(cfg["psd"], B, N, cfg["dt"], cfg["oversample"], "f32", cfg["seed"], 0,
                                  want_xnorm=False)
    # S1 at full size: the sorted draw is ascending and perm0 is a valid permutation
    assert bool((srt[:, 1:] >= srt[:, :-1]).all())
    # first step (fills x_sim,2 and the permutation after one iteration), then the step that is checked
    o1 = ag.agnvar_e13_iterate(an, srt, perm, 1, want_hist=True)
    perm_prev = perm.clone()
    x_prev = o1["x"].clone()
    del o1
    out = ag.agnvar_e13_iterate(an, srt, perm, 1, want_hist=True, want_xadj=True)
    torch.cuda.synchronize()
    xadj, x, hist = out["x_adj"], out["x"], out["changed_hist"]
    ar = torch.arange(N, device="cuda")
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
    del ar
    # one curve, one whole step, against the fp64 oracle started from the GPU's own x_sim
    b = 1
    xadj64, _, _, _ = orc.e13_step(an[b].cpu().numpy(), srt[b].cpu().numpy(), u32(perm_prev[b]).copy(),
                                   x_prev[b].cpu().numpy())
    xg = xadj[b].cpu().numpy().astype(np.float64)
    rel = np.linalg.norm(xg - xadj64) / np.linalg.norm(xadj64)
    assert rel <= 1e-5, rel
    eps = np.max(np.abs(xg - xadj64))
    pn = u32(perm[b])
    assert (np.diff(xadj64[pn]) >= -2.0 * eps).all()
    print(f"C4 full size: x_adj rel L2 {rel:.2e}, eps {eps:.2e}, changed {hist[:, 0].tolist()}")

"""Pins (-m "not gpu") of the oracle's slice sampler (NEXT-3; Neal 2003, the paper's sampler for the random draw,
PAPER.md:124, :164).  The update's stationary law is the target density whatever the step width w and the
stepping-out limit m are (Neal 2003, sec. 4): so independent draws (ONE kept state per chain, after a burn-in) are
tested against closed-form CDFs for a spread of (w, m), against the two fractions the paper prints, and a long single
chain against quadrature.  A wrong slice level, a wrong shrink side, a biased split of the stepping-out budget or a
mis-indexed uniform all move these distributions."""
import math

import numpy as np
import pytest
from scipy import integrate, special, stats

from test_oracle_pins import _paper_numbers


def _indep(orc, erdf, n, seed, w, m, burn_in=40, table=None):
    """n independent draws: n chains, one kept state each."""
    return orc.slice_sample(erdf, n, n, seed, 0, 1, burn_in=burn_in, thin=1, w=w, m=m, table=table)


@pytest.mark.parametrize("w,m,n,burn_in", [(0.02, 64, 6000, 300), (0.3, 8, 10000, 200), (1.0, 1, 10000, 400),
                                          (1.0, 8, 20000, 40), (5.0, 3, 20000, 40), (50.0, 1, 20000, 40)])
def test_slice_bpl_closed_form_ks(orc, w, m, n, burn_in):
    """(A chain that can move by at most w m per update needs a longer burn-in from its uniform start.)"""
    d = 0.6
    e = dict(kind=0, lam_star=0.03, delta1=d, delta2=2 * d, lam_min=1e-4, lam_max=1.0)
    lam, u = _indep(orc, e, n, seed=11, w=w, m=m, burn_in=burn_in)
    assert lam.min() >= e["lam_min"] and lam.max() <= e["lam_max"]
    assert np.allclose(lam, 10.0 ** u, rtol=1e-15)

    def Gf(l):
        t = (l / e["lam_star"]) ** d
        return (-1.0 / t - np.log(t) + np.log1p(t)) / d

    cdf = lambda l: (Gf(l) - Gf(e["lam_min"])) / (Gf(e["lam_max"]) - Gf(e["lam_min"]))
    assert stats.kstest(lam, cdf).pvalue > 0.01


def test_slice_lognormal_ks(orc):
    e = dict(kind=1, mu_log10=-2.0, sigma_log10=0.7, lam_min=1e-5, lam_max=1.0)       # C3's ERDF
    lam, _ = _indep(orc, e, 30000, seed=12, w=1.0, m=8)
    a, b = (-5 + 2) / 0.7, (0 + 2) / 0.7
    Phi = lambda z: 0.5 * (1 + special.erf(z / math.sqrt(2)))
    cdf = lambda l: (Phi((np.log10(l) + 2) / 0.7) - Phi(a)) / (Phi(b) - Phi(a))
    assert stats.kstest(lam, cdf).pvalue > 0.01


def test_slice_paper_fractions(orc):
    """The ERDF numbers the paper prints for its own (slice-sampled) draws: PAPER.md:378, :391, :431."""
    gold = _paper_numbers()
    e = dict(kind=0, lam_star=0.11, delta1=0.47, delta2=2.53, lam_min=10 ** -3.75, lam_max=10 ** 0.5)
    lam, _ = _indep(orc, e, 60000, seed=13, w=1.0, m=8)
    v, tol = gold["active_fraction_above_0p01"]
    assert abs(np.mean(lam > 0.01) - v) < tol
    v, tol = gold["fraction_above_logl_m1p2"]
    assert abs(np.mean(lam > 10 ** -1.2) - v) < tol


def test_slice_tabulated_densities(orc):
    """kind 2, "additional functional forms": a table on a uniform grid in u, linearly interpolated."""
    e = dict(kind=2, lam_min=1e-3, lam_max=10.0)                  # u in [-3, 1]
    # a ramp g = u - u_lo: CDF = ((u - u_lo) / 4)^2, exact for a linearly interpolated table
    G = 33
    _, u = _indep(orc, e, 20000, seed=14, w=0.7, m=4, table=np.linspace(0.0, 4.0, G))
    assert stats.kstest(u, lambda x: ((x + 3.0) / 4.0) ** 2).pvalue > 0.01
    # two boxes with a zero-density gap between them (heights 1 and 3 on [-3,-2] and [0,1]; 8 cells per unit, the
    # edges of the boxes fall on linear ramps of one cell)
    G = 33
    g = np.zeros(G)
    uu = np.linspace(-3, 1, G)
    g[(uu >= -3) & (uu <= -2)] = 1.0
    g[(uu >= 0) & (uu <= 1)] = 3.0
    _, u = _indep(orc, e, 30000, seed=15, w=6.0, m=2, burn_in=60, table=g)
    dens = lambda x: np.interp(x, uu, g)
    tot = integrate.quad(dens, -3, 1, points=list(uu), limit=400)[0]
    cdf = lambda x: np.array([integrate.quad(dens, -3, xi, points=[p for p in uu if p < xi], limit=400)[0] / tot
                              for xi in np.atleast_1d(x)])
    assert dens(u).min() > 0.0                                    # never inside the gap
    xs = np.sort(u)
    assert stats.kstest(xs[::10], cdf).pvalue > 0.01             # (thinned: the quadrature CDF is slow)
    # a narrow step (w = 0.3, no stepping out) cannot cross the gap: chains stay in the box they started in
    _, u2 = _indep(orc, e, 4000, seed=16, w=0.3, m=1, burn_in=60, table=g)
    _, u0 = orc.slice_sample(e, 4000, 4000, 16, 0, 1, burn_in=0, thin=1, w=0.3, m=1, table=g)
    # (the first state is the first update from the uniform start; where the start had g = 0 the update lands
    # anywhere with g > 0, so only chains whose first state is well inside a box are compared)
    left0, left2 = u0 < -1.0, u2 < -1.0
    assert (left0 == left2).all()


def test_slice_long_single_chain_moments(orc):
    """Ergodic average of ONE chain (chains = 1, every state kept) against quadrature of the density."""
    e = dict(kind=0, lam_star=10 ** -1.5, delta1=0.45, delta2=2.5, lam_min=1e-5, lam_max=1.0)   # C2's ERDF
    _, u = orc.slice_sample(e, 200000, 1, 17, 0, 1, burn_in=100, thin=1, w=1.5, m=6)
    xi = lambda t: 1.0 / ((10 ** t / e["lam_star"]) ** e["delta1"] + (10 ** t / e["lam_star"]) ** e["delta2"])
    Z = integrate.quad(xi, -5, 0, epsabs=1e-13, epsrel=1e-12)[0]
    m1 = integrate.quad(lambda t: t * xi(t), -5, 0, epsabs=1e-13, epsrel=1e-12)[0] / Z
    m2 = integrate.quad(lambda t: (t - m1) ** 2 * xi(t), -5, 0, epsabs=1e-13, epsrel=1e-12)[0] / Z
    # effective sample size from the lag-1 autocorrelation (AR(1) approximation)
    r1 = np.corrcoef(u[:-1], u[1:])[0, 1]
    neff = u.size * (1 - r1) / (1 + r1)
    assert abs(u.mean() - m1) < 5 * math.sqrt(m2 / neff)
    assert abs(u.var() - m2) < 0.05 * m2
    assert -5 <= u.min() and u.max() <= 0


def test_slice_stream_layout(orc):
    """Chain c of curve b depends on (seed, b, c) only: its kept states are a prefix-stable sequence stored at
    n = j * chains + c; other curves and seeds give other chains; thin = 2 keeps every second state."""
    e = dict(kind=1, mu_log10=-2.0, sigma_log10=0.7, lam_min=1e-5, lam_max=1.0)
    C_ = 16
    _, a = orc.slice_sample(e, 4 * C_, C_, 5, 3, 1, burn_in=7, thin=1, w=1.0, m=4)
    _, b2 = orc.slice_sample(e, 8 * C_, C_, 5, 3, 1, burn_in=7, thin=1, w=1.0, m=4)
    assert (b2[:4 * C_] == a).all()
    _, c = orc.slice_sample(e, 2 * C_, C_, 5, 3, 1, burn_in=8, thin=2, w=1.0, m=4)
    assert (c.reshape(2, C_) == b2.reshape(8, C_)[[2, 4]]).all()
    _, d = orc.slice_sample(e, 4 * C_, C_, 5, 4, 1, burn_in=7, thin=1, w=1.0, m=4)
    _, f = orc.slice_sample(e, 4 * C_, C_, 6, 3, 1, burn_in=7, thin=1, w=1.0, m=4)
    assert not (d == a).any() and not (f == a).any()
    # fewer chains of the same numbers are the same chains
    _, g = orc.slice_sample(e, 4 * 4, 4, 5, 3, 1, burn_in=7, thin=1, w=1.0, m=4)
    assert (g.reshape(4, 4) == a.reshape(4, C_)[:, :4]).all()
    # fp32 output is the rounded fp64 output
    l32, _ = orc.slice_sample(e, 4 * C_, C_, 5, 3, 0, burn_in=7, thin=1, w=1.0, m=4)
    l64, _ = orc.slice_sample(e, 4 * C_, C_, 5, 3, 1, burn_in=7, thin=1, w=1.0, m=4)
    assert (l32 == l64.astype(np.float32).astype(np.float64)).all()

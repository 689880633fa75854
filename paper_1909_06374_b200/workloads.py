"""Seeded synthetic workloads: BASELINE.json's five configurations as plain parameter sets.

This module holds NONE of the method's arithmetic (no PSD, ERDF, FFT, sort): it only names shapes and
parameters and draws the per-curve parameters of C2 / C5, so that the CUDA path (tests, bench.py) and the
CPU oracle (tests) can be fed the same inputs without sharing code.  The per-curve draws follow SURVEY.md
8(d): parameter p of curve b is the uniform made from words (0, 1) of Philox4x32-10 with counter (p, 0, b, 2)
and key (seed lo, seed hi) -- a small generator of this module's own (neither the oracle's nor the
library's), so the workloads do not depend on any numpy version.
The paper measures on no public benchmark; these shapes stand in for its workloads (Table 1 / Table 2,
PAPER.md:261-270, :407-421; PTF-like and LSST-like cadences).  See DESIGN.md.
"""
import math

BPL, LOGNORMAL = 0, 1
_M32 = 0xFFFFFFFF


def _philox_words(seed, c0, c1, c2, c3):
    """Philox4x32-10 (published algorithm: Salmon et al. 2011), plain Python integers."""
    k0, k1 = seed & _M32, (seed >> 32) & _M32
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c0, 0xCD9E8D57 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & _M32, p1 & _M32, ((p0 >> 32) ^ c3 ^ k1) & _M32, p0 & _M32
        k0, k1 = (k0 + 0x9E3779B9) & _M32, (k1 + 0xBB67AE85) & _M32
    return c0, c1, c2, c3


def param_uniform(seed, p, b):
    """Uniform in (0, 1) for parameter number p of curve b (stream tag 2)."""
    w = _philox_words(seed, p, 0, b, 2)
    return (2 * ((w[0] << 20) + (w[1] >> 12)) + 1) * 2.0 ** -53


def _uniform(seed, p, lo, hi, n):
    return [lo + (hi - lo) * param_uniform(seed, p, b) for b in range(n)]


def _loguniform(seed, p, lo, hi, n):
    return [10.0 ** (math.log10(lo) + (math.log10(hi) - math.log10(lo)) * param_uniform(seed, p, b)) for b in range(n)]


def config(name, B=None):
    """Return dict(name, B, N, dt, oversample, dtype, max_iter, seed, grid_points, psd=[...], erdf=[...]).
    psd: list (length 1 or B) of dict(A, f_b, alpha_low, alpha_high), A = 0 -> unit-variance normalisation.
    erdf: list (length 1 or B) of dict(kind, lam_star, delta1, delta2, mu_log10, sigma_log10, lam_min, lam_max).
    B overrides the batch (a subset keeps the first B curves' parameters)."""
    name = name.upper()
    if name == "C1":  # PR1 reference, fp64
        c = dict(B=16, N=4096, dt=1.0, oversample=10, dtype="f64", max_iter=100, seed=0,
                 psd=[dict(A=0.0, f_b=1.0 / 300.0, alpha_low=1.0, alpha_high=2.0)],
                 erdf=[dict(kind=BPL, lam_star=0.1, delta1=0.4, delta2=2.4, lam_min=1e-4, lam_max=1.0)])
    elif name == "C2":  # PTF/iPTF-like
        Bf = 4096 if B is None else min(int(B), 4096)     # curve b's parameters do not depend on the subset size
        fb = _loguniform(2, 0, 1.0 / 1000.0, 1.0 / 50.0, Bf)
        c = dict(B=4096, N=2 ** 14, dt=1.0, oversample=10, dtype="f32", max_iter=200, seed=2,
                 psd=[dict(A=0.0, f_b=float(f), alpha_low=1.0, alpha_high=2.5) for f in fb],
                 erdf=[dict(kind=BPL, lam_star=10 ** -1.5, delta1=0.45, delta2=2.5, lam_min=1e-5, lam_max=1.0)])
    elif name == "C3":  # LSST-like
        c = dict(B=256, N=2 ** 20, dt=7.0, oversample=1, dtype="f32", max_iter=100, seed=3,
                 psd=[dict(A=0.0, f_b=1.0 / (365.0 * 5.0), alpha_low=1.0, alpha_high=2.5)],
                 erdf=[dict(kind=LOGNORMAL, mu_log10=-2.0, sigma_log10=0.7, lam_min=1e-5, lam_max=1.0)],
                 nbins=64)
    elif name == "C4":  # long baseline: the configuration the metric is quoted on
        c = dict(B=4, N=2 ** 26, dt=7.0, oversample=1, dtype="f32", max_iter=50, seed=4,
                 psd=[dict(A=0.0, f_b=1.0 / (365.0 * 1e3), alpha_low=1.0, alpha_high=2.0)],
                 erdf=[dict(kind=BPL, lam_star=0.05, delta1=0.2, delta2=2.2, lam_min=1e-6, lam_max=1.0)])
    elif name == "C5":  # parameter sweep
        Bf = 65536 if B is None else min(int(B), 65536)
        alo, ahi = _uniform(7, 0, 0.5, 1.5, Bf), _uniform(7, 1, 2.0, 3.0, Bf)
        fb = _loguniform(7, 2, 1e-3, 1e-1, Bf)
        d1, d2 = _uniform(7, 3, 0.1, 0.6, Bf), _uniform(7, 4, 2.0, 3.0, Bf)
        c = dict(B=65536, N=1024, dt=1.0, oversample=1, dtype="f32", max_iter=100, seed=7,
                 psd=[dict(A=0.0, f_b=float(fb[i]), alpha_low=float(alo[i]), alpha_high=float(ahi[i]))
                      for i in range(Bf)],
                 erdf=[dict(kind=BPL, lam_star=10 ** -1.5, delta1=float(d1[i]), delta2=float(d2[i]), lam_min=1e-5,
                            lam_max=1.0) for i in range(Bf)])
    else:
        raise ValueError(f"unknown config {name!r}")
    c["name"] = name
    c.setdefault("grid_points", 4096)
    c.setdefault("nbins", 0)
    if B is not None:
        B = int(B)
        if B > c["B"]:
            raise ValueError("subset larger than the configuration")
        c["B"] = B
        for k in ("psd", "erdf"):
            if len(c[k]) > 1:
                c[k] = c[k][:B]
    return c


def log_bin_edges(N, nbins=64):
    """Q19: integer edges j_e = ceil((N/2)^(e/nbins)), e = 0..nbins, deduplicated; last edge N/2 + 1."""
    half = N // 2
    raw = [int(math.ceil(half ** (e / nbins) - 1e-12)) for e in range(nbins + 1)]
    raw[0] = 1
    raw[-1] = half + 1
    out = []
    for j in raw:
        if not out or j > out[-1]:
            out.append(j)
    return out


def tiny(N=256, B=3, dtype="f64", oversample=1, kind=BPL, seed=11, max_iter=20):
    """A small generic case for smoke and edge tests."""
    erdf = (dict(kind=BPL, lam_star=0.1, delta1=0.4, delta2=2.4, lam_min=1e-4, lam_max=1.0) if kind == BPL else
            dict(kind=LOGNORMAL, mu_log10=-2.0, sigma_log10=0.7, lam_min=1e-5, lam_max=1.0))
    return dict(name="tiny", B=B, N=N, dt=1.0, oversample=oversample, dtype=dtype, max_iter=max_iter, seed=seed,
                grid_points=4096, nbins=0,
                psd=[dict(A=0.0, f_b=1.0 / 50.0, alpha_low=1.0, alpha_high=2.0)], erdf=[erdf])

"""Evidence for reading P2 of DESIGN.md (CPU, -m "not gpu"): BASELINE's ">= 99.9 % of samples equal in value to the
oracle's" is a property of a correct fp32 E13 step only up to N = 2^12.

The measurement: one E13 step (O6) computed with a TEXTBOOK LIBRARY FFT IN SINGLE PRECISION (scipy/pocketfft on
float32 -> complex64; not the product's kernels, not the oracle) from the oracle's own fp64 trajectory, compared in
value with the oracle's fp64 step on the same x_sim.  The fraction of equal values is set by the density of the keys
against the fp32 FFT error (near-ties flip), not by the implementation: at N = 2^14 it sits in a band around
0.997-0.999, below 0.999 for some steps, which is why tests/test_gpu_parity.py gates the product's fp32 one-step
figure at 0.995 there and only reports it above (every flip is separately proven to be a near-tie by the
eps-sortedness clause)."""
import numpy as np
import pytest

scipy_fft = pytest.importorskip("scipy.fft")

BPL = dict(kind=0, lam_star=0.1, delta1=0.4, delta2=2.4, lam_min=1e-4, lam_max=1.0)


def _one_step_fractions(orc, N, os_, seeds, steps):
    out = []
    for seed in seeds:
        srt, perm, _ = orc.erdf_sample_sorted(BPL, 4096, N, seed, 0, 0)
        an = orc.tk_generate(0.0, 1.0 / 300.0, 1.0, 2.0, N, 1.0, os_, seed, 0)["A_norm"]
        x = np.empty(N)
        x[perm] = srt
        for _ in range(steps):
            _, idx64, xnext64, _ = orc.e13_step(an, srt, perm, x)
            X = scipy_fft.rfft(x.astype(np.float32))
            assert X.dtype == np.complex64            # the library really computed in single precision
            m = np.abs(X)
            a32 = an.astype(np.float32)
            Xp = np.where(m > 0, a32 * X / np.where(m > 0, m, 1), a32).astype(np.complex64)
            xa32 = scipy_fft.irfft(Xp, n=N).astype(np.float32) + np.float32(0.0)
            idx32 = np.argsort(xa32, kind="stable")
            xn32 = np.empty(N)
            xn32[idx32] = srt
            out.append(float(np.mean(xn32 == xnext64)))
            x, perm = xnext64, idx64                  # follow the oracle's trajectory
    return out


def test_library_fp32_fft_one_step_band(orc):
    f12 = _one_step_fractions(orc, 4096, 10, (1, 2, 3), 6)
    f14 = _one_step_fractions(orc, 2 ** 14, 10, (1, 2, 3), 6) + _one_step_fractions(orc, 2 ** 14, 1, (1, 2, 3), 6)
    print(f"library complex64 FFT, one-step value-equal fraction: N=2^12 min {min(f12):.5f}; "
          f"N=2^14 min {min(f14):.5f} max {max(f14):.5f} mean {np.mean(f14):.5f}")
    assert min(f12) >= 0.999                     # BASELINE's figure holds at 2^12 ...
    assert 0.995 <= min(f14) < 0.999             # ... and not at 2^14, for a correct fp32 FFT
    assert max(f14) < 0.9999

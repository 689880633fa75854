// agnvar_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, single-threaded fp64 CPU statement of the hot path of Sartori et al. 2019
// (arXiv:1909.06374): Timmer & Koenig series + random draw from the ERDF + Emmanoulopoulos-style
// iterative amplitude adjustment.  It exists so that the CUDA library (paper_1909_06374_b200/csrc)
// can be checked against something that was written from the paper and is checkable by eye.
// It shares no code, header, table or constant generator with the CUDA path and neither includes
// the other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// leg may load it.
//
// Citations are to /root/reference/PAPER.md (line numbers) and to SURVEY.md section 8(c) readings
// (O1..O7, Q-numbers), which DESIGN.md restates.
//
// Pin status (tests/test_oracle_pins.py, all "-m 'not gpu'"):
//   orc_philox4x32_10      pinned: three published known-answer vectors
//   orc_u53 / normals      pinned: exact dyadic values; moments / KS against N(0,1)
//   orc_dft_naive          pinned: closed forms (delta, single tone, constant), linearity
//   orc_fft                pinned: vs orc_dft_naive for N<=256 incl. 5*2^k, Parseval, inverse round trip
//   orc_psd_bpl            pinned: asymptotic slopes, value at f_b = A/2, symmetric in the two slopes
//   orc_psd_unit_variance_A pinned: ensemble variance of TK series = 1
//   orc_tk_generate        pinned: ensemble-mean periodogram within 5% of PSD (1e4 realisations),
//                                  zero mean, Hermitian => real, crop position
//   orc_erdf_table/draw    pinned: KS vs closed-form CDF (delta2 = 2 delta1), vs erf (log-normal),
//                                  paper's ~10% / ~1.7% fractions
//   orc_stable_argsort     pinned: brute-force ranks on tiny inputs with ties
//   orc_e13_step/iterate   pinned: exact-permutation invariant, amplitude invariances (scale, DC),
//                                  |X'| == A_norm after the replace, restart reproducibility
//   orc_periodogram        pinned: Parseval identity A5, single tone, white noise
//   orc_delta_rms / orc_e13_iterate_delta   pinned: 0 at a fixed point, closed form for one swapped pair,
//                                  exactly 1 for x -> 10 x (the log is log10), threshold honoured
//   orc_structure_function pinned: brute force over all pairs, a^2 l^2 for a ramp, 2 sigma^2 (1 - cos) for a tone,
//                                  random-walk ensemble slope beta = (alpha - 1)/2 = 1/2, magnitude invariances
//   orc_delta_m_prob       pinned: brute force, 0 beyond 2.5 x the dynamic range, monotone in dm_ref
//   orc_sf_representative  pinned: by hand (Eq. 6)
//   orc_ensemble_sf        pinned: reduces to orc_structure_function for one curve, whole series, keep fraction 1;
//                                  brute force with the mask rebuilt from the (KAT-pinned) Philox words; pooled pair
//                                  count ~ p^2 (n_sub - l) B; unbiased for a random-walk ensemble
//   orc_moments            pinned: closed forms (two-point and uniform distributions), scipy.stats on random data
//   orc_slice_sample       pinned: one kept draw per chain (independent draws) KS-tested against the closed-form CDF
//                                  (delta2 = 2 delta1), erf (log-normal) and closed forms of tabulated densities
//                                  (triangle, two boxes with a zero-density gap), for step widths from 0.02 to 50 dex
//                                  and 1 to 64 stepping-out steps (the stationary law must not depend on them); the
//                                  paper's ~10% / ~1.7% fractions; support; a long single chain's
//                                  mean / variance against quadrature; prefix property of the chain layout
//
// Build: g++ -O2 -std=c++17 -shared -fPIC -o liboracle.so agnvar_oracle.cpp   (oracle/build.py)

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>

typedef std::complex<double> cd;
static const double kPi = 3.14159265358979323846264338327950288;

extern "C" {

// ----------------------------------------------------------------------------------------------
// O1. Philox4x32-10 (the paper only names cuRAND).
// Ten rounds; round: p0 = 0xD2511F53*c0, p1 = 0xCD9E8D57*c2 (64-bit products),
// c <- (hi(p1)^c1^k0, lo(p1), hi(p0)^c3^k1, lo(p0)); key bumped by (0x9E3779B9, 0xBB67AE85) after
// each round.
// ----------------------------------------------------------------------------------------------
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Stream layout (O1): key = (seed lo, seed hi); counter = (i lo, i hi, curve b, stream tag).
// tag 0 = TK normals (i = frequency index j), tag 1 = ERDF uniforms (i = n >> 1).
void orc_philox_stream(uint64_t seed, uint64_t i, uint32_t b, uint32_t tag, uint32_t out[4]) {
    uint32_t ctr[4] = {(uint32_t)i, (uint32_t)(i >> 32), b, tag};
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    orc_philox4x32_10(ctr, key, out);
}

// Uniform in (0,1) from two words: u = (2*(wa*2^20 + (wb>>12)) + 1) * 2^-53  (O1). Exact in fp64.
double orc_u53(uint32_t wa, uint32_t wb) {
    uint64_t m = ((uint64_t)wa << 20) + (uint64_t)(wb >> 12);
    return (double)(2 * m + 1) * (1.0 / 9007199254740992.0);
}

// TK normals from one Philox call (O1): u1 from words (0,1), u2 from words (2,3);
// g_re = sqrt(-2 ln u1) cos(2 pi u2), g_im = sqrt(-2 ln u1) sin(2 pi u2).
void orc_tk_normal_pair(uint64_t seed, uint64_t j, uint32_t b, double* g_re, double* g_im) {
    uint32_t w[4];
    orc_philox_stream(seed, j, b, 0u, w);
    double u1 = orc_u53(w[0], w[1]);
    double u2 = orc_u53(w[2], w[3]);
    double r = std::sqrt(-2.0 * std::log(u1));
    *g_re = r * std::cos(2.0 * kPi * u2);
    *g_im = r * std::sin(2.0 * kPi * u2);
}

// ----------------------------------------------------------------------------------------------
// Discrete Fourier transform, the plain definition (Eq. A1, with the usual sign
// convention: sign=-1 forward, sign=+1 inverse, no normalisation; SURVEY O5 on the sign).
//   out[k] = sum_m in[m] * exp(sign * 2 pi i * m k / n)
// The angle index (m*k mod n) is reduced exactly in integers before the trigonometric call.
// ----------------------------------------------------------------------------------------------
void orc_dft_naive(const double* re, const double* im, int64_t n, int sign, double* ore, double* oim) {
    std::vector<cd> w((size_t)n);
    for (int64_t q = 0; q < n; ++q) {
        double a = (double)sign * 2.0 * kPi * (double)q / (double)n;
        w[(size_t)q] = cd(std::cos(a), std::sin(a));
    }
    for (int64_t k = 0; k < n; ++k) {
        cd acc(0.0, 0.0);
        for (int64_t m = 0; m < n; ++m) {
            int64_t q = (int64_t)(((__int128)m * (__int128)k) % (__int128)n);
            acc += cd(re[m], im ? im[m] : 0.0) * w[(size_t)q];
        }
        ore[k] = acc.real();
        oim[k] = acc.imag();
    }
}

}  // extern "C"

// ----------------------------------------------------------------------------------------------
// Textbook recursive FFT (decimation in time, radix 2 while the length is even; the plain DFT
// sum for what is left, i.e. an odd factor such as the 5 in M = 10 N, or n <= 4).
// tw holds exp(sign 2 pi i q / n_top) for q in [0, n_top/2) when n_top is even (the other half
// is minus the first), or for all q when n_top is odd.
// ----------------------------------------------------------------------------------------------
namespace {

struct Twiddles {
    std::vector<cd> w;
    size_t n_top;
    bool half;
    Twiddles(size_t n, int sign) : n_top(n), half(n % 2 == 0 && n > 1) {
        size_t cnt = half ? n / 2 : n;
        w.resize(cnt);
        for (size_t q = 0; q < cnt; ++q) {
            double a = (double)sign * 2.0 * kPi * (double)q / (double)n;
            w[q] = cd(std::cos(a), std::sin(a));
        }
    }
    inline cd at(size_t q) const {  // q in [0, n_top)
        if (!half) return w[q];
        return q < n_top / 2 ? w[q] : -w[q - n_top / 2];
    }
};

void fft_rec(const cd* in, size_t stride, cd* out, size_t n, const Twiddles& tw, size_t tw_stride) {
    if (n <= 4 || (n % 2) != 0) {
        for (size_t k = 0; k < n; ++k) {
            cd acc(0.0, 0.0);
            for (size_t m = 0; m < n; ++m) acc += in[m * stride] * tw.at(((m * k) % n) * tw_stride);
            out[k] = acc;
        }
        return;
    }
    size_t h = n / 2;
    fft_rec(in, 2 * stride, out, h, tw, 2 * tw_stride);               // even samples
    fft_rec(in + stride, 2 * stride, out + h, h, tw, 2 * tw_stride);  // odd samples
    for (size_t k = 0; k < h; ++k) {
        cd e = out[k];
        cd o = out[k + h] * tw.at(k * tw_stride);
        out[k] = e + o;
        out[k + h] = e - o;
    }
}

// BASELINE north_star: "a naive O(N^2) DFT for tiny N and a textbook recursive FFT otherwise".
// n <= 256 -> the definition (orc_dft_naive); larger -> fft_rec.  force_recursive lets the pin
// tests compare fft_rec against the definition on the sizes where both are affordable.
void fft_complex(const std::vector<cd>& in, std::vector<cd>& out, int sign, bool force_recursive = false) {
    size_t n = in.size();
    out.resize(n);
    if (n == 0) return;
    if (n <= 256 && !force_recursive) {
        std::vector<double> re(n), im(n), ore(n), oim(n);
        for (size_t i = 0; i < n; ++i) { re[i] = in[i].real(); im[i] = in[i].imag(); }
        orc_dft_naive(re.data(), im.data(), (int64_t)n, sign, ore.data(), oim.data());
        for (size_t i = 0; i < n; ++i) out[i] = cd(ore[i], oim[i]);
        return;
    }
    Twiddles tw(n, sign);
    fft_rec(in.data(), 1, out.data(), n, tw, 1);
}

// Forward DFT of a real series; returns bins j = 0..n/2 (Eq. A1 and the list of Fourier
// frequencies).
void rfft(const double* x, size_t n, std::vector<cd>& X) {
    std::vector<cd> in(n), out;
    for (size_t i = 0; i < n; ++i) in[i] = cd(x[i], 0.0);
    fft_complex(in, out, -1);
    X.assign(out.begin(), out.begin() + (n / 2 + 1));
}

// Inverse of the above: Hermitian extension, inverse DFT, factor 1/n, real part.
void irfft(const std::vector<cd>& X, size_t n, double* x) {
    std::vector<cd> in(n), out;
    for (size_t j = 0; j <= n / 2; ++j) in[j] = X[j];
    for (size_t j = n / 2 + 1; j < n; ++j) in[j] = std::conj(X[n - j]);
    fft_complex(in, out, +1);
    for (size_t i = 0; i < n; ++i) x[i] = out[i].real() / (double)n;
}

// Eq. 3: PSD(f) = A [ (f/f_b)^a_low + (f/f_b)^a_high ]^-1
inline double psd_shape(double f, double f_b, double a_lo, double a_hi) {
    double r = f / f_b;
    return 1.0 / (std::pow(r, a_lo) + std::pow(r, a_hi));
}

// Eq. 1 / Eq. 2 as a function of u = log10(lambda), up to the constant xi*.
// kind 0: broken power law [ (l/l*)^d1 + (l/l*)^d2 ]^-1 ; kind 1: log-normal in log10(lambda).
inline double erdf_xi(int kind, double u, double lam_star, double d1, double d2, double mu, double sigma) {
    if (kind == 0) {
        double r = std::pow(10.0, u) / lam_star;
        return 1.0 / (std::pow(r, d1) + std::pow(r, d2));
    }
    double z = (u - mu) / sigma;
    return std::exp(-0.5 * z * z);
}

}  // namespace

extern "C" {

// Always the recursive FFT (never the naive branch), so that "orc_fft vs orc_dft_naive" is a real pin.
void orc_fft(const double* re, const double* im, int64_t n, int sign, double* ore, double* oim) {
    std::vector<cd> in((size_t)n), out;
    for (int64_t i = 0; i < n; ++i) in[(size_t)i] = cd(re[i], im ? im[i] : 0.0);
    fft_complex(in, out, sign, true);
    for (int64_t i = 0; i < n; ++i) { ore[i] = out[(size_t)i].real(); oim[i] = out[(size_t)i].imag(); }
}

void orc_rfft(const double* x, int64_t n, double* Xre, double* Xim) {
    std::vector<cd> X;
    rfft(x, (size_t)n, X);
    for (int64_t j = 0; j <= n / 2; ++j) { Xre[j] = X[(size_t)j].real(); Xim[j] = X[(size_t)j].imag(); }
}

void orc_irfft(const double* Xre, const double* Xim, int64_t n, double* x) {
    std::vector<cd> X((size_t)(n / 2 + 1));
    for (int64_t j = 0; j <= n / 2; ++j) X[(size_t)j] = cd(Xre[j], Xim[j]);
    irfft(X, (size_t)n, x);
}

// ----------------------------------------------------------------------------------------------
// O2. PSD (Eq. 3) at given frequencies.
// ----------------------------------------------------------------------------------------------
void orc_psd_bpl(const double* f, int64_t n, double A, double f_b, double a_lo, double a_hi, double* out) {
    for (int64_t i = 0; i < n; ++i) out[i] = A * psd_shape(f[i], f_b, a_lo, a_hi);
}

// Q4: "A set so the Gaussian series has unit variance": with f_j = j/(M dt) and
// s_j the shape of Eq. 3, A = M^2 / (2 sum_{1<=j<M/2} s_j + s_{M/2}) makes the expected sample
// variance of the length-M TK series equal to 1 (the realisation is not rescaled).
double orc_psd_unit_variance_A(int64_t M, double dt, double f_b, double a_lo, double a_hi) {
    double acc = 0.0;
    for (int64_t j = 1; j < M / 2; ++j) acc += 2.0 * psd_shape((double)j / ((double)M * dt), f_b, a_lo, a_hi);
    acc += psd_shape((double)(M / 2) / ((double)M * dt), f_b, a_lo, a_hi);
    return (double)M * (double)M / acc;
}

// ----------------------------------------------------------------------------------------------
// O3. Timmer & Koenig (described there by reference only).
// X_0 = 0; X_j = sqrt(S_j/2) (g_re + i g_im), 1 <= j < M/2; X_{M/2} = sqrt(S_{M/2}) g_re;
// x = inverse real DFT of length M with 1/M.  Oversampling (BASELINE C1): simulate
// M = oversample*N samples and keep the central N: x_norm = x[(M-N)/2 .. (M-N)/2 + N - 1].
// A_norm = |DFT_N(x_norm)|, j = 0..N/2 (O5 / Q2).
// A <= 0 requests the unit-variance normalisation above.
// Xre/Xim (M/2+1), x_full (M), x_norm (N), A_norm (N/2+1) may each be NULL.
// ----------------------------------------------------------------------------------------------
int orc_tk_generate(double A, double f_b, double a_lo, double a_hi, int64_t N, double dt, int oversample,
                    uint64_t seed, uint32_t b, double* Xre, double* Xim, double* x_full, double* x_norm,
                    double* A_norm) {
    if (N < 2 || oversample < 1) return 1;
    size_t M = (size_t)N * (size_t)oversample;
    if (A <= 0.0) A = orc_psd_unit_variance_A((int64_t)M, dt, f_b, a_lo, a_hi);
    std::vector<cd> X(M / 2 + 1);
    X[0] = cd(0.0, 0.0);
    for (size_t j = 1; j <= M / 2; ++j) {
        double f = (double)j / ((double)M * dt);
        double S = A * psd_shape(f, f_b, a_lo, a_hi);
        double gr, gi;
        orc_tk_normal_pair(seed, (uint64_t)j, b, &gr, &gi);
        if (j < M / 2) X[j] = std::sqrt(0.5 * S) * cd(gr, gi);
        else X[j] = cd(std::sqrt(S) * gr, 0.0);
    }
    if (Xre && Xim) for (size_t j = 0; j <= M / 2; ++j) { Xre[j] = X[j].real(); Xim[j] = X[j].imag(); }
    std::vector<double> x(M);
    irfft(X, M, x.data());
    if (x_full) std::memcpy(x_full, x.data(), M * sizeof(double));
    size_t off = (M - (size_t)N) / 2;
    if (x_norm) std::memcpy(x_norm, x.data() + off, (size_t)N * sizeof(double));
    if (A_norm) {
        std::vector<cd> Y;
        rfft(x.data() + off, (size_t)N, Y);
        for (size_t j = 0; j <= (size_t)N / 2; ++j) A_norm[j] = std::abs(Y[j]);
    }
    return 0;
}

// ----------------------------------------------------------------------------------------------
// O4. ERDF table and draw.  Q10: Eq. 1/2 give xi = dN/dlog(lambda) and the code samples dN/dlambda
// "uniformly in linear space": lambda has density xi/(lambda ln 10), i.e.
// u = log10(lambda) has density proportional to xi(10^u) on [log10 lam_min, log10 lam_max].
// Table: u_k = u_lo + k D, k = 0..G-1; p_k = xi(10^{u_k}); C_0 = 0, C_k = C_{k-1} + (p_k+p_{k-1}) D/2;
// C divided by C_{G-1}.
// ----------------------------------------------------------------------------------------------
void orc_erdf_table(int kind, double lam_star, double d1, double d2, double mu, double sigma, double lam_min,
                    double lam_max, int64_t G, double* u, double* p, double* C) {
    double u_lo = std::log10(lam_min), u_hi = std::log10(lam_max);
    double D = (u_hi - u_lo) / (double)(G - 1);
    for (int64_t k = 0; k < G; ++k) {
        u[k] = u_lo + (double)k * D;
        p[k] = erdf_xi(kind, u[k], lam_star, d1, d2, mu, sigma);
    }
    C[0] = 0.0;
    for (int64_t k = 1; k < G; ++k) C[k] = C[k - 1] + 0.5 * (p[k] + p[k - 1]) * D;
    double tot = C[G - 1];
    for (int64_t k = 0; k < G; ++k) C[k] /= tot;
}

// Draw (O4): U from Philox stream tag 1 (sample n uses words (0,1) of call i = n>>1 if n is even,
// words (2,3) if odd); find k with C_k <= U < C_{k+1} (U < C_1 -> k = 0); u = u_k + (U - C_k) /
// (C_{k+1} - C_k) * D; lambda = 10^u, rounded to the output type (dtype 0: fp32, 1: fp64).
void orc_erdf_draw(int kind, double lam_star, double d1, double d2, double mu, double sigma, double lam_min,
                   double lam_max, int64_t G, int64_t N, uint64_t seed, uint32_t b, int dtype, double* lam,
                   double* U_out) {
    std::vector<double> u((size_t)G), p((size_t)G), C((size_t)G);
    orc_erdf_table(kind, lam_star, d1, d2, mu, sigma, lam_min, lam_max, G, u.data(), p.data(), C.data());
    double D = (std::log10(lam_max) - std::log10(lam_min)) / (double)(G - 1);
    for (int64_t n = 0; n < N; ++n) {
        uint32_t w[4];
        orc_philox_stream(seed, (uint64_t)(n >> 1), b, 1u, w);
        double U = (n & 1) ? orc_u53(w[2], w[3]) : orc_u53(w[0], w[1]);
        // largest k in [0, G-2] with C_k <= U
        int64_t lo = 0, hi = G - 1;  // invariant: C[lo] <= U < C[hi]  (C[0] = 0 < U < 1 = C[G-1])
        while (hi - lo > 1) {
            int64_t mid = (lo + hi) / 2;
            if (C[(size_t)mid] <= U) lo = mid; else hi = mid;
        }
        double uu = u[(size_t)lo] + (U - C[(size_t)lo]) / (C[(size_t)lo + 1] - C[(size_t)lo]) * D;
        double l = std::pow(10.0, uu);
        if (dtype == 0) l = (double)(float)l;
        lam[n] = l;
        if (U_out) U_out[n] = U;
    }
}

// ----------------------------------------------------------------------------------------------
// Stable ascending argsort: idx[r] = position of the r-th smallest key, ties keep index order
// (O6 step 4; tie-break is part of the result).  Keys are compared with '<'.
// ----------------------------------------------------------------------------------------------
void orc_stable_argsort(const double* x, int64_t n, uint32_t* idx) {
    std::vector<uint32_t> v((size_t)n);
    std::iota(v.begin(), v.end(), 0u);
    std::stable_sort(v.begin(), v.end(), [x](uint32_t a, uint32_t c) { return x[a] < x[c]; });
    std::memcpy(idx, v.data(), (size_t)n * sizeof(uint32_t));
}

// Brute-force rank (pin for the above): rank[t] = #{s: x[s] < x[t]} + #{s < t: x[s] == x[t]}.
void orc_rank_bruteforce(const double* x, int64_t n, uint32_t* rank) {
    for (int64_t t = 0; t < n; ++t) {
        uint32_t r = 0;
        for (int64_t s = 0; s < n; ++s) r += (x[s] < x[t]) || (x[s] == x[t] && s < t);
        rank[t] = r;
    }
}

// ----------------------------------------------------------------------------------------------
// O6. One E13 / IAAFT iteration (steps in SURVEY 8(c) O6):
//  1. X = DFT_N(x_sim)
//  2. j = 0..N/2: m = |X_j|; X'_j = A_norm_j X_j / m if m > 0 else A_norm_j; DC and Nyquist real.
//  3. x_adj = IDFT_N(X') with 1/N; x_adj += 0.0 (turns -0 into +0, Q13)
//  4. idx_new = stable argsort of x_adj
//  5. changed = #{r: idx_new[r] != idx_old[r]}; x_next[idx_new[r]] = sorted[r]
// ----------------------------------------------------------------------------------------------
void orc_e13_step(int64_t N, const double* A_norm, const double* sorted, const uint32_t* idx_old,
                  const double* x_sim, double* x_adj, uint32_t* idx_new, double* x_next, int64_t* changed) {
    size_t n = (size_t)N;
    std::vector<cd> X;
    rfft(x_sim, n, X);
    for (size_t j = 0; j <= n / 2; ++j) {
        cd v = X[j];
        if (j == 0 || j == n / 2) v = cd(v.real(), 0.0);
        double m = std::hypot(v.real(), v.imag());
        X[j] = (m > 0.0) ? (A_norm[j] * v / m) : cd(A_norm[j], 0.0);
    }
    std::vector<double> xa(n);
    irfft(X, n, xa.data());
    for (size_t i = 0; i < n; ++i) xa[i] = xa[i] + 0.0;
    std::vector<uint32_t> idx(n);
    orc_stable_argsort(xa.data(), N, idx.data());
    int64_t ch = 0;
    for (size_t r = 0; r < n; ++r) ch += (idx[r] != idx_old[r]);
    if (x_next) for (size_t r = 0; r < n; ++r) x_next[idx[r]] = sorted[r];
    if (x_adj) std::memcpy(x_adj, xa.data(), n * sizeof(double));
    if (idx_new) std::memcpy(idx_new, idx.data(), n * sizeof(uint32_t));
    if (changed) *changed = ch;
}

// Full loop for one curve.  perm: in = perm0 (argsort of the raw draw; x_sim,1[perm0[r]] = sorted[r],
// Q15), out = final permutation.  Stops when changed == 0 (iters_used = k) or after max_iter
// iterations (iters_used = max_iter).  changed_hist (max_iter entries) gets the count of every
// executed iteration and 0 afterwards.  x_adj_last: x_adj of the last executed iteration.
int orc_e13_iterate(int64_t N, const double* A_norm, const double* sorted, uint32_t* perm, double* x,
                    int max_iter, int32_t* iters_used, int64_t* changed_hist, double* x_adj_last) {
    if (N < 2 || max_iter < 1) return 1;
    size_t n = (size_t)N;
    std::vector<double> xs(n), xn(n), xa(n);
    std::vector<uint32_t> idx(n);
    for (size_t r = 0; r < n; ++r) xs[perm[r]] = sorted[r];
    if (changed_hist) for (int k = 0; k < max_iter; ++k) changed_hist[k] = 0;
    int used = max_iter;
    for (int k = 1; k <= max_iter; ++k) {
        int64_t ch = 0;
        orc_e13_step(N, A_norm, sorted, perm, xs.data(), xa.data(), idx.data(), xn.data(), &ch);
        std::memcpy(perm, idx.data(), n * sizeof(uint32_t));
        xs.swap(xn);
        if (changed_hist) changed_hist[k - 1] = ch;
        if (ch == 0) { used = k; break; }
    }
    std::memcpy(x, xs.data(), n * sizeof(double));
    if (x_adj_last) std::memcpy(x_adj_last, xa.data(), n * sizeof(double));
    if (iters_used) *iters_used = used;
    return 0;
}

// ----------------------------------------------------------------------------------------------
// O7. Periodogram, j = 1..N/2 (DC excluded).  norm 0: Eq. A2 P_j = (2/N^2)|X_j|^2;
// norm 1: Eq. A4 P_j = (2 dt / (mu^2 N)) |X_j|^2, mu = sample mean.
// Binned variant (Q19): bin e = arithmetic mean of P_j for edges[e] <= j < edges[e+1]; the last
// bin is closed at N/2 (edges[nb] may equal N/2 or N/2+1).
// ----------------------------------------------------------------------------------------------
void orc_periodogram(const double* x, int64_t N, double dt, int norm, double* P) {
    std::vector<cd> X;
    rfft(x, (size_t)N, X);
    double scale;
    if (norm == 0) scale = 2.0 / ((double)N * (double)N);
    else {
        double mu = 0.0;
        for (int64_t i = 0; i < N; ++i) mu += x[i];
        mu /= (double)N;
        scale = 2.0 * dt / (mu * mu * (double)N);
    }
    for (int64_t j = 1; j <= N / 2; ++j) P[j - 1] = scale * std::norm(X[(size_t)j]);
}

void orc_periodogram_binned(const double* x, int64_t N, double dt, int norm, int nb, const int64_t* edges,
                            double* out, int64_t* counts) {
    std::vector<double> P((size_t)(N / 2));
    orc_periodogram(x, N, dt, norm, P.data());
    for (int e = 0; e < nb; ++e) {
        int64_t j0 = edges[e], j1 = edges[e + 1];
        if (e == nb - 1 && j1 < N / 2 + 1) j1 = N / 2 + 1;
        if (j1 > N / 2 + 1) j1 = N / 2 + 1;
        double acc = 0.0;
        for (int64_t j = j0; j < j1; ++j) acc += P[(size_t)(j - 1)];
        counts[e] = j1 - j0;
        out[e] = (j1 > j0) ? acc / (double)(j1 - j0) : 0.0;
    }
}

// ----------------------------------------------------------------------------------------------
// NEXT-1. The paper's own convergence measure (Eq. 4):
//   delta_i = rms[ log( x_i(t_n) / x_{i-1}(t_n) ) ], n = 1..N,
// "log" read as log10 (the paper speaks in dex; Q14).  rms = sqrt of the mean of the squares.
// ----------------------------------------------------------------------------------------------
double orc_delta_rms(const double* x_new, const double* x_old, int64_t n) {
    double acc = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        double d = std::log10(x_new[i] / x_old[i]);
        acc += d * d;
    }
    return std::sqrt(acc / (double)n);
}

// The loop of orc_e13_iterate with the paper's stopping rule added: after iteration k, delta_k is Eq. 4 between
// x_sim,k+1 and x_sim,k; the curve stops at the first k with changed == 0 or (threshold > 0 and delta_k <= threshold).
// delta_hist (max_iter entries): delta_k of every executed iteration, 0 afterwards.
int orc_e13_iterate_delta(int64_t N, const double* A_norm, const double* sorted, uint32_t* perm, double* x,
                          int max_iter, double threshold, int32_t* iters_used, int64_t* changed_hist,
                          double* delta_hist) {
    if (N < 2 || max_iter < 1) return 1;
    size_t n = (size_t)N;
    std::vector<double> xs(n), xn(n), xa(n);
    std::vector<uint32_t> idx(n);
    for (size_t r = 0; r < n; ++r) xs[perm[r]] = sorted[r];
    for (int k = 0; k < max_iter; ++k) {
        if (changed_hist) changed_hist[k] = 0;
        if (delta_hist) delta_hist[k] = 0.0;
    }
    int used = max_iter;
    for (int k = 1; k <= max_iter; ++k) {
        int64_t ch = 0;
        orc_e13_step(N, A_norm, sorted, perm, xs.data(), xa.data(), idx.data(), xn.data(), &ch);
        double delta = orc_delta_rms(xn.data(), xs.data(), N);
        std::memcpy(perm, idx.data(), n * sizeof(uint32_t));
        xs.swap(xn);
        if (changed_hist) changed_hist[k - 1] = ch;
        if (delta_hist) delta_hist[k - 1] = delta;
        if (ch == 0 || (threshold > 0.0 && delta <= threshold)) { used = k; break; }
    }
    std::memcpy(x, xs.data(), n * sizeof(double));
    if (iters_used) *iters_used = used;
    return 0;
}

// ----------------------------------------------------------------------------------------------
// NEXT-2. Structure function (Eq. A6) of an evenly sampled series at integer lags l (tau = l dt):
//   SF(tau)^2 = (1/P) sum over the P = N - l pairs (i, j = i + l) of [ x(t_i) - x(t_j) ]^2 .
// mag != 0: the series is first converted to magnitudes, m = -2.5 log10(x) (for a constant
// bolometric correction m(t2) - m(t1) = -2.5 log[L(t2)/L(t1)]; the zero point cancels in the differences).
// A lag with no pair (l >= N) gets sf2 = 0, pairs = 0.
// ----------------------------------------------------------------------------------------------
void orc_structure_function(const double* x, int64_t N, const int64_t* lags, int nlags, int mag, double* sf2,
                            int64_t* pairs) {
    std::vector<double> v((size_t)N);
    for (int64_t i = 0; i < N; ++i) v[(size_t)i] = mag ? -2.5 * std::log10(x[i]) : x[i];
    for (int q = 0; q < nlags; ++q) {
        const int64_t l = lags[q];
        double acc = 0.0;
        int64_t P = 0;
        for (int64_t i = 0; i + l < N; ++i) {
            double d = v[(size_t)i] - v[(size_t)(i + l)];
            acc += d * d;
            ++P;
        }
        sf2[q] = P > 0 ? acc / (double)P : 0.0;
        if (pairs) pairs[q] = P;
    }
}

// Representative structure function (Eq. 6): SF_rep(tau)^2 = mean over the N_sim realisations of
// SF_i(tau)^2; its standard error from the scatter of the SF_i^2 (sample standard deviation / sqrt(N_sim)).
// sf2: [nsim][nlags] row-major.
void orc_sf_representative(const double* sf2, int nsim, int nlags, double* mean, double* stderr_) {
    for (int q = 0; q < nlags; ++q) {
        double m = 0.0;
        for (int i = 0; i < nsim; ++i) m += sf2[(size_t)i * nlags + q];
        m /= (double)nsim;
        double var = 0.0;
        for (int i = 0; i < nsim; ++i) {
            double d = sf2[(size_t)i * nlags + q] - m;
            var += d * d;
        }
        mean[q] = m;
        if (stderr_) stderr_[q] = nsim > 1 ? std::sqrt(var / (double)(nsim - 1) / (double)nsim) : 0.0;
    }
}

// P(|dm| > dm_ref given tau) (Figs 16-17): for each lag, the number of pairs separated by that lag
// with |m_i - m_j| > dm_ref divided by the number of pairs considered, m = m_zero - 2.5 log10(x).
// use_cut != 0 (Fig. 17): every point with m > m_cut is replaced by the upper limit m_cut, and only pairs in which
// at least one point is detected (m <= m_cut) are considered.
// prob: [nlags][nref]; considered: [nlags] (may be NULL).  No pair considered -> probabilities 0.
void orc_delta_m_prob(const double* x, int64_t N, const int64_t* lags, int nlags, const double* dm_ref, int nref,
                      double m_zero, int use_cut, double m_cut, double* prob, int64_t* considered) {
    std::vector<double> m((size_t)N);
    std::vector<char> det((size_t)N);
    for (int64_t i = 0; i < N; ++i) {
        double mi = m_zero - 2.5 * std::log10(x[i]);
        det[(size_t)i] = (!use_cut || mi <= m_cut) ? 1 : 0;
        if (use_cut && mi > m_cut) mi = m_cut;
        m[(size_t)i] = mi;
    }
    for (int q = 0; q < nlags; ++q) {
        const int64_t l = lags[q];
        std::vector<int64_t> cnt((size_t)nref, 0);
        int64_t P = 0;
        for (int64_t i = 0; i + l < N; ++i) {
            if (!(det[(size_t)i] || det[(size_t)(i + l)])) continue;
            ++P;
            double d = std::fabs(m[(size_t)i] - m[(size_t)(i + l)]);
            for (int r = 0; r < nref; ++r) cnt[(size_t)r] += (d > dm_ref[r]);
        }
        for (int r = 0; r < nref; ++r) prob[(size_t)q * nref + r] = P > 0 ? (double)cnt[(size_t)r] / (double)P : 0.0;
        if (considered) considered[q] = P;
    }
}

// ----------------------------------------------------------------------------------------------
// NEXT-4. Ensemble structure function of sparsely sampled sub-segments (PAPER.md:253-259 sec. 3.2.5-3.2.6, :276,
// Fig. 7-8): from every light curve a CONSECUTIVE sub-sample of n_sub points is selected at a random position, the
// sub-sample is masked to mimic sparse measurements (a random fraction `keep` of its points is kept: 0.5 %, 1 %, 10 %
// in Fig. 8), and the SF at lag l is Eq. A6 over ALL pairs of kept points separated by l, in all the curves at once
// ("considering simultaneously all the pairs of data points separated by a corresponding time lag, in all the sources").
// The paper does not say how the positions and the mask are drawn; reading (Q23): Philox stream tag 3, call 0
// of curve b: offset_b = floor(u (N - n_sub + 1)), u from words (0, 1); tag 4: point j of the sub-sample is kept iff
// u_j < keep, u_j from call j >> 1 of curve b, words (0, 1) if j is even, (2, 3) if odd.
// x: [B][N] row-major.  sf2[q] = pooled mean (0 if no pair), pairs[q] = pooled number of pairs; offsets[b] may be NULL.
// ----------------------------------------------------------------------------------------------
void orc_ensemble_sf(const double* x, int64_t B, int64_t N, int64_t n_sub, double keep, uint64_t seed, uint32_t curve0,
                     const int64_t* lags, int nlags, int mag, double* sf2, int64_t* pairs, int64_t* offsets) {
    std::vector<double> acc((size_t)nlags, 0.0);
    std::vector<int64_t> cnt((size_t)nlags, 0);
    std::vector<double> v((size_t)n_sub);
    std::vector<char> kept((size_t)n_sub);
    for (int64_t b = 0; b < B; ++b) {
        uint32_t w[4];
        orc_philox_stream(seed, 0, curve0 + (uint32_t)b, 3u, w);
        const int64_t off = (int64_t)std::floor(orc_u53(w[0], w[1]) * (double)(N - n_sub + 1));
        if (offsets) offsets[b] = off;
        for (int64_t j = 0; j < n_sub; ++j) {
            orc_philox_stream(seed, (uint64_t)(j >> 1), curve0 + (uint32_t)b, 4u, w);
            const double u = (j & 1) ? orc_u53(w[2], w[3]) : orc_u53(w[0], w[1]);
            kept[(size_t)j] = (u < keep) ? 1 : 0;
            const double xv = x[(size_t)b * (size_t)N + (size_t)(off + j)];
            v[(size_t)j] = mag ? -2.5 * std::log10(xv) : xv;
        }
        for (int q = 0; q < nlags; ++q) {
            const int64_t l = lags[q];
            for (int64_t j = 0; j + l < n_sub; ++j) {
                if (!(kept[(size_t)j] && kept[(size_t)(j + l)])) continue;
                const double d = v[(size_t)j] - v[(size_t)(j + l)];
                acc[(size_t)q] += d * d;
                cnt[(size_t)q] += 1;
            }
        }
    }
    for (int q = 0; q < nlags; ++q) {
        sf2[q] = cnt[(size_t)q] > 0 ? acc[(size_t)q] / (double)cnt[(size_t)q] : 0.0;
        if (pairs) pairs[q] = cnt[(size_t)q];
    }
}

// Moments of the value distribution of a series (the TK95 output-PDF check of sec. 3.2.1 / Fig. 2):
// mean, variance (1/N), skewness m3 / m2^1.5, excess kurtosis m4 / m2^2 - 3, central moments m_k = (1/N) sum (x - mean)^k.
void orc_moments(const double* x, int64_t N, double out[4]) {
    double mu = 0.0;
    for (int64_t i = 0; i < N; ++i) mu += x[i];
    mu /= (double)N;
    double m2 = 0.0, m3 = 0.0, m4 = 0.0;
    for (int64_t i = 0; i < N; ++i) {
        const double d = x[i] - mu, d2 = d * d;
        m2 += d2; m3 += d2 * d; m4 += d2 * d2;
    }
    m2 /= (double)N; m3 /= (double)N; m4 /= (double)N;
    out[0] = mu;
    out[1] = m2;
    out[2] = m2 > 0.0 ? m3 / (m2 * std::sqrt(m2)) : 0.0;
    out[3] = m2 > 0.0 ? m4 / (m2 * m2) - 3.0 : 0.0;
}

// ----------------------------------------------------------------------------------------------
// NEXT-3. Slice sampling (Neal 2003, Ann. Statist. 31, 705), the paper's sampler for the random draw
// ("for the random draw step we apply slice sampling (Neal 2003) from a normalised ERDF ...
// additional functional forms can be added if needed"; PAPER.md:164 names it as what limits the running time).
// The paper gives no detail beyond the citation; this is Neal's univariate update with the "stepping out"
// procedure (his Fig. 3) followed by the "shrinkage" procedure (his Fig. 5), applied to u = log10(lambda), whose
// density g(u) is proportional to xi(10^u) on [log10 lam_min, log10 lam_max] and 0 outside (reading Q10).
//
// density kinds: 0 / 1 = Eq. 1 / Eq. 2 (erdf_xi above); 2 = an arbitrary un-normalised density given as a table
// gtab[0..G-1] >= 0 on the uniform grid u_k = u_lo + k D, linearly interpolated ("additional functional forms").
//
// Reading Q24 for what the paper leaves open:
//   chains   `chains` independent Markov chains per curve; chain c starts at x = u_lo + U (u_hi - u_lo), makes
//            burn_in + (N / chains) * thin updates and keeps every thin-th state after the burn-in; the j-th kept
//            state of chain c is sample n = j * chains + c (N must be a multiple of chains).
//   uniforms Philox stream tag 5, counter (call, chain c, curve b, 5): the chain's uniform number q is u53 of words
//            (0,1) of call q >> 1 if q is even, of words (2,3) if odd; a chain uses its uniforms in order.
//   update   y = g(x) U;  U: L = x - w U, R = L + w;  V: J = floor(m V), K = (m - 1) - J;
//            while J > 0 and y < g(L): L -= w, J -= 1;   while K > 0 and y < g(R): R += w, K -= 1;
//            repeat: U: x1 = L + U (R - L); accept if y < g(x1), else L = x1 if x1 < x, else R = x1.
//            (At most 1000 shrinkage draws, then the chain stays at x: only reachable where g = 0 around x.)
//   output   lambda = 10^x rounded to the output type.
// Plain arithmetic, one rounding per operation, in the order written (built with -ffp-contract=off).
// ----------------------------------------------------------------------------------------------
static double slice_density(int kind, double u, double lam_star, double d1, double d2, double mu, double sigma,
                            double u_lo, double u_hi, const double* gtab, int64_t G) {
    if (u < u_lo || u > u_hi) return 0.0;
    if (kind == 2) {
        double D = (u_hi - u_lo) / (double)(G - 1);
        double t = (u - u_lo) / D;
        int64_t k = (int64_t)t;
        if (k > G - 2) k = G - 2;
        double f = t - (double)k;
        return gtab[k] + f * (gtab[k + 1] - gtab[k]);
    }
    return erdf_xi(kind, u, lam_star, d1, d2, mu, sigma);
}

void orc_slice_sample(int kind, double lam_star, double d1, double d2, double mu, double sigma, double lam_min,
                      double lam_max, const double* gtab, int64_t G, int64_t N, int64_t chains, int burn_in, int thin,
                      double w, int m, uint64_t seed, uint32_t b, int dtype, double* lam, double* u_out) {
    const double u_lo = std::log10(lam_min), u_hi = std::log10(lam_max);
    const int64_t n_keep = N / chains;
    auto g = [&](double u) { return slice_density(kind, u, lam_star, d1, d2, mu, sigma, u_lo, u_hi, gtab, G); };
    for (int64_t c = 0; c < chains; ++c) {
        uint64_t q = 0;                                   // uniforms used by this chain so far
        auto next_uniform = [&]() {
            uint32_t wd[4];
            orc_philox_stream(seed, ((uint64_t)c << 32) | (q >> 1), b, 5u, wd);
            double U = (q & 1) ? orc_u53(wd[2], wd[3]) : orc_u53(wd[0], wd[1]);
            ++q;
            return U;
        };
        double x = u_lo + next_uniform() * (u_hi - u_lo);
        const int64_t total = (int64_t)burn_in + n_keep * (int64_t)thin;
        for (int64_t t = 1; t <= total; ++t) {
            // the slice
            double y = g(x) * next_uniform();
            // stepping out (Neal 2003, Fig. 3)
            double L = x - w * next_uniform();
            double R = L + w;
            int J = (int)std::floor((double)m * next_uniform());
            int K = (m - 1) - J;
            while (J > 0 && y < g(L)) { L -= w; --J; }
            while (K > 0 && y < g(R)) { R += w; --K; }
            // shrinkage (Neal 2003, Fig. 5)
            for (int it = 0; it < 1000; ++it) {
                double x1 = L + next_uniform() * (R - L);
                if (y < g(x1)) { x = x1; break; }
                if (x1 < x) L = x1; else R = x1;
            }
            if (t > burn_in && (t - burn_in) % thin == 0) {
                int64_t n = ((t - burn_in) / thin - 1) * chains + c;
                double l = std::pow(10.0, x);
                if (dtype == 0) l = (double)(float)l;
                lam[n] = l;
                if (u_out) u_out[n] = x;
            }
        }
    }
}

}  // extern "C"

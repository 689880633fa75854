// kernels.cuh -- the non-FFT, non-sort kernels of the path: PSD (Eq. 3), ERDF table + inverse-CDF draw
// (Eq. 1-2), Timmer & Koenig spectrum fill, real-FFT untangle / amplitude replace (L2), rank scatter +
// change count (L5), convergence bookkeeping (L6), periodogram (Eq. A2/A4).
#pragma once
#include "common.cuh"
#include "fft.cuh"

namespace agn {

struct PsdDev { double A, f_b, a_lo, a_hi; };
struct ErdfDev { int kind; int pad; double lam_star, d1, d2, mu, sigma, u_lo, u_hi; };

// O1: raw Philox words, one call per thread
__global__ void philox_words_kernel(uint64_t seed, uint64_t i0, long long n, uint32_t curve, uint32_t tag,
                                    uint4* __restrict__ out) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = philox_stream(seed, i0 + (uint64_t)i, curve, tag);
}

// Eq. 3 bracket: [ (f/f_b)^a_lo + (f/f_b)^a_hi ]^-1
// (r^a as exp2(a log2 r): one logarithm for both powers; the exponent a log2 r stays below ~100 in magnitude, so the
//  result is within ~1e-14 relative of pow(): PSD values are gated at 1e-13 against the oracle)
__device__ __forceinline__ double psd_shape(double f, double f_b, double a_lo, double a_hi) {
    // a slope of exactly 0 gives the term 1 at every f, f = 0 included (pow(0, 0) = 1; 0 * log2(0) would be NaN)
    const double l = log2(f / f_b);
    const double t_lo = a_lo == 0.0 ? 1.0 : exp2(a_lo * l);
    const double t_hi = a_hi == 0.0 ? 1.0 : exp2(a_hi * l);
    return 1.0 / (t_lo + t_hi);
}

__global__ void psd_bpl_kernel(const double* __restrict__ f, long long n, PsdDev p, double* __restrict__ out) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = p.A * psd_shape(f[i], p.f_b, p.a_lo, p.a_hi);
}

// deterministic block sum (fixed tree)
template <int THREADS> __device__ __forceinline__ double block_sum(double v, double* sh) {
    sh[threadIdx.x] = v;
    __syncthreads();
#pragma unroll
    for (int o = THREADS / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    double r = sh[0];
    __syncthreads();
    return r;
}

// Q4 unit-variance normalisation: acc = 2 sum_{1<=j<M/2} s_j + s_{M/2};  A = M^2 / acc.
// stage 1: partial[b][chunk]
__global__ void psd_norm_partial_kernel(const PsdDev* __restrict__ psd, long long M, double dt, int chunk,
                                        double* __restrict__ partial, int nchunks, int B) {
    __shared__ double sh[256];
    const int b = (int)bidx();
    if (b >= B) return;
    PsdDev p = psd[b];
    long long half = M / 2;
    long long beg = 1 + (long long)blockIdx.x * chunk, end = beg + chunk;
    if (end > half + 1) end = half + 1;
    double acc = 0.0;
    for (long long j = beg + threadIdx.x; j < end; j += 256) {
        double s = psd_shape((double)j / ((double)M * dt), p.f_b, p.a_lo, p.a_hi);
        acc += (j < half) ? 2.0 * s : s;
    }
    double tot = block_sum<256>(acc, sh);
    if (threadIdx.x == 0) partial[(long long)b * nchunks + blockIdx.x] = tot;
}
// stage 2: one block per curve; writes A into psd[b].A when the caller asked for it (A <= 0)
__global__ void psd_norm_final_kernel(PsdDev* __restrict__ psd, const double* __restrict__ partial, int nchunks,
                                      long long M) {
    __shared__ double sh[256];
    const int b = blockIdx.x;
    double acc = 0.0;
    for (int i = threadIdx.x; i < nchunks; i += 256) acc += partial[(long long)b * nchunks + i];
    double tot = block_sum<256>(acc, sh);
    if (threadIdx.x == 0 && !(psd[b].A > 0.0)) psd[b].A = (double)M * (double)M / tot;
}

// O3 spectrum value X_j (fp64) for 1 <= j <= M/2 (X_0 = 0): sqrt(S_j/2)(g_re + i g_im), Nyquist sqrt(S)*g_re.
__device__ __forceinline__ double2 tk_X(const PsdDev& p, long long j, long long M, double dt, uint64_t seed,
                                        uint32_t curve) {
    if (j == 0) return make_double2(0.0, 0.0);
    double S = p.A * psd_shape((double)j / ((double)M * dt), p.f_b, p.a_lo, p.a_hi);
    uint4 w = philox_stream(seed, (uint64_t)j, curve, 0u);
    double u1 = u53(w.x, w.y), u2 = u53(w.z, w.w);
    double r = sqrt(-2.0 * log(u1));
    double sn, cs;
    sincospi(2.0 * u2, &sn, &cs);
    if (2 * j == M) return make_double2(sqrt(S) * r * cs, 0.0);
    double a = sqrt(0.5 * S) * r;
    return make_double2(a * cs, a * sn);
}

// Power-of-two M: fill Z (position order, L = M/2 complex) such that the inverse complex FFT of length L
// (unnormalised, then scale 1/L) yields z[n] = x[2n] + i x[2n+1] with x = irfft_M(X).
// a = (X_k + conj X_{L-k})/2, b = (X_k - conj X_{L-k})/2, O = b conj(w_M^k), Z_k = a + i O.
// One thread per PAIR of bins (k, L - k), 0 <= k <= L/2: both spectrum values are evaluated once (Philox, Box-Muller, Eq. 3)
// and give both Z_k and Z_{L-k} (the second one goes to a scattered position: a plain 8-byte store).
template <typename T>
__global__ void tk_fill_kernel(typename Cx<T>::type* __restrict__ Z, const PsdDev* __restrict__ psd, Digits dg,
                               double dt, uint64_t seed, uint32_t curve0, int B) {
    const long long L = 1ll << dg.logL, M = 2 * L;
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int b = (int)bidx();
    if (2 * k > L || b >= B) return;
    PsdDev ps = psd[b];
    const long long k2 = L - k;                                 // k = 0 pairs with the Nyquist bin L
    const double2 X1 = tk_X(ps, k, M, dt, seed, curve0 + b);
    const double2 X2 = tk_X(ps, k2, M, dt, seed, curve0 + b);
    double sn, cs;
    sincos_2pi_frac((uint64_t)k, dg.logL + 1, &sn, &cs);        // conj(w_M^k) = cos + i sin
    {
        const double2 a = make_double2(0.5 * (X1.x + X2.x), 0.5 * (X1.y - X2.y));
        const double2 bb = make_double2(0.5 * (X1.x - X2.x), 0.5 * (X1.y + X2.y));
        const double2 O = make_double2(bb.x * cs - bb.y * sn, bb.x * sn + bb.y * cs);
        Z[(long long)b * L + k2pos(dg, (uint32_t)k)] = mk<T>((T)(a.x - O.y), (T)(a.y + O.x));
    }
    if (k > 0 && k2 != k) {
        // the same formula with the roles of the two bins exchanged; conj(w_M^{L-k}) = -cos + i sin
        const double2 a = make_double2(0.5 * (X2.x + X1.x), 0.5 * (X2.y - X1.y));
        const double2 bb = make_double2(0.5 * (X2.x - X1.x), 0.5 * (X2.y + X1.y));
        const double c2 = -cs, s2 = sn;
        const double2 O = make_double2(bb.x * c2 - bb.y * s2, bb.x * s2 + bb.y * c2);
        Z[(long long)b * L + k2pos(dg, (uint32_t)k2)] = mk<T>((T)(a.x - O.y), (T)(a.y + O.x));
    }
}

// M = 5 * Mp (oversample 10 or 20): three decimated spectra X_r[q] = Xfull[5q + r], r = 0,1,2, each a
// complex inverse FFT of length Mp; Xfull[j] = conj(X[M-j]) for j > M/2.  Layout [b][r][Mp], position order.
template <typename T>
__global__ void tk_fill5_kernel(typename Cx<T>::type* __restrict__ Z, const PsdDev* __restrict__ psd, Digits dg,
                                double dt, uint64_t seed, uint32_t curve0, int B) {
    const long long Mp = 1ll << dg.logL, M = 5 * Mp;
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long by = bidx();
    if (p >= Mp || by >= 3ll * B) return;
    const int b = (int)(by / 3), r = (int)(by % 3);
    PsdDev ps = psd[b];
    long long q = pos2k(dg, (uint32_t)p);
    long long j = 5 * q + r;
    double2 X;
    if (2 * j <= M) X = tk_X(ps, j, M, dt, seed, curve0 + b);
    else { X = tk_X(ps, M - j, M, dt, seed, curve0 + b); X.y = -X.y; }
    Z[((long long)b * 3 + r) * Mp + p] = mk<T>((T)X.x, (T)X.y);
}

// x[n] = (1/M) [ Re Y0[n'] + 2 Re(w^n Y1[n']) + 2 Re(w^{2n} Y2[n']) ], w = e^{+2 pi i / M}, n' = n mod Mp,
// evaluated for the kept window n = off .. off + N - 1 only.
template <typename T>
__global__ void tk_combine5_kernel(const typename Cx<T>::type* __restrict__ Y, T* __restrict__ xn, long long Mp,
                                   long long N, long long off, int B) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int b = (int)bidx();
    if (i >= N || b >= B) return;
    const long long M = 5 * Mp, n = off + i, np = n & (Mp - 1);
    typename Cx<T>::type y0 = Y[((long long)b * 3 + 0) * Mp + np];
    typename Cx<T>::type y1 = Y[((long long)b * 3 + 1) * Mp + np];
    typename Cx<T>::type y2 = Y[((long long)b * 3 + 2) * Mp + np];
    double s1, c1, s2, c2;
    sincospi(2.0 * (double)n / (double)M, &s1, &c1);
    sincospi(2.0 * (double)((2 * n) % M) / (double)M, &s2, &c2);
    double acc = (double)y0.x + 2.0 * ((double)y1.x * c1 - (double)y1.y * s1) +
                 2.0 * ((double)y2.x * c2 - (double)y2.y * s2);
    xn[(long long)b * N + i] = (T)(acc / (double)M);
}

template <typename T>
__global__ void crop_kernel(const T* __restrict__ src, long long src_stride, long long off, T* __restrict__ dst,
                            long long N, int B) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long b = bidx();
    if (i < N && b < B) dst[b * N + i] = src[b * src_stride + off + i];
}

// ------------------------------------------------------------------------------------------------
// real-FFT untangle.  Z = FFT_L(z), z[n] = x[2n] + i x[2n+1], N = 2L.  For the pair (k, L-k):
//   a = (Z_k + conj Z_{L-k})/2,  o = (Z_k - conj Z_{L-k})/(2i),  b = w_N^k o,
//   X_k = a + b,  X_{L-k} = conj(a - b);  k = 0:  X_0 = Re Z_0 + Im Z_0, X_L = Re Z_0 - Im Z_0.
// ------------------------------------------------------------------------------------------------
template <typename T> struct PairX { typename Cx<T>::type X1, X2, w; };

template <typename T>
__device__ __forceinline__ PairX<T> untangle_pair(typename Cx<T>::type z1, typename Cx<T>::type z2,
                                                  typename Cx<T>::type w) {
    typedef typename Cx<T>::type C;
    const T h = (T)0.5;
    C a = mk<T>(h * (z1.x + z2.x), h * (z1.y - z2.y));
    C d = mk<T>(z1.x - z2.x, z1.y + z2.y);             // Z_k - conj Z_{L-k}
    C o = mk<T>(h * d.y, -h * d.x);                    // d / (2i)
    C b = cmul(w, o);
    PairX<T> r;
    r.X1 = cadd(a, b);
    r.X2 = cconj(csub(a, b));
    r.w = w;
    return r;
}
__device__ __forceinline__ float abs2(float2 v) { return hypotf(v.x, v.y); }
__device__ __forceinline__ double abs2(double2 v) { return hypot(v.x, v.y); }

// MODE 0: out_amp[b][k] = |X_k|, k = 0..L (type T, row stride L+1)
// MODE 1: out_pow[b][k-1] = scale[b] |X_k|^2, k = 1..L (fp64, row stride L)
template <typename T, int MODE>
__global__ void untangle_out_kernel(const typename Cx<T>::type* __restrict__ Z, Digits dg, TwLevel<T> lv,
                                    T* __restrict__ out_amp, double* __restrict__ out_pow,
                                    const double* __restrict__ scale, int B) {
    typedef typename Cx<T>::type C;
    const long long L = 1ll << dg.logL;
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long b = bidx();
    if (p >= L || b >= B) return;
    const uint32_t k = pos2k(dg, (uint32_t)p);
    if (2ll * k > L) return;
    const C* z = Z + b * L;
    if (k == 0) {
        C z0 = z[0];
        T x0 = z0.x + z0.y, xl = z0.x - z0.y;
        if (MODE == 0) { out_amp[b * (L + 1)] = fabs(x0); out_amp[b * (L + 1) + L] = fabs(xl); }
        else { out_pow[b * L + (L - 1)] = scale[b] * (double)xl * (double)xl; }
        return;
    }
    const uint32_t p2 = k2pos(dg, (uint32_t)(L - k));
    PairX<T> r = untangle_pair<T>(z[p], z[p2], tw_lookup<T>(lv, k));
    if (MODE == 0) {
        out_amp[b * (L + 1) + k] = abs2(r.X1);
        out_amp[b * (L + 1) + (L - k)] = abs2(r.X2);
    } else {
        double sc = scale[b];
        out_pow[b * L + (k - 1)] = sc * ((double)r.X1.x * (double)r.X1.x + (double)r.X1.y * (double)r.X1.y);
        out_pow[b * L + (L - k - 1)] = sc * ((double)r.X2.x * (double)r.X2.x + (double)r.X2.y * (double)r.X2.y);
    }
}

// A_norm natural order [B][L+1] -> position order [B][L+kApPad] (entry L stays at L); the padded curve stride keeps
// every row of 2^13 amplitudes 16-byte aligned for the asynchronous copies of the fused middle kernel
constexpr int kApPad = 4;
template <typename T>
__global__ void perm_anorm_kernel(const T* __restrict__ A, T* __restrict__ Ap, Digits dg, int B) {
    const long long L = 1ll << dg.logL;
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long b = bidx();
    if (p > L || b >= B) return;
    Ap[b * (L + kApPad) + p] = (p == L) ? A[b * (L + 1) + L] : A[b * (L + 1) + pos2k(dg, (uint32_t)p)];
}

// L2 amplitude replace (O6 step 2) in position order, in place:
// X'_j = A_j X_j / |X_j| (A_j if |X_j| = 0), then back to Z' for the inverse complex FFT.
template <typename T>
__device__ __forceinline__ typename Cx<T>::type replace_amp(typename Cx<T>::type X, T A) {
    T m = abs2(X);
    if (m > (T)0) { T s = A / m; return mk<T>(X.x * s, X.y * s); }
    return mk<T>(A, (T)0);
}
// fp32: 1/|X| from the hardware reciprocal square root plus one Newton step (<= 1 ulp) whenever |X|^2 is a normal
// number that cannot overflow; the scaled hypot and the IEEE division above only for the rest (they were 45 % of
// the fused middle kernel's time).
template <>
__device__ __forceinline__ float2 replace_amp<float>(float2 X, float A) {
    const float m2 = fmaf(X.x, X.x, X.y * X.y);
    if (m2 > 1e-30f && m2 < 1e30f) {
        float r = rsqrtf(m2);
        r = r * fmaf(-0.5f * m2, r * r, 1.5f);
        const float s = A * r;
        return make_float2(X.x * s, X.y * s);
    }
    const float m = hypotf(X.x, X.y);
    if (m > 0.f) { const float s = A / m; return make_float2(X.x * s, X.y * s); }
    return make_float2(A, 0.f);
}

template <typename T>
__device__ __forceinline__ void replace_pair(typename Cx<T>::type& z1, typename Cx<T>::type& z2,
                                             typename Cx<T>::type w, T A1, T A2) {
    typedef typename Cx<T>::type C;
    PairX<T> r = untangle_pair<T>(z1, z2, w);
    C X1 = replace_amp<T>(r.X1, A1), X2 = replace_amp<T>(r.X2, A2);
    const T h = (T)0.5;
    C a = mk<T>(h * (X1.x + X2.x), h * (X1.y - X2.y));     // (X1 + conj X2)/2
    C bb = mk<T>(h * (X1.x - X2.x), h * (X1.y + X2.y));    // (X1 - conj X2)/2
    C o = cmulc(bb, w);                                    // b conj(w)
    z1 = mk<T>(a.x - o.y, a.y + o.x);                      // a + i o
    z2 = mk<T>(a.x + o.y, -(a.y - o.x));                   // conj(a - i o)
}

template <typename T>
__global__ void replace_kernel(typename Cx<T>::type* __restrict__ Z, const T* __restrict__ Ap, Digits dg,
                               TwLevel<T> lv, int B) {
    typedef typename Cx<T>::type C;
    const long long L = 1ll << dg.logL;
    long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long b = bidx();
    if (p >= L || b >= B) return;
    const uint32_t k = pos2k(dg, (uint32_t)p);
    if (2ll * k > L) return;
    C* z = Z + b * L;
    const T* A = Ap + b * (L + kApPad);
    if (k == 0) {
        C z0 = z[0];
        T x0 = z0.x + z0.y, xl = z0.x - z0.y;
        T a0 = A[0], al = A[L];
        T y0 = (x0 != (T)0) ? (x0 > (T)0 ? a0 : -a0) : a0;
        T yl = (xl != (T)0) ? (xl > (T)0 ? al : -al) : al;
        z[0] = mk<T>((T)0.5 * (y0 + yl), (T)0.5 * (y0 - yl));
        return;
    }
    const uint32_t p2 = k2pos(dg, (uint32_t)(L - k));
    C z1 = z[p], z2 = z[p2];
    replace_pair<T>(z1, z2, tw_lookup<T>(lv, k), A[p], A[p2]);
    z[p] = z1;
    z[p2] = z2;
}

// ------------------------------------------------------------------------------------------------
// L5 rank scatter + change count:  x[idx_new[r]] = sorted[r];  changed[b] += (idx_new[r] != idx_old[r])
// COUNT = false: plain scatter (initial x_sim from perm0, Q15)
// ------------------------------------------------------------------------------------------------
template <typename T, bool COUNT>
__global__ void __launch_bounds__(256) scatter_count_kernel(const uint32_t* __restrict__ idx_new,
                                                            const uint32_t* __restrict__ idx_old,
                                                            const T* __restrict__ sorted, T* __restrict__ x,
                                                            long long N, unsigned long long* __restrict__ changed,
                                                            int B, const uint32_t* __restrict__ gate = nullptr) {
    const long long b = bidx();
    if (b >= B) return;
    if (gate && gate[b] == 0u) return;          // fallback of the write-back sort: only the curves it gave up on
    const long long off = b * N;
    unsigned int local = 0;
    for (long long r = ((long long)blockIdx.x * 256 + threadIdx.x) * 4; r < N; r += (long long)gridDim.x * 1024) {
        // N is a multiple of 4
        uint4 in = *reinterpret_cast<const uint4*>(idx_new + off + r);
        T s0 = sorted[off + r], s1 = sorted[off + r + 1], s2 = sorted[off + r + 2], s3 = sorted[off + r + 3];
        if (COUNT) {
            uint4 io = *reinterpret_cast<const uint4*>(idx_old + off + r);
            local += (in.x != io.x) + (in.y != io.y) + (in.z != io.z) + (in.w != io.w);
        }
        x[off + in.x] = s0; x[off + in.y] = s1; x[off + in.z] = s2; x[off + in.w] = s3;
    }
    if (COUNT) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) local += __shfl_xor_sync(0xffffffffu, local, o);
        __shared__ unsigned int ws[8];
        if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = local;
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned int t = 0;
            for (int i = 0; i < 8; ++i) t += ws[i];
            if (t) atomicAdd(&changed[b], (unsigned long long)t);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// delta_k (Eq. 4; NEXT-1): rms over the samples of log10(x_new / x_old).  Stage 1: one fixed-order
// partial sum of squares per chunk of kDeltaChunk samples; stage 2 (inside post_iter_kernel): fixed-order sum of the
// partials.  Deterministic (no atomics).  fp32: the ratio is formed first, then log1p(q - 1) near 1 (q - 1 is exact
// for 1/2 <= q <= 2), so the per-sample error is an unbiased rounding of the ratio; squares accumulate in fp64.
// ------------------------------------------------------------------------------------------------
constexpr int kDeltaChunk = 16384;
__device__ __forceinline__ double log10_ratio(float a, float b) {
    const float q = a / b;
    const float l = (q >= 0.5f && q <= 2.0f) ? log1pf(q - 1.0f) : logf(q);
    return (double)l * 0.43429448190325182765;
}
__device__ __forceinline__ double log10_ratio(double a, double b) { return log10(a / b); }

template <typename T>
__global__ void __launch_bounds__(256) delta_partial_kernel(const T* __restrict__ x_old, const T* __restrict__ x_new,
                                                            long long N, double* __restrict__ partial, int nchunks, int B) {
    __shared__ double sh[256];
    const long long b = bidx();
    if (b >= B) return;
    const long long beg = (long long)blockIdx.x * kDeltaChunk;
    const long long end = beg + kDeltaChunk < N ? beg + kDeltaChunk : N;
    double acc = 0.0;
    for (long long i = beg + threadIdx.x; i < end; i += 256) {
        const double d = log10_ratio(x_new[b * N + i], x_old[b * N + i]);
        acc += d * d;
    }
    const double tot = block_sum<256>(acc, sh);
    if (threadIdx.x == 0) partial[b * nchunks + blockIdx.x] = tot;
}

// L6 bookkeeping after iteration k (1-based), one CTA per curve: record the change count (and delta_k), latch the
// first k at which the curve stops (changed = 0, or delta_k <= threshold when a threshold is set), count the curves
// that have stopped, count the iterations that took the LSD fallback.
struct PostArgs {
    unsigned long long* changed;    // [B] reset here
    int* first_stop;                // [B] 0 = still running
    long long* hist;                // [B][max_iter] or NULL
    const double* partial;          // [B][nchunks] or NULL (delta not requested)
    double* delta_hist;             // [B][max_iter] or NULL
    double threshold;               // <= 0: off
    long long N;
    int nchunks, k, max_iter;
    unsigned int* n_stopped;        // [1]
    const uint32_t* overflow;       // [B] or NULL: the sort's per-curve fallback flag of this iteration
    int* fallbacks;                 // [B] or NULL
};
__global__ void __launch_bounds__(256) post_iter_kernel(PostArgs a) {
    __shared__ double sh[256];
    const int b = blockIdx.x;
    double delta = 0.0;
    if (a.partial) {
        double acc = 0.0;
        for (int i = threadIdx.x; i < a.nchunks; i += 256) acc += a.partial[(long long)b * a.nchunks + i];
        delta = sqrt(block_sum<256>(acc, sh) / (double)a.N);
    }
    if (threadIdx.x != 0) return;
    const unsigned long long c = a.changed[b];
    if (a.hist) a.hist[(long long)b * a.max_iter + (a.k - 1)] = (long long)c;
    if (a.delta_hist) a.delta_hist[(long long)b * a.max_iter + (a.k - 1)] = delta;
    const bool stop = (c == 0) || (a.partial && a.threshold > 0.0 && delta <= a.threshold);
    if (stop && a.first_stop[b] == 0) {
        a.first_stop[b] = a.k;
        atomicAdd(a.n_stopped, 1u);
    }
    a.changed[b] = 0;
    if (a.fallbacks && a.overflow && a.overflow[b]) a.fallbacks[b] += 1;
}
__global__ void finalize_iters_kernel(const int* __restrict__ first_stop, int* __restrict__ iters_used, int max_iter,
                                      int B) {
    int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    iters_used[b] = first_stop[b] ? first_stop[b] : max_iter;
}

// delta mode: the state of curve b after iteration first_stop[b] is copied out when the curve stops (want = k), and the
// curves that never stopped are copied out at the end (want = 0).  A CTA whose curve does not match exits at once.
template <typename T>
__global__ void __launch_bounds__(256) snapshot_kernel(const int* __restrict__ first_stop, int want, const T* __restrict__ x_src,
                                                       const uint32_t* __restrict__ p_src, T* __restrict__ x_dst,
                                                       uint32_t* __restrict__ p_dst, long long N, int B) {
    const long long b = bidx();
    if (b >= B || first_stop[b] != want) return;
    const long long beg = (long long)blockIdx.x * 4096;
    for (long long i = beg + threadIdx.x; i < beg + 4096 && i < N; i += 256) {
        x_dst[b * N + i] = x_src[b * N + i];
        p_dst[b * N + i] = p_src[b * N + i];
    }
}

// x_adj + 0.0 (Q13: -0 -> +0) copy for the lock-step debug output
template <typename T> __global__ void copy_canon_kernel(const T* __restrict__ src, T* __restrict__ dst, long long n) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src[i] + (T)0;
}

// ------------------------------------------------------------------------------------------------
// ERDF (O4)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double erdf_xi(const ErdfDev& e, double u) {
    if (e.kind == 0) {
        double r = exp10(u) / e.lam_star;         // (exp10: same 1-ulp class as pow(10, u), a third of its cost)
        return 1.0 / (pow(r, e.d1) + pow(r, e.d2));
    }
    double z = (u - e.mu) / e.sigma;
    return exp(-0.5 * z * z);
}

// One CTA per table: C_0 = 0, C_k = C_{k-1} + (p_k + p_{k-1}) D / 2, then C /= C_{G-1}.
// p_k is evaluated once per grid point (parked in the output row), every thread adds up the trapezoids of its own
// contiguous stretch, the stretch totals are scanned by the whole CTA (fixed order), and a last walk writes C.
__device__ __forceinline__ void erdf_table_body(const ErdfDev& e, int G, double* __restrict__ Cc) {
    __shared__ double sh[256];
    const double D = (e.u_hi - e.u_lo) / (double)(G - 1);
    for (int k = threadIdx.x; k < G; k += 256) Cc[k] = erdf_xi(e, e.u_lo + (double)k * D);
    __syncthreads();
    const int per = (G + 255) / 256;
    const int k0 = threadIdx.x * per, k1 = min(G, k0 + per);
    const double p_before = (k0 > 0 && k0 < G) ? Cc[k0 - 1] : 0.0;
    double acc = 0.0, pm = p_before;
    for (int k = k0; k < k1; ++k) {
        const double pk = Cc[k];
        if (k > 0) acc += 0.5 * (pk + pm) * D;
        pm = pk;
    }
    // inclusive scan of the stretch totals (Hillis-Steele in shared memory: the order is fixed)
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = 1; o < 256; o <<= 1) {
        const double v = (threadIdx.x >= o) ? sh[threadIdx.x - o] : 0.0;
        __syncthreads();
        sh[threadIdx.x] += v;
        __syncthreads();
    }
    const double tot = sh[255];
    double run = sh[threadIdx.x] - acc;
    pm = p_before;
    for (int k = k0; k < k1; ++k) {
        const double pk = Cc[k];
        if (k > 0) run += 0.5 * (pk + pm) * D;
        pm = pk;
        Cc[k] = (k == G - 1) ? 1.0 : run / tot;
    }
}
__global__ void __launch_bounds__(256) erdf_table_kernel(const ErdfDev* __restrict__ erdf, int G, double* __restrict__ Ctab) {
    const ErdfDev e = erdf[blockIdx.x];
    erdf_table_body(e, G, Ctab + (long long)blockIdx.x * G);
}
// the same table from parameters passed by value (agnvar_erdf_table: no device scratch)
constexpr int kErdfArgBatch = 32;
struct ErdfBatch { ErdfDev e[kErdfArgBatch]; };
__global__ void __launch_bounds__(256) erdf_table_args_kernel(ErdfBatch eb, int G, double* __restrict__ Ctab) {
    const ErdfDev e = eb.e[blockIdx.x];
    erdf_table_body(e, G, Ctab + (long long)blockIdx.x * G);
}

// One thread per Philox call = two samples (n = 2i uses words (0,1), n = 2i+1 words (2,3)).
template <typename T>
__global__ void erdf_sample_kernel(const ErdfDev* __restrict__ erdf, int per_curve, const double* __restrict__ Ctab,
                                   int G, long long N, uint64_t seed, uint32_t curve0, T* __restrict__ out, int B) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int b = (int)bidx();
    if (2 * i >= N || b >= B) return;
    const int t = per_curve ? b : 0;
    ErdfDev e = erdf[t];
    const double* Cc = Ctab + (long long)t * G;
    const double D = (e.u_hi - e.u_lo) / (double)(G - 1);
    uint4 w = philox_stream(seed, (uint64_t)i, curve0 + b, 1u);
    double U[2] = {u53(w.x, w.y), u53(w.z, w.w)};
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        int lo = 0, hi = G - 1;                    // invariant C[lo] <= U < C[hi]
        while (hi - lo > 1) {
            int mid = (lo + hi) >> 1;
            if (Cc[mid] <= U[q]) lo = mid; else hi = mid;
        }
        double c0 = Cc[lo], c1 = Cc[lo + 1];
        double uu = (e.u_lo + (double)lo * D) + (U[q] - c0) / (c1 - c0) * D;
        out[(long long)b * N + 2 * i + q] = (T)exp10(uu);
    }
}

// ------------------------------------------------------------------------------------------------
// periodogram helpers
// ------------------------------------------------------------------------------------------------
// per-curve scale: norm 0 -> 2/N^2 ; norm 1 -> 2 dt / (mu^2 N), mu = sample mean (fixed-order sums)
template <typename T>
__global__ void pgram_scale_kernel(const T* __restrict__ x, long long N, double dt, int norm, double* __restrict__ scale) {
    __shared__ double sh[256];
    const long long b = blockIdx.x;
    if (norm == 0) {
        if (threadIdx.x == 0) scale[b] = 2.0 / ((double)N * (double)N);
        return;
    }
    double acc = 0.0;
    for (long long i = threadIdx.x; i < N; i += 256) acc += (double)x[b * N + i];
    double tot = block_sum<256>(acc, sh);
    if (threadIdx.x == 0) {
        double mu = tot / (double)N;
        scale[b] = 2.0 * dt / (mu * mu * (double)N);
    }
}

// mean of P_j over j in [e0, e1) ; one block per (bin, curve)
__global__ void pgram_bin_kernel(const double* __restrict__ P, long long half, const long long* __restrict__ edges,
                                 int nbins, double* __restrict__ out, long long* __restrict__ counts, int B) {
    __shared__ double sh[256];
    const int e = blockIdx.x;
    const long long b = bidx();
    if (b >= B) return;
    long long j0 = edges[e], j1 = edges[e + 1];
    if (e == nbins - 1 && j1 < half + 1) j1 = half + 1;
    if (j1 > half + 1) j1 = half + 1;
    double acc = 0.0;
    for (long long j = j0 + threadIdx.x; j < j1; j += 256) acc += P[b * half + (j - 1)];
    double tot = block_sum<256>(acc, sh);
    if (threadIdx.x == 0) {
        out[b * nbins + e] = (j1 > j0) ? tot / (double)(j1 - j0) : 0.0;
        if (counts && b == 0) counts[e] = j1 - j0;
    }
}

}  // namespace agn

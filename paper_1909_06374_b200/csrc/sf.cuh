// sf.cuh -- NEXT-2: the observables the paper builds on the generated light curves (evenly sampled, lag l = tau / dt):
//   structure function (Eq. A6)   SF(tau)^2 = mean over the N - l pairs (i, i + l) of [v_i - v_{i+l}]^2,
//       v = x (L/L_Edd units) or v = -2.5 log10 x (magnitudes: the zero point cancels);
//   representative SF (Eq. 6)      mean over the realisations of SF_i^2 and its standard error;
//   P(|dm| > dm_ref | tau)         fraction of the pairs at lag l with |m_i - m_{i+l}| > dm_ref,
//       optionally with a magnitude cut (points fainter than m_cut become upper limits at m_cut; only pairs with at
//       least one detected point count).
// Pair reductions are bandwidth-bound: every sample is read once per lag (twice when the lag exceeds the chunk); the
// magnitudes are computed ONCE per call into the workspace (fp64), not once per lag.  All differences and sums are fp64
// (fp32 inputs are exact in fp64); sums are fixed-order (per-chunk partials, then a fixed tree): deterministic.
#pragma once
#include "common.cuh"
#include "kernels.cuh"

namespace agn {

constexpr int kSfChunk = 8192;          // pairs per CTA and lag
constexpr int kSfMaxRef = 16;

// v[i] = m_zero - 2.5 log10(x[i]) (fp64), optionally clipped at m_cut with a detection flag (1 = detected, m <= m_cut)
template <typename T>
__global__ void __launch_bounds__(256) sf_mag_kernel(const T* __restrict__ x, long long n, double m_zero, int use_cut,
                                                     double m_cut, double* __restrict__ v, unsigned char* __restrict__ det) {
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    double m = m_zero - 2.5 * log10((double)x[i]);
    if (det) det[i] = (!use_cut || m <= m_cut) ? 1 : 0;
    if (use_cut && m > m_cut) m = m_cut;
    v[i] = m;
}

// partial[b][q][chunk] = sum over the chunk's pairs of (v_i - v_{i+l})^2.  V = T (raw series) or double (magnitudes).
// A CTA owns one chunk of first members i and kSfLagGroup consecutive lags: a thread converts its 32 first members to
// fp64 ONCE and keeps them in registers, so a pair costs one load and one float -> double conversion instead of two
// (ncu, round 3: with two conversions per pair the kernel sat at 78 % of the conversion (XU) pipe, fp64 pipe 22 %,
// DRAM one pass over x -- a curve's lags run close together and find it in L2).  Order of the additions per (b, q,
// chunk) is fixed: per thread by ascending i, then the block tree.
constexpr int kSfLagGroup = 8;
constexpr int kSfSub = 8;                 // first members held in registers at a time
template <typename V>
__global__ void __launch_bounds__(256, 4) sf_partial_kernel(const V* __restrict__ v, long long N, const long long* __restrict__ lags,
                                                            int nlags, double* __restrict__ partial, int nchunks, int B) {
    __shared__ double sh[256];
    constexpr int PER = kSfChunk / 256;
    const long long b = blockIdx.z;
    const int q0 = blockIdx.y * kSfLagGroup;
    const long long beg = (long long)blockIdx.x * kSfChunk + threadIdx.x;
    const V* vb = v + b * N;
    long long lag[kSfLagGroup];
    double acc[kSfLagGroup];
#pragma unroll
    for (int g = 0; g < kSfLagGroup; ++g) {
        lag[g] = q0 + g < nlags ? lags[q0 + g] : N;          // a lag of N has no pair
        acc[g] = 0.0;
    }
    for (int k0 = 0; k0 < PER; k0 += kSfSub) {
        double own[kSfSub];
#pragma unroll
        for (int k = 0; k < kSfSub; ++k) {
            const long long i = beg + 256ll * (k0 + k);
            own[k] = i < N ? (double)vb[i] : 0.0;
        }
#pragma unroll
        for (int g = 0; g < kSfLagGroup; ++g) {
            const long long P = N - lag[g];                  // number of pairs (<= 0: none)
#pragma unroll
            for (int k = 0; k < kSfSub; ++k) {
                const long long i = beg + 256ll * (k0 + k);
                if (i < P) {
                    const double d = own[k] - (double)vb[i + lag[g]];
                    acc[g] += d * d;
                }
            }
        }
    }
#pragma unroll
    for (int g = 0; g < kSfLagGroup; ++g) {
        const double tot = block_sum<256>(acc[g], sh);
        if (threadIdx.x == 0 && q0 + g < nlags) partial[(b * nlags + q0 + g) * nchunks + blockIdx.x] = tot;
    }
}
inline unsigned sf_lag_groups(int nlags) { return (unsigned)((nlags + kSfLagGroup - 1) / kSfLagGroup); }

// sf2[b][q] = (sum of the partials) / (N - l); pairs[q] = N - l
__global__ void __launch_bounds__(256) sf_final_kernel(const double* __restrict__ partial, int nchunks, long long N,
                                                       const long long* __restrict__ lags, int nlags, double* __restrict__ sf2,
                                                       long long* __restrict__ pairs) {
    __shared__ double sh[256];
    const long long b = blockIdx.y;
    const int q = blockIdx.x;
    const long long P = N - lags[q];
    double acc = 0.0;
    for (int i = threadIdx.x; i < nchunks; i += 256) acc += partial[(b * nlags + q) * nchunks + i];
    const double tot = block_sum<256>(acc, sh);
    if (threadIdx.x == 0) {
        sf2[b * nlags + q] = P > 0 ? tot / (double)P : 0.0;
        if (pairs && b == 0) pairs[q] = P > 0 ? P : 0;
    }
}

// Eq. 6: mean over the B realisations and the standard error of that mean (sample standard deviation / sqrt(B))
__global__ void __launch_bounds__(256) sf_rep_kernel(const double* __restrict__ sf2, int B, int nlags, double* __restrict__ mean,
                                                     double* __restrict__ se) {
    __shared__ double sh[256];
    const int q = blockIdx.x;
    double acc = 0.0;
    for (int b = threadIdx.x; b < B; b += 256) acc += sf2[(long long)b * nlags + q];
    const double m = block_sum<256>(acc, sh) / (double)B;
    double var = 0.0;
    for (int b = threadIdx.x; b < B; b += 256) { const double d = sf2[(long long)b * nlags + q] - m; var += d * d; }
    const double tv = block_sum<256>(var, sh);
    if (threadIdx.x == 0) {
        if (mean) mean[q] = m;
        if (se) se[q] = B > 1 ? sqrt(tv / (double)(B - 1) / (double)B) : 0.0;
    }
}

// counts[b][q][r] += #{pairs of the chunk considered with |m_i - m_{i+l}| > ref_r}; considered[b][q] += #{pairs considered}
struct DmRefs { double ref[kSfMaxRef]; };
__global__ void __launch_bounds__(256) dm_count_kernel(const double* __restrict__ m, const unsigned char* __restrict__ det,
                                                       long long N, const long long* __restrict__ lags, int nlags, DmRefs refs,
                                                       int nref, unsigned long long* __restrict__ counts,
                                                       unsigned long long* __restrict__ considered, int B) {
    const long long b = blockIdx.z;
    const int q = blockIdx.y;
    const long long l = lags[q];
    const long long P = N - l;
    const long long beg = (long long)blockIdx.x * kSfChunk;
    const long long end = beg + kSfChunk < P ? beg + kSfChunk : P;
    const double* mb = m + b * N;
    const unsigned char* db = det + b * N;
    unsigned int c[kSfMaxRef];
#pragma unroll
    for (int r = 0; r < kSfMaxRef; ++r) c[r] = 0u;
    unsigned int np = 0u;
    for (long long i = beg + threadIdx.x; i < end; i += 256) {
        if (!(db[i] | db[i + l])) continue;
        ++np;
        const double d = fabs(mb[i] - mb[i + l]);
#pragma unroll
        for (int r = 0; r < kSfMaxRef; ++r) c[r] += (r < nref && d > refs.ref[r]) ? 1u : 0u;
    }
    // warp totals, then one integer atomic per warp and counter (integer sums are order-independent: deterministic)
#pragma unroll
    for (int r = 0; r < kSfMaxRef; ++r) {
        if (r < nref) {
            unsigned int t = c[r];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
            if ((threadIdx.x & 31) == 0 && t) atomicAdd(&counts[(b * nlags + q) * nref + r], (unsigned long long)t);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) np += __shfl_xor_sync(0xffffffffu, np, o);
    if ((threadIdx.x & 31) == 0 && np) atomicAdd(&considered[b * nlags + q], (unsigned long long)np);
}

__global__ void dm_final_kernel(const unsigned long long* __restrict__ counts, const unsigned long long* __restrict__ considered,
                                long long n_bq, int nref, double* __restrict__ prob, long long* __restrict__ considered_out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_bq * nref) return;
    const long long bq = i / nref;
    const unsigned long long P = considered[bq];
    prob[i] = P ? (double)counts[i] / (double)P : 0.0;
    if (considered_out && i % nref == 0) considered_out[bq] = (long long)P;
}

// ------------------------------------------------------------------------------------------------
// NEXT-4: ensemble SF of masked sub-segments (Fig. 7-8; Q23) and moments (Fig. 2)
// ------------------------------------------------------------------------------------------------
// one thread per (curve, point j of the sub-sample): offset from Philox tag 3, keep flag from tag 4, value (or magnitude)
template <typename T>
__global__ void __launch_bounds__(256) ens_prepare_kernel(const T* __restrict__ x, long long N, long long n_sub, double keep,
                                                          uint64_t seed, uint32_t curve0, int mag, double* __restrict__ v,
                                                          unsigned char* __restrict__ kept, long long* __restrict__ offsets, int B) {
    const long long b = bidx();
    const long long j = (long long)blockIdx.x * 256 + threadIdx.x;
    if (b >= B || j >= n_sub) return;
    const uint4 w3 = philox_stream(seed, 0ull, curve0 + (uint32_t)b, 3u);
    const long long off = (long long)floor(u53(w3.x, w3.y) * (double)(N - n_sub + 1));
    if (j == 0 && offsets) offsets[b] = off;
    const uint4 w4 = philox_stream(seed, (uint64_t)(j >> 1), curve0 + (uint32_t)b, 4u);
    const double u = (j & 1) ? u53(w4.z, w4.w) : u53(w4.x, w4.y);
    kept[b * n_sub + j] = (u < keep) ? 1 : 0;
    const double xv = (double)x[b * N + off + j];
    v[b * n_sub + j] = mag ? -2.5 * log10(xv) : xv;
}

// partial[b][q][chunk] = sum over the chunk's kept pairs of (v_j - v_{j+l})^2; count[q] += number of kept pairs
__global__ void __launch_bounds__(256) ens_partial_kernel(const double* __restrict__ v, const unsigned char* __restrict__ kept,
                                                          long long n_sub, const long long* __restrict__ lags, int nlags,
                                                          double* __restrict__ partial, unsigned long long* __restrict__ count,
                                                          int nchunks, int B) {
    __shared__ double sh[256];
    const long long b = blockIdx.z;
    const int q = blockIdx.y;
    const long long l = lags[q];
    const long long P = n_sub - l;
    const long long beg = (long long)blockIdx.x * kSfChunk;
    const long long end = beg + kSfChunk < P ? beg + kSfChunk : P;
    const double* vb = v + b * n_sub;
    const unsigned char* kb = kept + b * n_sub;
    double acc = 0.0;
    unsigned int np = 0;
    for (long long i = beg + threadIdx.x; i < end; i += 256) {
        if (kb[i] & kb[i + l]) {
            const double d = vb[i] - vb[i + l];
            acc += d * d;
            ++np;
        }
    }
    const double tot = block_sum<256>(acc, sh);
    if (threadIdx.x == 0) partial[(b * nlags + q) * nchunks + blockIdx.x] = tot;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) np += __shfl_xor_sync(0xffffffffu, np, o);
    if ((threadIdx.x & 31) == 0 && np) atomicAdd(&count[q], (unsigned long long)np);
}

// pooled over the curves, fixed order: sf2[q] = (sum_b sum_chunk partial) / count[q]
__global__ void __launch_bounds__(256) ens_final_kernel(const double* __restrict__ partial, const unsigned long long* __restrict__ count,
                                                        int nchunks, int nlags, int B, double* __restrict__ sf2,
                                                        long long* __restrict__ pairs) {
    __shared__ double sh[256];
    const int q = blockIdx.x;
    double acc = 0.0;
    const long long per = nchunks;
    for (long long i = threadIdx.x; i < (long long)B * per; i += 256) {
        const long long b = i / per, c = i - b * per;
        acc += partial[(b * nlags + q) * nchunks + c];
    }
    const double tot = block_sum<256>(acc, sh);
    if (threadIdx.x == 0) {
        const unsigned long long n = count[q];
        sf2[q] = n ? tot / (double)n : 0.0;
        if (pairs) pairs[q] = (long long)n;
    }
}

// per curve: mean, variance (1/N), skewness, excess kurtosis (two passes, fixed-order fp64 sums)
template <typename T>
__global__ void __launch_bounds__(256) moments_kernel(const T* __restrict__ x, long long N, double* __restrict__ out) {
    __shared__ double sh[256];
    const long long b = blockIdx.x;
    const T* xb = x + b * N;
    double s1 = 0.0;
    for (long long i = threadIdx.x; i < N; i += 256) s1 += (double)xb[i];
    const double mu = block_sum<256>(s1, sh) / (double)N;
    double a2 = 0.0, a3 = 0.0, a4 = 0.0;
    for (long long i = threadIdx.x; i < N; i += 256) {
        const double d = (double)xb[i] - mu, d2 = d * d;
        a2 += d2; a3 += d2 * d; a4 += d2 * d2;
    }
    const double m2 = block_sum<256>(a2, sh) / (double)N;
    const double m3 = block_sum<256>(a3, sh) / (double)N;
    const double m4 = block_sum<256>(a4, sh) / (double)N;
    if (threadIdx.x == 0) {
        out[b * 4 + 0] = mu;
        out[b * 4 + 1] = m2;
        out[b * 4 + 2] = m2 > 0.0 ? m3 / (m2 * sqrt(m2)) : 0.0;
        out[b * 4 + 3] = m2 > 0.0 ? m4 / (m2 * m2) - 3.0 : 0.0;
    }
}

}  // namespace agn

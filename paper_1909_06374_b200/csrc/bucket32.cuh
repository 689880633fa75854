// bucket32.cuh -- L4 for long fp32 curves as a TWO-LEVEL sort (SURVEY 8(d) "2-level" model: every key crosses HBM
// twice instead of four LSD round trips):
//
//   cdf_sample_kernel    one key in 64 -> a 65536-bin histogram of the key's top 16 bits (per curve)
//   cdf_table_kernel     exclusive scan -> table (cum, cnt) per bin: a piecewise-linear estimate of the CDF of the
//                        keys.  bucket(key) = (cum*2^16 + low16(key)*cnt) >> 22 is a MONOTONE map of the key onto
//                        N/4096 equal-depth buckets (64 samples = 4096 keys per bucket on average).
//   bucket_part_kernel   one pass over x_adj: (key, time index) pairs appended to their bucket's slab
//                        (kBkCap = 8192 slots, cursor per bucket).  4 B in + 8 B out per sample.
//   bucket_base_kernel   exclusive scan of the bucket populations -> first rank of every bucket
//   bucket_sort_kernel   one CTA per bucket: the slab is sorted in shared memory by (key, index) -- an
//                        interpolation counting sort into 8192 slots followed by an exact rank among the few
//                        slot mates -- and the indices are written at their ranks.  8 B in + 4 B out per sample.
//
// Order inside a slab is arbitrary (atomic cursors), so the final order is defined by the comparison of the 64-bit
// (key, index) words alone: equal keys come out by ascending time index, which is the stable order the definition
// asks for (O6 step 4), independently of the run.
// A bucket that would overflow its slab (inputs with massive ties, or a distribution the sampled CDF misses) raises
// the curve's `overflow` flag; the LSD passes of sort32.cuh then sort that curve instead (they are always enqueued
// and exit at once when the flag is clear: the decision is taken on the device, no host synchronisation).
#pragma once
#include "common.cuh"
#include "sort.cuh"

namespace agn {

constexpr int kBkMeanLog = 12;                    // mean bucket population 2^12
constexpr int kBkCap = 8192;                      // slab slots per bucket
constexpr int kBkSampleLog = 6;                   // one sample per 64 keys
constexpr int kBkBinLog = 16;                     // CDF bins = top 16 key bits
constexpr int kBkBins = 1 << kBkBinLog;
constexpr int kBkShift = kBkBinLog + kBkMeanLog - kBkSampleLog;     // 22
constexpr int kBkSortThreads = 512;
constexpr int kBkSlots = 8192;                    // interpolation slots of the in-CTA sort
constexpr int kBkEpt = kBkCap / kBkSortThreads;   // 16 elements per thread

// keys above the largest sampled bin have cum = all samples: clamp them into the last bucket (still monotone)
__device__ __forceinline__ uint32_t bucket_of(uint32_t key, const uint2* __restrict__ tab, uint32_t nb) {
    const uint2 e = __ldg(tab + (key >> (32 - kBkBinLog)));
    const unsigned long long pos = ((unsigned long long)e.x << kBkBinLog) + (unsigned long long)(key & (kBkBins - 1)) * e.y;
    return min((uint32_t)(pos >> kBkShift), nb - 1u);
}

__global__ void __launch_bounds__(256) cdf_sample_kernel(const float* __restrict__ vals, uint32_t* __restrict__ hist,
                                                         uint32_t N, long long B) {
    const long long b = bidx();
    if (b >= B) return;
    const uint32_t i = blockIdx.x * 256 + threadIdx.x;          // sample number
    if (i >= (N >> kBkSampleLog)) return;
    // the sample of block i of 64 keys sits at a position that varies with i (no fixed phase)
    const uint32_t e = (i << kBkSampleLog) + ((i * 0x9E3779B1u) >> (32 - kBkSampleLog));
    const uint32_t k = key_of(vals[(size_t)b * N + e]);
    atomicAdd(&hist[(size_t)b * kBkBins + (k >> (32 - kBkBinLog))], 1u);
}

// one CTA (1024 threads) per curve: tab[bin] = (exclusive cum, cnt)
__global__ void __launch_bounds__(1024) cdf_table_kernel(const uint32_t* __restrict__ hist, uint2* __restrict__ tab) {
    __shared__ uint32_t ws[32];
    const uint32_t* h = hist + (size_t)blockIdx.x * kBkBins;
    uint2* t = tab + (size_t)blockIdx.x * kBkBins;
    constexpr int PER = kBkBins / 1024;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t c[PER], sum = 0;
#pragma unroll
    for (int i = 0; i < PER; ++i) { c[i] = h[threadIdx.x * PER + i]; sum += c[i]; }
    uint32_t inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t n = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += n;
    }
    if (lane == 31) ws[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        uint32_t v = ws[lane], w = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t n = __shfl_up_sync(0xffffffffu, w, o);
            if (lane >= o) w += n;
        }
        ws[lane] = w - v;
    }
    __syncthreads();
    uint32_t run = inc - sum + ws[warp];
#pragma unroll
    for (int i = 0; i < PER; ++i) { t[threadIdx.x * PER + i] = make_uint2(run, c[i]); run += c[i]; }
}

constexpr int kBkPartThreads = 256;
constexpr int kBkPartEpt = 16;

__global__ void __launch_bounds__(kBkPartThreads) bucket_part_kernel(const float* __restrict__ vals,
                                                                     const uint2* __restrict__ tab,
                                                                     uint32_t* __restrict__ cursor,
                                                                     uint2* __restrict__ slabs, uint32_t* __restrict__ overflow,
                                                                     uint32_t N, uint32_t nb, long long B) {
    const long long b = bidx();
    if (b >= B) return;
    const float* v = vals + (size_t)b * N;
    const uint2* t = tab + (size_t)b * kBkBins;
    uint32_t* cur = cursor + (size_t)b * nb;
    uint2* sl = slabs + (size_t)b * nb * kBkCap;
    const uint32_t e0 = blockIdx.x * (kBkPartThreads * kBkPartEpt) + threadIdx.x;
    uint32_t key[kBkPartEpt], bk[kBkPartEpt];
#pragma unroll
    for (int j = 0; j < kBkPartEpt; ++j) key[j] = key_of(__ldcs(v + e0 + j * kBkPartThreads));
#pragma unroll
    for (int j = 0; j < kBkPartEpt; ++j) bk[j] = bucket_of(key[j], t, nb);
    bool over = false;
#pragma unroll
    for (int j = 0; j < kBkPartEpt; ++j) {
        const uint32_t s = atomicAdd(&cur[bk[j]], 1u);
        if (s < (uint32_t)kBkCap) sl[(size_t)bk[j] * kBkCap + s] = make_uint2(key[j], e0 + j * kBkPartThreads);
        else over = true;
    }
    if (over) overflow[b] = 1u;
}

// one CTA (1024 threads) per curve: base[k] = sum of the populations of buckets < k (populations clamped to the slab)
__global__ void __launch_bounds__(1024) bucket_base_kernel(const uint32_t* __restrict__ cursor, uint32_t* __restrict__ base,
                                                           uint32_t nb) {
    __shared__ uint32_t ws[32];
    __shared__ uint32_t carry;
    const uint32_t* c = cursor + (size_t)blockIdx.x * nb;
    uint32_t* o = base + (size_t)blockIdx.x * nb;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry = 0u;
    __syncthreads();
    for (uint32_t k0 = 0; k0 < nb; k0 += 1024) {
        const uint32_t k = k0 + threadIdx.x;
        const uint32_t n = (k < nb) ? min(c[k], (uint32_t)kBkCap) : 0u;
        uint32_t inc = n;
#pragma unroll
        for (int s = 1; s < 32; s <<= 1) {
            const uint32_t m = __shfl_up_sync(0xffffffffu, inc, s);
            if (lane >= s) inc += m;
        }
        if (lane == 31) ws[warp] = inc;
        __syncthreads();
        uint32_t add = carry;
        for (int w = 0; w < warp; ++w) add += ws[w];
        if (k < nb) o[k] = inc - n + add;
        __syncthreads();
        if (threadIdx.x == 1023) carry = inc + add;
        __syncthreads();
    }
}

struct BkSmem {
    unsigned long long pair[kBkCap];      // (key << 32) | index
    uint32_t cnt[kBkSlots];               // slot populations, then slot starts
    uint32_t wsum[kBkSortThreads / 32];
    uint32_t kmin, kmax;
};

__global__ void __launch_bounds__(kBkSortThreads, 2) bucket_sort_kernel(const uint2* __restrict__ slabs,
                                                                        const uint32_t* __restrict__ cursor,
                                                                        const uint32_t* __restrict__ base,
                                                                        const uint32_t* __restrict__ overflow,
                                                                        uint32_t* __restrict__ idx_out,
                                                                        float* __restrict__ sorted_out, uint32_t N,
                                                                        uint32_t nb, long long B) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    BkSmem& sm = *reinterpret_cast<BkSmem*>(smem_raw);
    const long long b = bidx();
    if (b >= B) return;
    if (overflow[b]) return;                       // this curve is sorted by the LSD passes instead
    const uint32_t bk = blockIdx.x;
    const uint32_t n = cursor[(size_t)b * nb + bk];          // <= kBkCap (no overflow)
    if (n == 0) return;
    const uint32_t r0 = base[(size_t)b * nb + bk];
    const uint2* sl = slabs + ((size_t)b * nb + bk) * kBkCap;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    if (t == 0) { sm.kmin = 0xffffffffu; sm.kmax = 0u; }
#pragma unroll
    for (int i = 0; i < kBkSlots / kBkSortThreads; ++i) sm.cnt[i * kBkSortThreads + t] = 0u;
    uint2 kv[kBkEpt];
    uint32_t lo = 0xffffffffu, hi = 0u;
#pragma unroll
    for (int j = 0; j < kBkEpt; ++j) {
        const uint32_t e = j * kBkSortThreads + t;
        if (e < n) {
            kv[j] = __ldcs(sl + e);
            lo = min(lo, kv[j].x); hi = max(hi, kv[j].x);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    __syncthreads();
    if (lane == 0) { atomicMin(&sm.kmin, lo); atomicMax(&sm.kmax, hi); }
    __syncthreads();
    const uint32_t kmin = sm.kmin;
    // monotone map of (key - kmin) onto the slots: int -> float conversion, multiplication by a positive constant and
    // truncation are all monotone, so equal keys share a slot and a larger key never lands in an earlier slot
    const float scale = (float)kBkSlots / ((float)(sm.kmax - kmin) + 1.0f) * 0.999f;
    uint32_t sc[kBkEpt];            // slot << 16 | arrival number inside the slot
#pragma unroll
    for (int j = 0; j < kBkEpt; ++j) {
        const uint32_t e = j * kBkSortThreads + t;
        if (e < n) {
            const uint32_t s = min((uint32_t)(__uint2float_rz(kv[j].x - kmin) * scale), (uint32_t)(kBkSlots - 1));
            const uint32_t c = atomicAdd(&sm.cnt[s], 1u);
            sc[j] = (s << 16) | c;            // c < 8192 < 2^16
        }
    }
    __syncthreads();
    // exclusive scan of the slot populations (16 consecutive slots per thread)
    {
        constexpr int PER = kBkSlots / kBkSortThreads;
        uint32_t c[PER], sum = 0;
#pragma unroll
        for (int i = 0; i < PER; ++i) { c[i] = sm.cnt[t * PER + i]; sum += c[i]; }
        uint32_t inc = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t m = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += m;
        }
        if (lane == 31) sm.wsum[warp] = inc;
        __syncthreads();
        uint32_t add = 0;
#pragma unroll
        for (int w = 0; w < kBkSortThreads / 32; ++w) add += (w < warp) ? sm.wsum[w] : 0u;
        uint32_t run = inc - sum + add;
#pragma unroll
        for (int i = 0; i < PER; ++i) { sm.cnt[t * PER + i] = run; run += c[i]; }
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kBkEpt; ++j) {
        const uint32_t e = j * kBkSortThreads + t;
        if (e < n) sm.pair[sm.cnt[sc[j] >> 16] + (sc[j] & 0xffffu)] = ((unsigned long long)kv[j].x << 32) | kv[j].y;
    }
    __syncthreads();
    // exact rank among the slot mates (they are contiguous); (key, index) words are all distinct
    for (uint32_t p = t; p < n; p += kBkSortThreads) {
        const unsigned long long me = sm.pair[p];
        const uint32_t key = (uint32_t)(me >> 32);
        const uint32_t s = min((uint32_t)(__uint2float_rz(key - kmin) * scale), (uint32_t)(kBkSlots - 1));
        const uint32_t a = sm.cnt[s];
        const uint32_t z = (s + 1 < (uint32_t)kBkSlots) ? sm.cnt[s + 1] : n;
        uint32_t r = a;
        for (uint32_t q = a; q < z; ++q) r += (sm.pair[q] < me);
        const size_t g = (size_t)b * N + r0 + r;
        idx_out[g] = (uint32_t)me;
        if (sorted_out) sorted_out[g] = val_of(key);
    }
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
inline bool bucket32_applicable(size_t elem_size, long long N) {
    return elem_size == 4 && N >= (1ll << 18) && N <= (1ll << 27);
}

inline cudaError_t bucket32_set_attrs() {
    cudaFuncSetAttribute(bucket_sort_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    return cudaFuncSetAttribute(bucket_sort_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(BkSmem));
}

// control words: hist [B][65536] u32 | cursor [B][nb] | overflow [B] (zeroed per call) | tab [B][65536] uint2 | base [B][nb]
inline size_t bucket32_ctl_bytes(long long B, long long N) {
    const size_t nb = (size_t)(N >> kBkMeanLog);
    return align_up((size_t)B * kBkBins * 4 + (size_t)B * nb * 4 + (size_t)B * 4, 256) +
           align_up((size_t)B * kBkBins * 8, 256) + align_up((size_t)B * nb * 4, 256);
}

// vals [B][N] -> idx_out (and optionally the sorted values) for the curves whose buckets all fit; *overflow_out points
// at the per-curve flags (1 = not sorted here).  slabs: B*N*2 (key, index) pairs of scratch.
inline cudaError_t bucket32_sort(const float* vals, uint32_t* idx_out, float* sorted_out, long long B, long long N,
                                 uint2* slabs, void* ctl, const uint32_t** overflow_out, cudaStream_t st) {
    const uint32_t nb = (uint32_t)(N >> kBkMeanLog);
    unsigned char* w = (unsigned char*)ctl;
    uint32_t* hist = (uint32_t*)w;
    uint32_t* cursor = hist + (size_t)B * kBkBins;
    uint32_t* overflow = cursor + (size_t)B * nb;
    const size_t zero_bytes = (size_t)B * kBkBins * 4 + (size_t)B * nb * 4 + (size_t)B * 4;
    w += align_up(zero_bytes, 256);
    uint2* tab = (uint2*)w; w += align_up((size_t)B * kBkBins * 8, 256);
    uint32_t* base = (uint32_t*)w;
    cudaError_t e = cudaMemsetAsync(hist, 0, zero_bytes, st);
    if (e != cudaSuccess) return e;
    const uint32_t nsamp = (uint32_t)(N >> kBkSampleLog);
    AGN_LAUNCH(K_SORT_CDF, st, (cdf_sample_kernel<<<bgrid((nsamp + 255) / 256, B), 256, 0, st>>>(vals, hist, (uint32_t)N, B)));
    AGN_LAUNCH(K_SORT_CDF, st, (cdf_table_kernel<<<(unsigned)B, 1024, 0, st>>>(hist, tab)));
    AGN_LAUNCH(K_SORT_PART, st, (bucket_part_kernel<<<bgrid((unsigned)(N / (kBkPartThreads * kBkPartEpt)), B), kBkPartThreads, 0, st>>>(
        vals, tab, cursor, slabs, overflow, (uint32_t)N, nb, B)));
    AGN_LAUNCH(K_SORT_CDF, st, (bucket_base_kernel<<<(unsigned)B, 1024, 0, st>>>(cursor, base, nb)));
    AGN_LAUNCH(K_SORT_BUCKET, st, (bucket_sort_kernel<<<bgrid(nb, B), kBkSortThreads, sizeof(BkSmem), st>>>(
        slabs, cursor, base, overflow, idx_out, sorted_out, (uint32_t)N, nb, B)));
    *overflow_out = overflow;
    return cudaGetLastError();
}

}  // namespace agn

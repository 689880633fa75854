// bucket32.cuh -- L4 for long fp32 curves (N >= 2^18) as a distribution sort: every key is routed by an estimate of
// the CDF of the keys to one of N/2048 equal-depth buckets, and each bucket is finished in shared memory.
//
//   cdf_sample_kernel    one key in 64 -> a 65536-bin histogram of the key's top 16 bits (per curve)
//   cdf_table_kernel     exclusive scan of the add-one smoothed bin weights -> table (cumw << 7, w): a piecewise-
//                        linear, strictly monotone estimate of the CDF.  bs_of(key) = bucket << 11 | slot costs one
//                        table look-up, one 32x32 multiply and one multiply-high.
//   bucket_part_kernel   <0> x_adj -> (key, time index) pairs in N^(1/2)-ish coarse slabs (high bits of the bucket),
//                        <1> coarse slab -> fine slabs (kBkCap = 4096 slots per bucket, mean population 2048),
//                        <2> the bin step of the two-level rank scatter L5 (same tile logic, digit = window of dst).
//                        A tile counts its keys per digit in shared memory, reserves one range per (tile, digit) with
//                        one global atomic, orders the tile by digit in shared memory and writes coalesced runs.
//   bucket_base_kernel   exclusive scan of the bucket populations -> first rank of every bucket
//   bucket_bounds_kernel smallest key of every bucket (inverse of bs_of at the bucket boundaries)
//   bucket_sort_kernel   one CTA per bucket: counting sort into 2048 interpolation slots (a linear map of the key
//                        onto the bucket's key interval), then the exact rank of every pair among its few slot
//                        mates; indices written at their ranks.
//
// HBM bytes per sample: 0.5 (sample) + 12 (<0>: 4 in, 8 out) + 16 (<1>) + 12 (finish: 8 in, 4 out).
// Order inside a slab is arbitrary (atomic cursors), so the final order is defined by the comparison of the 64-bit
// (key, index) words alone: equal keys come out by ascending time index, which is the stable order the definition
// asks for (O6 step 4), independently of the run.
// A slab that would overflow (inputs with massive ties, or a distribution the sampled CDF misses) raises the curve's
// `overflow` flag; the LSD passes of sort32.cuh then sort that curve instead (they are always enqueued and exit at
// once when the flag is clear: the decision is taken on the device, no host synchronisation).
#pragma once
#include "common.cuh"
#include "sort.cuh"

namespace agn {

constexpr int kBkMeanLog = 11;                    // mean bucket population 2^11
constexpr int kBkCap = 4096;                      // slab slots per bucket
constexpr int kBkSampleLog = 6;                   // one sample per 64 keys
constexpr int kBkBinLog = 16;                     // CDF bins = top 16 key bits
constexpr int kBkBins = 1 << kBkBinLog;
constexpr int kBkSortThreads = 512;
constexpr int kBkSlotLog = 11;
constexpr int kBkSlots = 1 << kBkSlotLog;         // interpolation slots of the in-CTA sort

// Position of a key on the smoothed CDF: bin weights w = cnt * K + 1 (K = 2^24 / samples, so that the sampled mass is
// 2^24 and the add-one mass 2^16 whatever N is: keys of an unsampled bin still spread linearly over their own
// stretch instead of collapsing onto one point), pos = cumw * 2^16 + low16(key) * w < (2^24 + 2^16) * 2^16.
// The table holds (cumw << 7, w), so that pos >> 9 = tab.x + ((low16 * w) >> 9) fits 32 bits, and
// bs = bucket << 11 | slot = floor((pos >> 9) * M / 2^32) with M = floor(2^32 * nb * 2048 * 512 / (total * 2^16)):
// one multiply-high.  Every step is monotone in the key, and equal keys get equal bs.
// The number of bins follows the curve length (bl = log2 of it, 11 .. 16: a short curve has few buckets to tell apart,
// and a 65536-bin table per curve would cost more than its sort): bin = top bl key bits, the low 32 - bl bits
// interpolate, add-one mass 2^bl, pos >> (25 - bl) = tab.x + ((low * w) >> (25 - bl)); tab.x = cumw << 7 for every bl.
constexpr unsigned long long kBkTotalW = (1ull << 24) + (1ull << 16);       // bl = 16
__host__ __device__ constexpr unsigned long long bk_total_w(int bl) { return (1ull << 24) + (1ull << bl); }
inline int bk_binlog(long long N) {
    const int l = ilog2_u64((uint64_t)N) - 4;
    return l < 11 ? 11 : (l > kBkBinLog ? kBkBinLog : l);
}
__device__ __forceinline__ uint32_t bs_of(uint32_t key, const uint2* __restrict__ tab, uint32_t M, int bl = kBkBinLog) {
    const uint2 e = __ldg(tab + (key >> (32 - bl)));
    const uint32_t pos = e.x + (uint32_t)(((unsigned long long)(key & ((1u << (32 - bl)) - 1u)) * e.y) >> (25 - bl));
    return __umulhi(pos, M);
}
inline uint32_t bucket32_magic(uint32_t nb) {
    return (uint32_t)((((unsigned __int128)nb) << (32 + kBkSlotLog + 9)) / (kBkTotalW << 16));
}

// (kCdfSampleIlp samples per thread, all loads issued before the first histogram update: the kernel is bound by DRAM
//  latency -- every sample costs a 32-byte sector -- and one load in flight per thread left the memory system at 3 TB/s)
constexpr int kCdfSampleIlp = 4;
__global__ void __launch_bounds__(256) cdf_sample_kernel(const float* __restrict__ vals, uint32_t* __restrict__ hist,
                                                         uint32_t N, long long B, int bl = kBkBinLog) {
    const long long b = bidx();
    if (b >= B) return;
    const uint32_t nsamp = N >> kBkSampleLog;
    uint32_t bin[kCdfSampleIlp];
#pragma unroll
    for (int u = 0; u < kCdfSampleIlp; ++u) {
        const uint32_t i = (blockIdx.x * kCdfSampleIlp + u) * 256 + threadIdx.x;          // sample number
        // the sample of block i of 64 keys sits at a position that varies with i (no fixed phase)
        const uint32_t e = (i << kBkSampleLog) + ((i * 0x9E3779B1u) >> (32 - kBkSampleLog));
        bin[u] = i < nsamp ? (key_of(vals[(size_t)b * N + e]) >> (32 - bl)) : 0xffffffffu;
    }
#pragma unroll
    for (int u = 0; u < kCdfSampleIlp; ++u) {
        // neighbouring samples of a smooth series share their bin: one atomic per distinct bin and warp
        const uint32_t peers = __match_any_sync(0xffffffffu, bin[u]);
        if (bin[u] != 0xffffffffu && (threadIdx.x & 31) == (uint32_t)(__ffs(peers) - 1))
            atomicAdd(&hist[((size_t)b << bl) + bin[u]], (uint32_t)__popc(peers));
    }
}
inline unsigned cdf_sample_grid(uint32_t nsamp) { return (nsamp + 256 * kCdfSampleIlp - 1) / (256 * kCdfSampleIlp); }

// tab[bin] = (exclusive cumulative weight << 7, weight), weight = (cnt << logK) + 1.  kCdfChunks CTAs per curve, each
// owning 65536 / kCdfChunks consecutive bins: a CTA first adds up the weights of all bins before its chunk (the
// histogram is L2-resident, the reads are coalesced), then scans its own chunk 1024 bins at a time.  No CTA waits for
// another one.
constexpr int kCdfChunks = 16;
__device__ __forceinline__ uint32_t block_sum_1024(uint32_t v, uint32_t* ws) {      // sum over the CTA, returned to all
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if (lane == 0) ws[warp] = v;
    __syncthreads();
    uint32_t t = ws[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    return t;
}
// exclusive scan over the CTA's 1024 values; *total receives the sum
__device__ __forceinline__ uint32_t block_excl_scan_1024(uint32_t v, uint32_t* ws, uint32_t* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t n = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += n;
    }
    __syncthreads();
    if (lane == 31) ws[warp] = inc;
    __syncthreads();
    uint32_t w = ws[lane], wi = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t n = __shfl_up_sync(0xffffffffu, wi, o);
        if (lane >= o) wi += n;
    }
    *total = __shfl_sync(0xffffffffu, wi, 31);
    return inc - v + __shfl_sync(0xffffffffu, wi - w, warp);
}
inline unsigned cdf_chunks(int bl) { return (1u << bl) >= 1024u * kCdfChunks ? (unsigned)kCdfChunks : (1u << bl) / 1024u; }
__global__ void __launch_bounds__(1024) cdf_table_kernel(const uint32_t* __restrict__ hist, uint2* __restrict__ tab, int logK,
                                                         int bl = kBkBinLog, uint32_t chunks = kCdfChunks) {
    __shared__ uint32_t ws[32];
    const uint32_t curve = blockIdx.x / chunks, chunk = blockIdx.x % chunks;
    const uint32_t* h = hist + ((size_t)curve << bl);
    uint2* t = tab + ((size_t)curve << bl);
    const uint32_t PER = (1u << bl) / chunks;               // bins per chunk (a multiple of 1024)
    uint32_t before = 0;
    for (uint32_t i = threadIdx.x; i < chunk * PER; i += 1024) before += (h[i] << logK) + 1u;
    uint32_t run = block_sum_1024(before, ws);
    for (uint32_t i0 = chunk * PER; i0 < (chunk + 1) * PER; i0 += 1024) {
        const uint32_t w = (h[i0 + threadIdx.x] << logK) + 1u;
        uint32_t total;
        const uint32_t ex = block_excl_scan_1024(w, ws, &total);
        t[i0 + threadIdx.x] = make_uint2((run + ex) << 7, w);
        run += total;
    }
}

// ------------------------------------------------------------------------------------------------
// partition: two levels (coarse = high bits of the bucket number, fine = low bits), each a tile kernel that counts
// its keys per digit in shared memory, reserves one range per digit in the digit's slab (one global atomic per
// non-empty digit and tile), orders the tile by digit in shared memory and writes the runs out coalesced.
// The order inside a slab is arbitrary (see the header), so ranking inside the tile is a plain counter per digit.
// ------------------------------------------------------------------------------------------------
constexpr int kBkPartThreads = 256;
// keys per thread and tile, by level: the two sort levels run best on 2048-key tiles (6 CTAs per SM: 1.37 against
// 1.49 ms per pass with 4096), the scatter's bin step on 4096-key tiles (1.36 against 1.57 ms)
__host__ __device__ constexpr int bk_part_ept(int level) { return level == 2 ? 16 : 8; }
__host__ __device__ constexpr int bk_part_tile(int level) { return kBkPartThreads * bk_part_ept(level); }
constexpr int kBkMaxDigits = 256;

template <int LEVEL> struct PartSmem {
    uint2 stage[bk_part_tile(LEVEL)];
    unsigned char sdig[bk_part_tile(LEVEL)];
    uint32_t cnt[kBkMaxDigits];         // digit populations of the tile
    uint32_t lstart[kBkMaxDigits];      // first stage position of the digit
    uint32_t gdst[kBkMaxDigits];        // slab position of stage position 0 of the digit (may wrap: used modulo 2^32)
    uint32_t wsum[kBkPartThreads / 32];
};

struct PartArgs {
    const float* vals;          // LEVEL 0 input [B][N]; LEVEL 2: the sorted ERDF draw [B][N]
    const uint32_t* idx_new;    // LEVEL 2 (rank scatter, bin step): permutation of this iteration,
    const uint32_t* idx_old;    //          of the previous one,
    unsigned long long* changed;//          and the change counters [B]
    const uint2* in;            // LEVEL 1 input: coarse slabs [B][nc][cap_in]
    const uint32_t* in_count;   // LEVEL 1: populations of the coarse slabs [B][nc]
    uint2* out;                 // slabs [B][n_out][cap_out]
    uint32_t* cursor;           // [B][n_out] zero on entry
    uint32_t* overflow;         // [B]
    const uint2* tab;           // [B][65536]
    uint32_t N, nb;             // keys per curve, fine buckets per curve
    uint32_t M;                 // bucket32_magic(nb)
    uint32_t lb;                // low (fine) bits of the bucket number; LEVEL 2: shift of the destination window
    uint32_t nc;                // coarse slabs per curve
    uint32_t cap_in, cap_out;
    uint32_t tiles_in;          // LEVEL 1: tiles per coarse slab
    const uint32_t* gate;       // LEVEL 2: if not null, only the curves with gate[b] != 0 are processed
    long long B;
};

template <int LEVEL>
__global__ void __launch_bounds__(kBkPartThreads, (LEVEL == 2 ? 4 : 6)) bucket_part_kernel(PartArgs a) {
    constexpr int kBkPartEpt = bk_part_ept(LEVEL), kBkPartTile = bk_part_tile(LEVEL);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    PartSmem<LEVEL>& sm = *reinterpret_cast<PartSmem<LEVEL>*>(smem_raw);
    const long long b = bidx();
    if (b >= a.B) return;
    if (LEVEL == 2 && a.gate && a.gate[b] == 0u) return;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const uint2* tab = a.tab + (size_t)b * kBkBins;
    uint32_t coarse = 0, tile = blockIdx.x, n_in = a.N;
    if (LEVEL == 1) {
        coarse = blockIdx.x / a.tiles_in;
        tile = blockIdx.x - coarse * a.tiles_in;
        n_in = min(a.in_count[(size_t)b * a.nc + coarse], a.cap_in);
        if (tile * kBkPartTile >= n_in) return;
    }
    sm.cnt[t] = 0u;
    const uint32_t e0 = tile * kBkPartTile + t;
    uint2 kv[kBkPartEpt];
    if (LEVEL == 0) {
        const float* v = a.vals + (size_t)b * a.N;
#pragma unroll
        for (int j = 0; j < kBkPartEpt; ++j) kv[j] = make_uint2(key_of(__ldcs(v + e0 + j * kBkPartThreads)), e0 + j * kBkPartThreads);
    } else if (LEVEL == 2) {
        // L5 bin step: (value, destination) pairs by destination window; L5's change count on the way
        const size_t g0 = (size_t)b * a.N + e0;
        uint32_t diff = 0;
#pragma unroll
        for (int j = 0; j < kBkPartEpt; ++j) {
            const uint32_t dst = __ldcs(a.idx_new + g0 + j * kBkPartThreads);
            diff += (dst != __ldcs(a.idx_old + g0 + j * kBkPartThreads));
            kv[j] = make_uint2(__float_as_uint(__ldcs(a.vals + g0 + j * kBkPartThreads)), dst);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) diff += __shfl_xor_sync(0xffffffffu, diff, o);
        if (lane == 0 && diff) atomicAdd(&a.changed[b], (unsigned long long)diff);
    } else {
        const uint2* v = a.in + ((size_t)b * a.nc + coarse) * a.cap_in;
#pragma unroll
        for (int j = 0; j < kBkPartEpt; ++j)
            if (e0 + j * kBkPartThreads < n_in) kv[j] = __ldcs(v + e0 + j * kBkPartThreads);
    }
    __syncthreads();
    // digit and arrival number inside the digit
    uint32_t dr[kBkPartEpt];            // digit << 16 | arrival number
    const uint32_t dmask = (LEVEL == 0) ? 0xffffffffu : ((1u << a.lb) - 1u);
    const uint32_t dshift = kBkSlotLog + ((LEVEL == 0) ? a.lb : 0u);
#pragma unroll
    for (int j = 0; j < kBkPartEpt; ++j) {
        const bool valid = (LEVEL != 1) || (e0 + j * kBkPartThreads < n_in);
        const uint32_t d = (LEVEL == 2) ? (kv[j].y >> a.lb) : (valid ? ((bs_of(kv[j].x, tab, a.M) >> dshift) & dmask) : 0xffffu);
        uint32_t r = 0;
        if (LEVEL == 0) {
            // coarse digits of neighbouring samples of a smooth series mostly agree: one atomic for lane 0's group
            const uint32_t d0 = __shfl_sync(0xffffffffu, d, 0);
            const uint32_t same = __ballot_sync(0xffffffffu, d == d0);
            if (lane == 0) r = atomicAdd(&sm.cnt[d0], (uint32_t)__popc(same));
            r = __shfl_sync(0xffffffffu, r, 0) + __popc(same & ((1u << lane) - 1u));
            if (d != d0) r = atomicAdd(&sm.cnt[d], 1u);
        } else if (valid) {
            r = atomicAdd(&sm.cnt[d], 1u);          // fine digits / destination windows are as good as random
        }
        dr[j] = (d << 16) | r;
    }
    __syncthreads();
    // thread == digit: reserve the digit's range in its slab, exclusive scan of the populations
    {
        const uint32_t c = sm.cnt[t];
        const uint32_t slab = (LEVEL != 1) ? (uint32_t)t : ((coarse << a.lb) | (uint32_t)t);
        const uint32_t n_out = (LEVEL != 1) ? a.nc : a.nb;
        uint32_t g = 0;
        if (c) {
            g = atomicAdd(&a.cursor[(size_t)b * n_out + slab], c);
            if (LEVEL != 2 && g + c > a.cap_out) a.overflow[b] = 1u;
        }
        uint32_t inc = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t m = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += m;
        }
        if (lane == 31) sm.wsum[warp] = inc;
        __syncthreads();
        uint32_t add = 0;
#pragma unroll
        for (int w = 0; w < kBkPartThreads / 32; ++w) add += (w < warp) ? sm.wsum[w] : 0u;
        const uint32_t ls = inc - c + add;
        sm.lstart[t] = ls;
        sm.gdst[t] = g - ls;
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kBkPartEpt; ++j) {
        const bool valid = (LEVEL != 1) || (e0 + j * kBkPartThreads < n_in);
        if (valid) {
            const uint32_t d = dr[j] >> 16, s = sm.lstart[d] + (dr[j] & 0xffffu);
            sm.stage[s] = kv[j];
            if (LEVEL != 2) sm.sdig[s] = (unsigned char)d;          // level 2 reads the digit off the pair itself
        }
    }
    __syncthreads();
    const uint32_t n_tile = min((uint32_t)kBkPartTile, n_in - tile * kBkPartTile);
    const uint32_t n_out = (LEVEL != 1) ? a.nc : a.nb;
    uint2* out = a.out + (size_t)b * n_out * a.cap_out;
    const uint32_t slab0 = (LEVEL != 1) ? 0u : (coarse << a.lb);
#pragma unroll 4
    for (uint32_t s = t; s < n_tile; s += kBkPartThreads) {
        const uint2 pr = sm.stage[s];
        const uint32_t d = (LEVEL == 2) ? (pr.y >> a.lb) : (uint32_t)sm.sdig[s];
        const uint32_t off = sm.gdst[d] + s;
        if (off < a.cap_out) out[(size_t)(slab0 + d) * a.cap_out + off] = pr;
    }
}

// base[k] = sum of the populations of buckets < k (populations clamped to the slab).  `chunks` CTAs per curve, same
// scheme as cdf_table_kernel: sum of everything before the chunk, then a scan of the chunk.
__global__ void __launch_bounds__(1024) bucket_base_kernel(const uint32_t* __restrict__ cursor, uint32_t* __restrict__ base,
                                                           uint32_t nb, uint32_t chunks, uint32_t cap) {
    __shared__ uint32_t ws[32];
    const uint32_t curve = blockIdx.x / chunks, chunk = blockIdx.x % chunks;
    const uint32_t* c = cursor + (size_t)curve * nb;
    uint32_t* o = base + (size_t)curve * nb;
    const uint32_t per = nb / chunks;
    uint32_t before = 0;
    for (uint32_t i = threadIdx.x; i < chunk * per; i += 1024) before += min(c[i], cap);
    uint32_t run = block_sum_1024(before, ws);
    for (uint32_t k0 = chunk * per; k0 < (chunk + 1) * per; k0 += 1024) {
        const uint32_t k = k0 + threadIdx.x;
        const uint32_t n = (k < (chunk + 1) * per) ? min(c[k], cap) : 0u;
        uint32_t total;
        const uint32_t ex = block_excl_scan_1024(n, ws, &total);
        if (k < (chunk + 1) * per) o[k] = run + ex;
        run += total;
    }
}

// klo[k] = smallest key that bs_of() sends to bucket k (k = 0 .. nb; klo[nb] = 2^32 - 1): the bucket's keys lie in
// [klo[k], klo[k+1]), so inside the finish kernel a slot is a plain linear map of the key onto that interval -- no
// table look-up per key there.  One thread per bucket: invert umulhi(pos, M) >= k << kBkSlotLog, then the table.
__global__ void __launch_bounds__(256) bucket_bounds_kernel(const uint2* __restrict__ tabs, uint32_t* __restrict__ klo,
                                                            uint32_t nb, uint32_t M, int slot_log, long long B,
                                                            int bl = kBkBinLog) {
    const long long b = bidx();
    if (b >= B) return;
    const uint32_t k = blockIdx.x * 256 + threadIdx.x;
    if (k > nb) return;
    uint32_t* out = klo + (size_t)b * (nb + 1);
    if (k == nb) { out[k] = 0xffffffffu; return; }
    const uint2* tab = tabs + ((size_t)b << bl);
    const unsigned long long want = ((unsigned long long)k << slot_log) << 32;
    const unsigned long long P = (want + M - 1) / M;               // smallest pos32 with umulhi(pos32, M) >= k << slotlog
    uint32_t lo = 0, hi = (1u << bl) - 1u;                          // largest bin with tab[bin].x <= P
    while (lo < hi) {
        const uint32_t mid = (lo + hi + 1) >> 1;
        if ((unsigned long long)tab[mid].x <= P) lo = mid; else hi = mid - 1;
    }
    const uint2 e = tab[lo];
    const unsigned long long need = (P - e.x) << (25 - bl);         // low * w >= need
    const unsigned long long low = min((need + e.y - 1) / e.y, (unsigned long long)((1u << (32 - bl)) - 1u));
    out[k] = (lo << (32 - bl)) | (uint32_t)low;
}

struct BkSmem {
    unsigned long long pair[kBkCap];      // (key << 32) | index, grouped by slot
    uint32_t cnt[kBkSlots];               // slot populations, then slot starts, then slot ends
    unsigned short slot[kBkCap];          // slot of slab element e
    uint32_t wsum[kBkSortThreads / 32];
};

__global__ void __launch_bounds__(kBkSortThreads, 4) bucket_sort_kernel(const uint2* __restrict__ slabs,
                                                                        const uint32_t* __restrict__ cursor,
                                                                        const uint32_t* __restrict__ base,
                                                                        const uint32_t* __restrict__ overflow,
                                                                        const uint32_t* __restrict__ klos,
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
    // linear slot map of this bucket's key interval (the outermost buckets, whose interval is open-ended, borrow
    // twice the width of their neighbour); monotone in the key, equal keys share a slot, out-of-range keys clamp
    uint32_t klo, width;
    {
        const uint32_t* kb = klos + (size_t)b * (nb + 1);
        klo = kb[bk];
        width = kb[bk + 1] - klo;
        if (bk + 1 == nb && nb > 1) width = 2u * min(klo - kb[bk - 1], 0x7fffffffu);
        if (bk == 0 && nb > 2) { width = 2u * min(kb[2] - kb[1], 0x7fffffffu); klo = kb[1] > width ? kb[1] - width : 0u; width = kb[1] - klo; }
    }
    const float scale = (float)kBkSlots / ((float)width + 1.0f);
    auto slot_of = [&](uint32_t key) -> uint32_t {
        const uint32_t d = key > klo ? key - klo : 0u;
        return min((uint32_t)(__uint2float_rz(d) * scale), (uint32_t)(kBkSlots - 1));
    };
    constexpr int PER = kBkSlots / kBkSortThreads;
#pragma unroll
    for (int i = 0; i < PER; ++i) sm.cnt[i * kBkSortThreads + t] = 0u;
    __syncthreads();
    // 1. slot populations (the slab stays in L2 for step 3)
#pragma unroll 4
    for (uint32_t e = t; e < n; e += kBkSortThreads) {
        const uint32_t s = slot_of(__ldcg(&sl[e].x));
        atomicAdd(&sm.cnt[s], 1u);
        sm.slot[e] = (unsigned short)s;
    }
    __syncthreads();
    // 2. exclusive scan of the slot populations (PER consecutive slots per thread)
    {
        static_assert(PER % 4 == 0, "whole uint4s of slot counters per thread");
        uint32_t c[PER], sum = 0;
#pragma unroll
        for (int i = 0; i < PER / 4; ++i) {
            const uint4 c4 = reinterpret_cast<const uint4*>(sm.cnt)[t * (PER / 4) + i];
            c[4 * i] = c4.x; c[4 * i + 1] = c4.y; c[4 * i + 2] = c4.z; c[4 * i + 3] = c4.w;
            sum += c4.x + c4.y + c4.z + c4.w;
        }
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
        for (int i = 0; i < PER / 4; ++i) {
            uint4 o4;
            o4.x = run; run += c[4 * i];
            o4.y = run; run += c[4 * i + 1];
            o4.z = run; run += c[4 * i + 2];
            o4.w = run; run += c[4 * i + 3];
            reinterpret_cast<uint4*>(sm.cnt)[t * (PER / 4) + i] = o4;
        }
    }
    __syncthreads();
    // 3. every pair into its slot's range (any order); cnt[s] ends as the END of slot s
#pragma unroll 4
    for (uint32_t e = t; e < n; e += kBkSortThreads) {
        const uint2 kv = __ldcs(sl + e);
        const uint32_t q = atomicAdd(&sm.cnt[sm.slot[e]], 1u);
        sm.pair[q] = ((unsigned long long)kv.x << 32) | kv.y;
    }
    __syncthreads();
    // 4. exact rank of every pair among its slot mates (they are contiguous; the 64-bit (key, index) words are all
    //    distinct), one pair per thread at a time, and the index goes to that rank
    uint32_t* io = idx_out + (size_t)b * N + r0;
    float* so = sorted_out ? sorted_out + (size_t)b * N + r0 : nullptr;
#pragma unroll 2
    for (uint32_t q = t; q < n; q += kBkSortThreads) {
        const unsigned long long v = sm.pair[q];
        const uint32_t key = (uint32_t)(v >> 32);
        const uint32_t s = slot_of(key);
        const uint32_t z = sm.cnt[s];
        const uint32_t a = s ? sm.cnt[s - 1] : 0u;
        uint32_t r = q;
        if (z - a > 1u) {
            r = a;
            for (uint32_t h = a; h < z; ++h) r += (sm.pair[h] < v);
        }
        io[r] = (uint32_t)v;
        if (so) so[r] = val_of(key);
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
    cudaFuncSetAttribute(bucket_part_kernel<0>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaFuncSetAttribute(bucket_part_kernel<1>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaFuncSetAttribute(bucket_part_kernel<2>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaError_t e = cudaFuncSetAttribute(bucket_part_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(PartSmem<0>));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bucket_part_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(PartSmem<1>));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bucket_part_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(PartSmem<2>));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bucket_sort_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(BkSmem));
    return e;
}

// geometry of the two partition levels for N keys per curve
struct BkGeom {
    uint32_t nb, lb, nc, cap1, tiles1;
};
inline BkGeom bucket32_geom(long long N) {
    BkGeom g;
    g.nb = (uint32_t)(N >> kBkMeanLog);
    const int nbits = ilog2_u64((uint64_t)g.nb);
    g.lb = (uint32_t)(nbits / 2);
    g.nc = g.nb >> g.lb;                                        // <= 256
    const uint32_t mean1 = (uint32_t)(N / g.nc);
    g.cap1 = mean1 + mean1 / 2;                                 // coarse slabs: 50% head room
    g.tiles1 = (g.cap1 + bk_part_tile(1) - 1) / bk_part_tile(1);
    return g;
}

// pair scratch (in uint2 units): fine slabs [B][nb][kBkCap] then coarse slabs [B][nc][cap1]
inline size_t bucket32_pair_elems(long long B, long long N) {
    const BkGeom g = bucket32_geom(N);
    return (size_t)B * g.nb * kBkCap + (size_t)B * g.nc * g.cap1;
}

// control words: hist [B][65536] u32 | cursor2 [B][nb] | cursor1 [B][256] | overflow [B] (zeroed per call) |
//                tab [B][65536] uint2 | base [B][nb]
inline size_t bucket32_zero_bytes(long long B, long long N) {
    const size_t nb = (size_t)(N >> kBkMeanLog);
    return (size_t)B * kBkBins * 4 + (size_t)B * nb * 4 + (size_t)B * kBkMaxDigits * 4 + (size_t)B * 4;
}
inline size_t bucket32_ctl_bytes(long long B, long long N) {
    const size_t nb = (size_t)(N >> kBkMeanLog);
    return align_up(bucket32_zero_bytes(B, N), 256) + align_up((size_t)B * kBkBins * 8, 256) + align_up((size_t)B * nb * 4, 256) +
           align_up((size_t)B * (nb + 1) * 4, 256);
}

// vals [B][N] -> idx_out (and optionally the sorted values) for the curves whose buckets all fit; *overflow_out points
// at the per-curve flags (1 = not sorted here).  pairs: bucket32_pair_elems(B, N) (key, index) pairs of scratch.
inline cudaError_t bucket32_sort(const float* vals, uint32_t* idx_out, float* sorted_out, long long B, long long N,
                                 uint2* pairs, void* ctl, const uint32_t** overflow_out, cudaStream_t st) {
    const BkGeom g = bucket32_geom(N);
    unsigned char* w = (unsigned char*)ctl;
    uint32_t* hist = (uint32_t*)w;
    uint32_t* cursor2 = hist + (size_t)B * kBkBins;
    uint32_t* cursor1 = cursor2 + (size_t)B * g.nb;
    uint32_t* overflow = cursor1 + (size_t)B * kBkMaxDigits;
    const size_t zero_bytes = bucket32_zero_bytes(B, N);
    w += align_up(zero_bytes, 256);
    uint2* tab = (uint2*)w; w += align_up((size_t)B * kBkBins * 8, 256);
    uint32_t* base = (uint32_t*)w; w += align_up((size_t)B * g.nb * 4, 256);
    uint32_t* klo = (uint32_t*)w;
    uint2* slabs2 = pairs;
    uint2* slabs1 = pairs + (size_t)B * g.nb * kBkCap;
    cudaError_t e;
    // the CDF tables are re-estimated in every call: reusing them for 3 out of 4 E13 iterations was measured to overflow
    // slabs (stale table -> LSD fallback) often enough to cost more than the 0.25 ms it saves
    e = cudaMemsetAsync(hist, 0, zero_bytes, st);
    if (e != cudaSuccess) return e;
    const uint32_t nsamp = (uint32_t)(N >> kBkSampleLog);
    AGN_LAUNCH(K_SORT_CDF, st, (cdf_sample_kernel<<<bgrid(cdf_sample_grid(nsamp), B), 256, 0, st>>>(vals, hist, (uint32_t)N, B)));
    AGN_LAUNCH(K_SORT_CDF, st, (cdf_table_kernel<<<(unsigned)(B * kCdfChunks), 1024, 0, st>>>(hist, tab, 24 - (ilog2_u64((uint64_t)N) - kBkSampleLog))));
    AGN_LAUNCH(K_SORT_CDF, st, (bucket_bounds_kernel<<<bgrid((g.nb + 256) / 256, B), 256, 0, st>>>(tab, klo, g.nb, bucket32_magic(g.nb), kBkSlotLog, B)));
    PartArgs a;
    memset(&a, 0, sizeof(a));
    a.vals = vals; a.in = slabs1; a.in_count = cursor1; a.overflow = overflow; a.tab = tab;
    a.N = (uint32_t)N; a.nb = g.nb; a.M = bucket32_magic(g.nb); a.lb = g.lb; a.nc = g.nc; a.cap_in = g.cap1; a.tiles_in = g.tiles1; a.B = B;
    a.out = slabs1; a.cursor = cursor1; a.cap_out = g.cap1;
    AGN_LAUNCH(K_SORT_PART0, st, (bucket_part_kernel<0><<<bgrid((unsigned)(N / bk_part_tile(0)), B), kBkPartThreads, sizeof(PartSmem<0>), st>>>(a)));
    a.out = slabs2; a.cursor = cursor2; a.cap_out = kBkCap;
    AGN_LAUNCH(K_SORT_PART1, st, (bucket_part_kernel<1><<<bgrid(g.tiles1 * g.nc, B), kBkPartThreads, sizeof(PartSmem<1>), st>>>(a)));
    const uint32_t bchunks = g.nb >= 16384 ? 16u : (g.nb >= 1024 ? g.nb / 1024 : 1u);
    AGN_LAUNCH(K_SORT_CDF, st, (bucket_base_kernel<<<(unsigned)(B * bchunks), 1024, 0, st>>>(cursor2, base, g.nb, bchunks, (uint32_t)kBkCap)));
    AGN_LAUNCH(K_SORT_BUCKET, st, (bucket_sort_kernel<<<bgrid(g.nb, B), kBkSortThreads, sizeof(BkSmem), st>>>(
        slabs2, cursor2, base, overflow, klo, idx_out, sorted_out, (uint32_t)N, g.nb, B)));
    *overflow_out = overflow;
    return cudaGetLastError();
}

}  // namespace agn

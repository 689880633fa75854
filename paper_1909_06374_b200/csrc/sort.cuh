// sort.cuh -- segmented, stable, ascending radix argsort (one segment per light curve), sm_100a.
//   * N <= kCtaSortMax<T>: the whole segment is sorted by one CTA in shared memory (all digit passes
//     on chip; HBM traffic = read keys once + write indices once).
//   * larger N: least-significant-digit passes over HBM, 8-bit digits, one sweep per pass with
//     decoupled look-back across tiles ("onesweep"): pass 0 reads raw values (index implicit),
//     the last pass writes indices only.
// Ranking inside a tile: warp-striped key arrangement, __match_any_sync digit matching, per-warp digit
// counters in shared memory (warp-shuffle histograms).  Stable: ties keep the lower time index first
// (O6 step 4; the tie-break is part of the result).
#pragma once
#include "common.cuh"

namespace agn {

constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;

__device__ __forceinline__ uint32_t lanemask_lt() {
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// Shared-memory scratch used by rank_keys: cm[W][256] {lane mask of the current round, running count},
// tile_off[256], tile_cnt[256], wsum[8]
template <int THREADS> struct RankScratch {
    static constexpr int W = THREADS / 32;
    static constexpr size_t words = (size_t)2 * W * kRadix + 2 * kRadix + 8;
};

// Computes, for every key of the tile, its position in the tile's stable order by the digit at `shift`.
// Keys are held warp-striped: item j of lane l of warp w is tile element w*32*KPT + j*32 + l.
// Digit matching inside a warp round does not use MATCH.ANY (measured on B200: ~60 clk per warp instruction
// for 8-bit digits, it loops over the distinct values): every lane ORs its lane bit into a per-(warp, digit)
// mask word in shared memory, reads the mask back together with the running count (one 64-bit load), and the
// lowest lane of each digit group folds the group size into the count and clears the mask.  Stable: the rank
// inside a round is the number of lower lanes with the same digit.
template <typename KeyU, int THREADS, int KPT>
__device__ __forceinline__ void rank_keys(const KeyU (&key)[KPT], int shift, uint32_t (&pos)[KPT],
                                          uint32_t* scratch) {
    constexpr int W = THREADS / 32;
    uint2* cm = reinterpret_cast<uint2*>(scratch);        // [W][256]
    uint32_t* tile_off = scratch + 2 * W * kRadix;
    uint32_t* tile_cnt = tile_off + kRadix;
    uint32_t* wsum = tile_cnt + kRadix;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < W * kRadix; i += THREADS) cm[i] = make_uint2(0u, 0u);
    __syncthreads();
    uint32_t r[KPT];
    const uint32_t lt = lanemask_lt();
    const uint32_t bit = 1u << lane;
    uint2* cw = cm + warp * kRadix;
#pragma unroll
    for (int j = 0; j < KPT; ++j) {
        const uint32_t d = (uint32_t)(key[j] >> shift) & (kRadix - 1);
        atomicOr(&cw[d].x, bit);
        __syncwarp();
        const uint2 mc = cw[d];
        r[j] = mc.y + __popc(mc.x & lt);
        __syncwarp();
        if ((mc.x & lt) == 0u) cw[d] = make_uint2(0u, mc.y + __popc(mc.x));
        __syncwarp();
    }
    __syncthreads();
    if (threadIdx.x < kRadix) {
        uint32_t run = 0;
#pragma unroll 4
        for (int w = 0; w < W; ++w) {
            uint32_t t = cm[w * kRadix + threadIdx.x].y;
            cm[w * kRadix + threadIdx.x].y = run;
            run += t;
        }
        tile_cnt[threadIdx.x] = run;
        // exclusive scan over the 256 digits: warp scan + 8 warp totals
        uint32_t inc = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t n = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += n;
        }
        if (lane == 31) wsum[warp] = inc;
        tile_off[threadIdx.x] = inc - run;   // exclusive within the warp
    }
    __syncthreads();
    if (threadIdx.x < kRadix) {
        uint32_t add = 0;
        for (int w = 0; w < warp; ++w) add += wsum[w];
        tile_off[threadIdx.x] += add;
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < KPT; ++j) {
        uint32_t d = (uint32_t)(key[j] >> shift) & (kRadix - 1);
        pos[j] = tile_off[d] + cw[d].y + r[j];
    }
}

// ------------------------------------------------------------------------------------------------
// one CTA per segment, everything in shared memory
// ------------------------------------------------------------------------------------------------
template <typename T, int THREADS, int KPT>
__global__ void __launch_bounds__(THREADS) cta_argsort_kernel(const T* __restrict__ vals, uint32_t* __restrict__ idx_out,
                                                              T* __restrict__ sorted_out, int N, long long seg_stride) {
    typedef typename KeyT<T>::type KeyU;
    constexpr int TILE = THREADS * KPT;
    constexpr int NP = KeyT<T>::bits / kRadixBits;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    KeyU* sk = reinterpret_cast<KeyU*>(smem_raw);
    uint32_t* si = reinterpret_cast<uint32_t*>(sk + TILE);
    uint32_t* scratch = si + TILE;
    const long long b = blockIdx.x;
    const T* v = vals + b * seg_stride;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    KeyU key[KPT];
    uint32_t idx[KPT], pos[KPT];
#pragma unroll
    for (int j = 0; j < KPT; ++j) {
        int e = warp * 32 * KPT + j * 32 + lane;
        key[j] = (e < N) ? key_of(v[e]) : (KeyU)~(KeyU)0;
        idx[j] = (uint32_t)e;
    }
    for (int p = 0; p < NP; ++p) {
        rank_keys<KeyU, THREADS, KPT>(key, p * kRadixBits, pos, scratch);
#pragma unroll
        for (int j = 0; j < KPT; ++j) { sk[pos[j]] = key[j]; si[pos[j]] = idx[j]; }
        __syncthreads();
        if (p < NP - 1) {
#pragma unroll
            for (int j = 0; j < KPT; ++j) {
                int e = warp * 32 * KPT + j * 32 + lane;
                key[j] = sk[e]; idx[j] = si[e];
            }
        }
    }
    for (int e = threadIdx.x; e < N; e += THREADS) {
        idx_out[b * seg_stride + e] = si[e];
        if (sorted_out) sorted_out[b * seg_stride + e] = val_of(sk[e]);
    }
}

// ------------------------------------------------------------------------------------------------
// HBM path: digit histogram of every pass in one read, then one sweep per pass
// ------------------------------------------------------------------------------------------------
template <typename T, int THREADS>
__global__ void __launch_bounds__(THREADS) digit_hist_kernel(const T* __restrict__ vals, uint32_t* __restrict__ hist,
                                                             long long N, long long seg_stride, int chunk, long long B,
                                                             const uint32_t* __restrict__ gate) {
    typedef typename KeyT<T>::type KeyU;
    constexpr int NP = KeyT<T>::bits / kRadixBits;
    __shared__ uint32_t h[NP * kRadix];
    if (gate && bidx() < B && gate[bidx()] == 0u) return;      // curve already sorted by the bucket path
    for (int i = threadIdx.x; i < NP * kRadix; i += THREADS) h[i] = 0;
    __syncthreads();
    const long long b = bidx();
    if (b >= B) return;
    const T* v = vals + b * seg_stride;
    long long beg = (long long)blockIdx.x * chunk, end = beg + chunk;
    if (end > N) end = N;
    for (long long e = beg + threadIdx.x; e < end; e += THREADS) {
        KeyU k = key_of(v[e]);
#pragma unroll
        for (int p = 0; p < NP; ++p) atomicAdd(&h[p * kRadix + ((uint32_t)(k >> (p * kRadixBits)) & (kRadix - 1))], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < NP * kRadix; i += THREADS)
        if (h[i]) atomicAdd(&hist[b * NP * kRadix + i], h[i]);
}

constexpr int kLookBatch = 8;
constexpr uint32_t kFlagAgg = 1u << 30, kFlagInc = 2u << 30, kFlagMask = 3u << 30;

template <typename T> struct SweepArgs {
    typedef typename KeyT<T>::type KeyU;
    const T* vals;            // FIRST: raw values
    const KeyU* keys_in;
    const uint32_t* idx_in;
    KeyU* keys_out;
    uint32_t* idx_out;
    T* sorted_out;            // LAST only, may be NULL
    long long N, seg_stride;
    int shift;
    const uint32_t* hist;     // [B][NP][256] digit counts
    int pass, npass;
    uint32_t* status;         // [B][ntiles][256] for this pass, zero-initialised
    uint32_t* ticket;         // [B] for this pass, zero-initialised
    int ntiles;
    long long B;
};

template <typename T, int THREADS, int KPT, bool FIRST, bool LAST>
__global__ void __launch_bounds__(THREADS, (sizeof(T) == 4 ? 2 : 1)) onesweep_kernel(SweepArgs<T> a) {
    typedef typename KeyT<T>::type KeyU;
    constexpr int TILE = THREADS * KPT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    KeyU* sk = reinterpret_cast<KeyU*>(smem_raw);
    uint32_t* si = reinterpret_cast<uint32_t*>(sk + TILE);
    uint32_t* scratch = si + TILE;
    constexpr int W = THREADS / 32;
    uint32_t* tile_off = scratch + 2 * W * kRadix;
    uint32_t* tile_cnt = tile_off + kRadix;
    __shared__ long long goff[kRadix];
    __shared__ uint32_t s_tile;
    __shared__ uint32_t s_wsum[8];
    const long long b = bidx();
    if (b >= a.B) return;
    if (threadIdx.x == 0) s_tile = atomicAdd(&a.ticket[b], 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const long long base = (long long)tile * TILE;
    const long long segoff = b * a.seg_stride;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    long long nvalid_ll = a.N - base;
    const int nvalid = nvalid_ll > TILE ? TILE : (int)nvalid_ll;
    KeyU key[KPT];
    uint32_t idx[KPT], pos[KPT];
#pragma unroll
    for (int j = 0; j < KPT; ++j) {
        int e = warp * 32 * KPT + j * 32 + lane;
        if (e < nvalid) {
            if (FIRST) { key[j] = key_of(a.vals[segoff + base + e]); idx[j] = (uint32_t)(base + e); }
            else { key[j] = a.keys_in[segoff + base + e]; idx[j] = a.idx_in[segoff + base + e]; }
        } else { key[j] = (KeyU)~(KeyU)0; idx[j] = 0xffffffffu; }
    }
    rank_keys<KeyU, THREADS, KPT>(key, a.shift, pos, scratch);
    // global start of every digit (exclusive scan of this pass's histogram) + look-back over earlier tiles
    if (threadIdx.x < kRadix) {
        const int d = threadIdx.x;
        uint32_t cntd = a.hist[(b * a.npass + a.pass) * kRadix + d];
        uint32_t inc = cntd;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t n = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += n;
        }
        if (lane == 31) s_wsum[warp] = inc;
        uint32_t gstart = inc - cntd;
        // named barrier over the first 256 threads (8 warps)
        asm volatile("bar.sync 1, 256;");
        for (int w = 0; w < warp; ++w) gstart += s_wsum[w];
        uint32_t agg = tile_cnt[d];
        if (d == kRadix - 1) agg -= (uint32_t)(TILE - nvalid);      // padding keys sit at the end of digit 255
        volatile uint32_t* st = a.status + ((size_t)b * a.ntiles) * kRadix;
        uint32_t excl = 0;
        if (tile == 0) {
            st[(size_t)tile * kRadix + d] = kFlagInc | agg;
        } else {
            st[(size_t)tile * kRadix + d] = kFlagAgg | agg;
            // decoupled look-back, kLookBatch predecessors per round trip (independent loads)
            int t = (int)tile - 1;
            bool done = false;
            while (!done) {
                uint32_t sv[kLookBatch];
#pragma unroll
                for (int i = 0; i < kLookBatch; ++i) sv[i] = (t - i >= 0) ? st[(size_t)(t - i) * kRadix + d] : (2u << 30);
                int used = kLookBatch;
#pragma unroll
                for (int i = 0; i < kLookBatch; ++i) {
                    if (!done && used == kLookBatch) {
                        const uint32_t f = sv[i] & kFlagMask;
                        if (f == 0) used = i;                      // not published yet: retry from here
                        else {
                            excl += sv[i] & ~kFlagMask;
                            if (f == kFlagInc) done = true;
                        }
                    }
                }
                t -= used;
            }
            st[(size_t)tile * kRadix + d] = kFlagInc | (excl + agg);
        }
        goff[d] = (long long)gstart + (long long)excl - (long long)tile_off[d];
    }
#pragma unroll
    for (int j = 0; j < KPT; ++j) { sk[pos[j]] = key[j]; si[pos[j]] = idx[j]; }
    __syncthreads();
    for (int s = threadIdx.x; s < nvalid; s += THREADS) {
        KeyU k = sk[s];
        uint32_t d = (uint32_t)(k >> a.shift) & (kRadix - 1);
        long long g = segoff + goff[d] + s;
        if (!LAST) a.keys_out[g] = k;
        a.idx_out[g] = si[s];
        if (LAST && a.sorted_out) a.sorted_out[g] = val_of(k);
    }
}

// ------------------------------------------------------------------------------------------------
// L5 for segments much larger than L2: two-level rank scatter.
//   bin pass   reads idx_new[r], idx_old[r], sorted[r]; counts idx_new != idx_old; appends (value, dst)
//              to the bin dst >> shift (256 bins per segment).  idx_new is a permutation, so bin d
//              receives exactly 2^shift pairs: its region is [d << shift, (d+1) << shift) and only a
//              cursor per bin is needed (order inside a bin is irrelevant: every pair carries its dst).
//   place pass streams the pairs of one bin and stores x[dst]; all stores of a bin fall into a window of
//              2^shift values, which stays in L2 until every sector of it is complete.
// A direct x[idx_new[r]] = sorted[r] over a 256 MB segment costs a 32-byte sector read-modify-write
// in HBM per 4-byte value; the two passes move 20 + 12 bytes per value instead.
// ------------------------------------------------------------------------------------------------
template <typename T, int THREADS, int KPT>
__global__ void __launch_bounds__(THREADS, (sizeof(T) == 4 ? 2 : 1)) scatter_bin_kernel(const uint32_t* __restrict__ idx_new,
                                                              const uint32_t* __restrict__ idx_old,
                                                              const T* __restrict__ sorted, T* __restrict__ pv,
                                                              uint32_t* __restrict__ pd, long long N, int shift,
                                                              uint32_t* __restrict__ cursor,
                                                              unsigned long long* __restrict__ changed, long long B) {
    constexpr int TILE = THREADS * KPT;
    constexpr int W = THREADS / 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T* sv = reinterpret_cast<T*>(smem_raw);
    uint32_t* sd = reinterpret_cast<uint32_t*>(sv + TILE);
    uint32_t* scratch = sd + TILE;
    uint32_t* tile_off = scratch + 2 * W * kRadix;
    uint32_t* tile_cnt = tile_off + kRadix;
    __shared__ long long goff[kRadix];
    __shared__ unsigned int s_diff[W];
    const long long b = bidx();
    if (b >= B) return;
    const long long base = (long long)blockIdx.x * TILE;
    const long long segoff = b * N;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t dst[KPT], pos[KPT];
    T val[KPT];
    unsigned int diff = 0;
    // N is a multiple of TILE here (N >= 2^22), so every tile is full
#pragma unroll
    for (int j = 0; j < KPT; ++j) {
        long long g = segoff + base + warp * 32 * KPT + j * 32 + lane;
        dst[j] = idx_new[g];
        diff += (dst[j] != idx_old[g]);
        val[j] = sorted[g];
    }
    rank_keys<uint32_t, THREADS, KPT>(dst, shift, pos, scratch);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) diff += __shfl_xor_sync(0xffffffffu, diff, o);
    if (lane == 0) s_diff[warp] = diff;
    if (threadIdx.x < kRadix) {
        const int d = threadIdx.x;
        uint32_t c = tile_cnt[d];
        uint32_t start = c ? atomicAdd(&cursor[b * kRadix + d], c) : 0u;
        goff[d] = ((long long)d << shift) + (long long)start - (long long)tile_off[d];
    }
#pragma unroll
    for (int j = 0; j < KPT; ++j) { sv[pos[j]] = val[j]; sd[pos[j]] = dst[j]; }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int t = 0;
        for (int i = 0; i < W; ++i) t += s_diff[i];
        if (t) atomicAdd(&changed[b], (unsigned long long)t);
    }
    for (int s = threadIdx.x; s < TILE; s += THREADS) {
        uint32_t d = sd[s];
        long long g = segoff + goff[(d >> shift) & (kRadix - 1)] + s;
        pv[g] = sv[s];
        pd[g] = d;
    }
}

template <typename T>
__global__ void __launch_bounds__(256) scatter_place_kernel(const T* __restrict__ pv, const uint32_t* __restrict__ pd,
                                                            T* __restrict__ x, long long N,
                                                            uint32_t* __restrict__ cursor, long long B) {
    const long long b = bidx();
    if (b >= B) return;
    if (blockIdx.x == 0) cursor[b * kRadix + threadIdx.x] = 0u;     // ready for the next iteration's bin pass
    const long long off = b * N;
    const long long g = off + ((long long)blockIdx.x * 256 + threadIdx.x) * 4;     // N is a multiple of 1024
    uint4 d = *reinterpret_cast<const uint4*>(pd + g);
    T v0 = pv[g], v1 = pv[g + 1], v2 = pv[g + 2], v3 = pv[g + 3];
    x[off + d.x] = v0; x[off + d.y] = v1; x[off + d.z] = v2; x[off + d.w] = v3;
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
template <typename T> struct SortCfg {
    static constexpr int NP = KeyT<T>::bits / kRadixBits;
    static constexpr int ctaMax = (sizeof(T) == 4) ? 16384 : 8192;     // largest segment sorted on chip
    static constexpr int SW_THREADS = 512;
    static constexpr int SW_KPT = (sizeof(T) == 4) ? 16 : 8;
    static constexpr int SW_TILE = SW_THREADS * SW_KPT;
};

template <typename T, int THREADS, int KPT> inline size_t cta_sort_smem() {
    return (size_t)THREADS * KPT * (sizeof(typename KeyT<T>::type) + 4) + RankScratch<THREADS>::words * 4;
}

template <typename T, int THREADS, int KPT> inline size_t scatter_bin_smem() {
    return (size_t)THREADS * KPT * (sizeof(T) + 4) + RankScratch<THREADS>::words * 4;
}
constexpr int kTwoLevelScatterLog = 22;     // segments of >= 2^22 values use the two-level rank scatter

template <typename T> inline long long sort_ntiles(long long N) { return (N + SortCfg<T>::SW_TILE - 1) / SortCfg<T>::SW_TILE; }

// workspace: key ping-pong (2), idx ping-pong (2), hist, tickets, status
template <typename T> inline size_t sort_ws_bytes(long long B, long long N) {
    if (N <= SortCfg<T>::ctaMax) return 256;
    typedef typename KeyT<T>::type KeyU;
    size_t s = 0;
    s += 2 * align_up((size_t)B * N * sizeof(KeyU), 256);
    s += 2 * align_up((size_t)B * N * 4, 256);
    size_t ctl = (size_t)B * SortCfg<T>::NP * kRadix * 4 + (size_t)B * SortCfg<T>::NP * 4 +
                 (size_t)B * SortCfg<T>::NP * sort_ntiles<T>(N) * kRadix * 4;
    s += align_up(ctl, 256);
    return s;
}

template <typename T> inline cudaError_t sort_set_attrs() {
    cudaError_t e;
    e = cudaFuncSetAttribute(cta_argsort_kernel<T, 1024, 16>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)cta_sort_smem<T, 1024, 16>());
    if (sizeof(T) == 8) e = cudaSuccess;   // the 16384 tile is not used for fp64 (too large); ignore
    cudaError_t e2 = cudaFuncSetAttribute(cta_argsort_kernel<T, 1024, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)cta_sort_smem<T, 1024, 8>());
    cudaError_t e3 = cudaFuncSetAttribute(cta_argsort_kernel<T, 512, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)cta_sort_smem<T, 512, 8>());
    constexpr int TH = SortCfg<T>::SW_THREADS, K = SortCfg<T>::SW_KPT;
    int sm = (int)cta_sort_smem<T, TH, K>();
    cudaError_t e4 = cudaFuncSetAttribute(onesweep_kernel<T, TH, K, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaError_t e5 = cudaFuncSetAttribute(onesweep_kernel<T, TH, K, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaError_t e6 = cudaFuncSetAttribute(onesweep_kernel<T, TH, K, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaError_t e7 = cudaFuncSetAttribute(scatter_bin_kernel<T, TH, K>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)scatter_bin_smem<T, TH, K>());
    // ask for the largest shared-memory carve-out, otherwise the driver sizes it for ONE resident CTA
    cudaFuncSetAttribute(onesweep_kernel<T, TH, K, true, false>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaFuncSetAttribute(onesweep_kernel<T, TH, K, false, false>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaFuncSetAttribute(onesweep_kernel<T, TH, K, false, true>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaFuncSetAttribute(scatter_bin_kernel<T, TH, K>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    (void)cudaGetLastError();
    if (e7 != cudaSuccess) return e7;
    if (e != cudaSuccess) return e;
    if (e2 != cudaSuccess) return e2;
    if (e3 != cudaSuccess) return e3;
    if (e4 != cudaSuccess) return e4;
    if (e5 != cudaSuccess) return e5;
    return e6;
}

// vals [B][N] -> idx_out [B][N] (u32), optionally the sorted values.  vals is not modified.
template <typename T>
inline cudaError_t seg_argsort(const T* vals, uint32_t* idx_out, T* sorted_out, long long B, long long N,
                               void* ws, cudaStream_t st) {
    typedef typename KeyT<T>::type KeyU;
    constexpr int NP = SortCfg<T>::NP;
    if (N <= SortCfg<T>::ctaMax) {
        if (N <= 1024)
            AGN_LAUNCH(K_SORT_CTA, st, (cta_argsort_kernel<T, 256, 4><<<(unsigned)B, 256, cta_sort_smem<T, 256, 4>(), st>>>(vals, idx_out, sorted_out, (int)N, N)));
        else if (N <= 4096)
            AGN_LAUNCH(K_SORT_CTA, st, (cta_argsort_kernel<T, 512, 8><<<(unsigned)B, 512, cta_sort_smem<T, 512, 8>(), st>>>(vals, idx_out, sorted_out, (int)N, N)));
        else if (N <= 8192)
            AGN_LAUNCH(K_SORT_CTA, st, (cta_argsort_kernel<T, 1024, 8><<<(unsigned)B, 1024, cta_sort_smem<T, 1024, 8>(), st>>>(vals, idx_out, sorted_out, (int)N, N)));
        else
            AGN_LAUNCH(K_SORT_CTA, st, (cta_argsort_kernel<T, 1024, 16><<<(unsigned)B, 1024, cta_sort_smem<T, 1024, 16>(), st>>>(vals, idx_out, sorted_out, (int)N, N)));
        return cudaGetLastError();
    }
    constexpr int TH = SortCfg<T>::SW_THREADS, K = SortCfg<T>::SW_KPT, TILE = SortCfg<T>::SW_TILE;
    unsigned char* w = (unsigned char*)ws;
    KeyU* k0 = (KeyU*)w; w += align_up((size_t)B * N * sizeof(KeyU), 256);
    KeyU* k1 = (KeyU*)w; w += align_up((size_t)B * N * sizeof(KeyU), 256);
    uint32_t* i0 = (uint32_t*)w; w += align_up((size_t)B * N * 4, 256);
    uint32_t* i1 = (uint32_t*)w; w += align_up((size_t)B * N * 4, 256);
    const long long ntiles = sort_ntiles<T>(N);
    uint32_t* hist = (uint32_t*)w;
    uint32_t* ticket = hist + (size_t)B * NP * kRadix;
    uint32_t* status = ticket + (size_t)B * NP;
    size_t ctl = (size_t)B * NP * kRadix * 4 + (size_t)B * NP * 4 + (size_t)B * NP * ntiles * kRadix * 4;
    cudaError_t e = cudaMemsetAsync(hist, 0, ctl, st);
    if (e != cudaSuccess) return e;
    const int chunk = 1 << 16;
    dim3 hg = bgrid((unsigned)((N + chunk - 1) / chunk), B);
    AGN_LAUNCH(K_SORT_HIST, st, (digit_hist_kernel<T, 512><<<hg, 512, 0, st>>>(vals, hist, N, N, chunk, B, nullptr)));
    const size_t sm = cta_sort_smem<T, TH, K>();
    dim3 grid = bgrid((unsigned)ntiles, B);
    for (int p = 0; p < NP; ++p) {
        SweepArgs<T> a;
        a.vals = vals;
        a.keys_in = (p & 1) ? k0 : k1;      // pass 0 writes k0/i0, pass 1 reads them and writes k1/i1, ...
        a.idx_in = (p & 1) ? i0 : i1;
        a.keys_out = (p & 1) ? k1 : k0;
        a.idx_out = (p == NP - 1) ? idx_out : ((p & 1) ? i1 : i0);
        a.sorted_out = sorted_out;
        a.N = N; a.seg_stride = N; a.shift = p * kRadixBits;
        a.hist = hist; a.pass = p; a.npass = NP;
        // per-pass control blocks: status laid out [pass][B][ntiles][256], tickets [pass][B]
        a.status = status + (size_t)p * B * ntiles * kRadix;
        a.ticket = ticket + (size_t)p * B;
        a.ntiles = (int)ntiles; a.B = B;
        if (p == 0) AGN_LAUNCH(K_SORT_SWEEP, st, (onesweep_kernel<T, TH, K, true, false><<<grid, TH, sm, st>>>(a)));
        else if (p == NP - 1) AGN_LAUNCH(K_SORT_SWEEP, st, (onesweep_kernel<T, TH, K, false, true><<<grid, TH, sm, st>>>(a)));
        else AGN_LAUNCH(K_SORT_SWEEP, st, (onesweep_kernel<T, TH, K, false, false><<<grid, TH, sm, st>>>(a)));
    }
    (void)TILE;
    return cudaGetLastError();
}

// L5 two-level (N >= 2^kTwoLevelScatterLog).  pv/pd: [B][N] scratch for the binned pairs; cursor: [B][256] u32,
// zero on entry (the place pass leaves it zero again).
template <typename T>
inline cudaError_t rank_scatter_two_level(const uint32_t* idx_new, const uint32_t* idx_old, const T* sorted, T* x,
                                          long long B, long long N, T* pv, uint32_t* pd, uint32_t* cursor,
                                          unsigned long long* changed, cudaStream_t st) {
    constexpr int TH = SortCfg<T>::SW_THREADS, K = SortCfg<T>::SW_KPT, TILE = SortCfg<T>::SW_TILE;
    const int shift = ilog2_u64((uint64_t)N) - kRadixBits;
    AGN_LAUNCH(K_SCATTER_BIN, st, (scatter_bin_kernel<T, TH, K><<<bgrid((unsigned)(N / TILE), B), TH, scatter_bin_smem<T, TH, K>(), st>>>(
        idx_new, idx_old, sorted, pv, pd, N, shift, cursor, changed, B)));
    AGN_LAUNCH(K_SCATTER_PLACE, st, (scatter_place_kernel<T><<<bgrid((unsigned)(N / 1024), B), 256, 0, st>>>(pv, pd, x, N, cursor, B)));
    return cudaGetLastError();
}

}  // namespace agn

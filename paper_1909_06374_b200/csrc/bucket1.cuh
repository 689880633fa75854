// bucket1.cuh -- L4 for long fp32 curves (2^18 <= N <= 2^26) as a ONE-LEVEL distribution sort: every key goes straight
// from x_adj to its equal-depth bucket (mean 8192 keys), and one CTA finishes a bucket in shared memory.
//
//   cdf_sample / cdf_table / bucket_bounds / bucket_base   as in bucket32.cuh (sampled piecewise-linear CDF of the keys)
//   part1_kernel         x_adj tile of 8192 keys -> (key, time index) pairs in the bucket slabs.  A tile counts its keys
//                        per bucket in shared memory (one 32-bit atomic per key), orders the tile by bucket in shared
//                        memory, reserves one range per non-empty (tile, bucket) with one global atomic and writes the
//                        runs out.  A light curve with a red PSD is smooth: the 8192 consecutive samples of a tile fall
//                        into ~15 % of the buckets, so a run is ~6-13 pairs (50-100 bytes).  For keys with no such
//                        locality (the i.i.d. ERDF draw that S1 sorts once per call) runs shrink to single pairs: still
//                        exact, slower; it is not the loop's case.
//   bucket1_sort_kernel  one CTA per bucket (slab of <= 12288 pairs, 96 KB of shared memory): counting sort into 8192
//                        interpolation slots (linear map of the key onto the bucket's key interval; 16-bit counters packed
//                        two per word), then the exact rank of every pair among its few slot mates by comparing the 64-bit
//                        (key, index) words; indices written at their ranks.
//
// HBM bytes per sample: 0.5 (sample) + 12 (partition: 4 in, 8 out) + 12 (finish: 8 in, 4 out) = 24.5 -- below the
// 28 of SURVEY 8(d)'s two-level model (which assumed a separate histogram read), against 40.5 for the two partition
// levels of bucket32.cuh.  Same exactness argument as there: the order inside a slab is arbitrary, the final order is
// defined by the (key, index) comparison alone, equal keys come out by ascending time index (O6 step 4).
// A slab that would overflow raises the curve's `overflow` flag and the LSD passes of sort32.cuh sort that curve.
#pragma once
#include "common.cuh"
#include "sort.cuh"
#include "bucket32.cuh"

namespace agn {

constexpr int kB1MeanLog = 13;                    // mean bucket population 2^13
constexpr int kB1Cap = 12288;                     // slab slots per bucket (1.5 x the mean: 5.6 sigma of the sampling noise)
constexpr int kB1SlotLog = 13;
constexpr int kB1Slots = 1 << kB1SlotLog;         // interpolation slots of the in-CTA sort
constexpr int kB1MaxBuckets = 8192;               // N <= 2^26
constexpr int kB1PartThreads = 512;        // 512 x 16 keys: 1.75 ms per C4 pass; 1024 x 8 at full occupancy measured the same (1.79)
constexpr int kB1PartEpt = 16;
constexpr int kB1Tile = kB1PartThreads * kB1PartEpt;      // 8192 keys
constexpr int kB1SortThreads = 1024;

inline bool bucket1_applicable(size_t elem_size, long long N) {
    return elem_size == 4 && N >= (1ll << 15) && N <= ((long long)kB1MaxBuckets << kB1MeanLog);
}
inline uint32_t bucket1_magic(uint32_t nb, int bl) {
    return (uint32_t)((((unsigned __int128)nb) << (32 + kB1SlotLog + 25 - bl)) / (bk_total_w(bl) << (32 - bl)));
}

struct Part1Args {
    const float* vals;          // [B][N]
    uint2* out;                 // slabs [B][nb][kB1Cap]
    uint32_t* cursor;           // [B][nb] zero on entry
    uint32_t* overflow;         // [B]
    const uint2* tab;           // [B][65536]
    uint32_t* loc;              // write-back mode (else null): [B][N] slab position (bucket * kB1Cap + offset) of the pair
    unsigned short* jrec;       //   at stage position s of the tile, and its sample number inside the tile, in STAGE order
    uint32_t N, nb, M;
    int bl;                     // log2 of the CDF table's bins per curve
    long long B;
};

// shared memory: stage uint2[kB1Tile] | cnt u32[nb] (populations -> first stage position -> slab offset of stage position 0)
inline size_t part1_smem(uint32_t nb) { return (size_t)kB1Tile * sizeof(uint2) + (size_t)nb * 4 + 64 * 4; }

// Bucket bookkeeping of a tile (zeroing, scan, reservation) is done 128 buckets ("chunk") at a time by one warp with
// 128-bit shared-memory accesses, lane l owning buckets 4 l .. 4 l + 3 of the chunk: conflict-free.  (A first version
// gave every thread 16 consecutive buckets: a 16-way bank conflict on every access, 87 wavefronts per 32 keys.)
constexpr int kB1Chunk = 128;
__global__ void __launch_bounds__(kB1PartThreads, 2) part1_kernel(Part1Args a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint2* stage = reinterpret_cast<uint2*>(smem_raw);
    uint32_t* cnt = reinterpret_cast<uint32_t*>(smem_raw + (size_t)kB1Tile * sizeof(uint2));
    uint4* cnt4 = reinterpret_cast<uint4*>(cnt);
    const long long b = bidx();
    if (b >= a.B) return;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    constexpr int NW = kB1PartThreads / 32;
    const uint2* tab = a.tab + ((size_t)b << a.bl);
    const uint32_t nb = a.nb;
    const uint32_t nv = nb >> 2;                          // uint4 words of counters (nb is a multiple of 32)
    const uint32_t nchunk = (nb + kB1Chunk - 1) / kB1Chunk;      // <= 64
    uint32_t* csum = cnt + nb;                            // [64] chunk totals
    for (uint32_t i = t; i < nv; i += kB1PartThreads) cnt4[i] = make_uint4(0u, 0u, 0u, 0u);
    const uint32_t tile0 = blockIdx.x * kB1Tile;
    const float* v = a.vals + (size_t)b * a.N + tile0;
    uint32_t key[kB1PartEpt];
#pragma unroll
    for (int j = 0; j < kB1PartEpt; ++j) key[j] = key_of(__ldcs(v + j * kB1PartThreads + t));
    __syncthreads();
    // bucket and arrival number inside the (tile, bucket) run
    uint32_t dr[kB1PartEpt];            // bucket << 14 | arrival number  (bucket < 2^13, arrival < 2^13)
    if (nb <= 1024u) {
        // few, wide buckets: neighbouring samples of a smooth series mostly share theirs -- one atomic for lane 0's group
#pragma unroll
        for (int j = 0; j < kB1PartEpt; ++j) {
            const uint32_t d = min(bs_of(key[j], tab, a.M, a.bl) >> kB1SlotLog, nb - 1u);
            const uint32_t dl = __shfl_sync(0xffffffffu, d, 0);
            const uint32_t same = __ballot_sync(0xffffffffu, d == dl);
            uint32_t r = 0;
            if (lane == 0) r = atomicAdd(&cnt[dl], (uint32_t)__popc(same));
            r = __shfl_sync(0xffffffffu, r, 0) + __popc(same & ((1u << lane) - 1u));
            if (d != dl) r = atomicAdd(&cnt[d], 1u);
            dr[j] = (d << 14) | r;
        }
    } else {
#pragma unroll
        for (int j = 0; j < kB1PartEpt; ++j) {
            const uint32_t d = min(bs_of(key[j], tab, a.M, a.bl) >> kB1SlotLog, nb - 1u);
            dr[j] = (d << 14) | atomicAdd(&cnt[d], 1u);
        }
    }
    __syncthreads();
    // chunk totals
    for (uint32_t c = warp; c < nchunk; c += NW) {
        const uint32_t vi = c * (kB1Chunk / 4) + lane;
        uint32_t s4 = 0;
        if (vi < nv) { const uint4 q = cnt4[vi]; s4 = q.x + q.y + q.z + q.w; }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s4 += __shfl_xor_sync(0xffffffffu, s4, o);
        if (lane == 0) csum[c] = s4;
    }
    __syncthreads();
    // every warp scans the (<= 64) chunk totals; then its own chunks: population -> first stage position | population << 16
    {
        const uint32_t c0 = lane < nchunk ? csum[lane] : 0u, c1 = lane + 32 < nchunk ? csum[lane + 32] : 0u;
        uint32_t i0 = c0, i1 = c1;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t m0 = __shfl_up_sync(0xffffffffu, i0, o), m1 = __shfl_up_sync(0xffffffffu, i1, o);
            if (lane >= o) { i0 += m0; i1 += m1; }
        }
        const uint32_t tot0 = __shfl_sync(0xffffffffu, i0, 31);
        const uint32_t e0 = i0 - c0, e1 = tot0 + i1 - c1;            // exclusive bases of chunks lane and lane + 32
        for (uint32_t c = warp; c < nchunk; c += NW) {
            const uint32_t base = c < 32 ? __shfl_sync(0xffffffffu, e0, c) : __shfl_sync(0xffffffffu, e1, c - 32);
            const uint32_t vi = c * (kB1Chunk / 4) + lane;
            uint4 q = make_uint4(0u, 0u, 0u, 0u);
            if (vi < nv) q = cnt4[vi];
            const uint32_t s4 = q.x + q.y + q.z + q.w;
            uint32_t inc = s4;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t m = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += m;
            }
            uint32_t run = base + inc - s4;
            uint4 w;
            w.x = run | (q.x << 16); run += q.x;
            w.y = run | (q.y << 16); run += q.y;
            w.z = run | (q.z << 16); run += q.z;
            w.w = run | (q.w << 16);
            if (vi < nv) cnt4[vi] = w;
        }
    }
    __syncthreads();
    // the tile ordered by bucket; an element carries its bucket and its position in the tile (the time index follows)
#pragma unroll
    for (int j = 0; j < kB1PartEpt; ++j) {
        const uint32_t d = dr[j] >> 14;
        stage[(cnt[d] & 0xffffu) + (dr[j] & 0x3fffu)] = make_uint2(key[j], (d << 13) | (uint32_t)(j * kB1PartThreads + t));
    }
    __syncthreads();
    // one global reservation per non-empty (tile, bucket); cnt[d] becomes (slab offset of the run) - (its stage position)
    {
        uint32_t* cur = a.cursor + (size_t)b * nb;
        for (uint32_t c = warp; c < nchunk; c += NW) {
            const uint32_t vi = c * (kB1Chunk / 4) + lane;
            if (vi < nv) {
                const uint4 q = cnt4[vi];
                const uint32_t qq[4] = {q.x, q.y, q.z, q.w};
                uint32_t o[4];
                bool over = false;
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const uint32_t n = qq[i] >> 16, s0 = qq[i] & 0xffffu;
                    uint32_t g = 0;
                    if (n) { g = atomicAdd(&cur[vi * 4 + i], n); over |= (g + n > (uint32_t)kB1Cap); }
                    o[i] = g - s0;
                }
                if (over) a.overflow[b] = 1u;
                cnt4[vi] = make_uint4(o[0], o[1], o[2], o[3]);
            }
        }
    }
    __syncthreads();
    uint2* out = a.out + (size_t)b * nb * kB1Cap;
    if (a.loc) {
        // write-back mode: remember, in stage order (coalesced), where every pair went and which sample it was
        uint32_t* lo = a.loc + (size_t)b * a.N + tile0;
        unsigned short* jo = a.jrec + (size_t)b * a.N + tile0;
#pragma unroll 4
        for (int s = t; s < kB1Tile; s += kB1PartThreads) {
            const uint2 e = stage[s];
            const uint32_t d = e.y >> 13;
            const uint32_t off = cnt[d] + (uint32_t)s;
            const uint32_t l = d * (uint32_t)kB1Cap + off;
            if (off < (uint32_t)kB1Cap) out[l] = make_uint2(e.x, tile0 + (e.y & 0x1fffu));
            lo[s] = l;
            jo[s] = (unsigned short)(e.y & 0x1fffu);
        }
        return;
    }
#pragma unroll 4
    for (int s = t; s < kB1Tile; s += kB1PartThreads) {
        const uint2 e = stage[s];
        const uint32_t d = e.y >> 13;
        const uint32_t off = cnt[d] + (uint32_t)s;
        if (off < (uint32_t)kB1Cap) out[(size_t)d * kB1Cap + off] = make_uint2(e.x, tile0 + (e.y & 0x1fffu));
    }
}

// ------------------------------------------------------------------------------------------------
// finish: one CTA per bucket
// ------------------------------------------------------------------------------------------------
struct B1Smem {
    unsigned long long pair[kB1Cap];      // (key << 32) | index, grouped by slot
    uint32_t cwpad[4];                    // cwpad[3] stays 0: the "end of slot -1" of the 16-bit view of cw
    uint32_t cw[kB1Slots / 2];            // two 16-bit counters per word: populations, then starts, then ends of the slots
    uint32_t wsum[kB1SortThreads / 32];
};
static_assert(sizeof(B1Smem) <= 115712, "two finish CTAs per SM");

// Write-back mode (the E13 loop, L4 + L5 in one go): the finish kernel does not only emit idx_new[r]; it also counts the
// rank changes against idx_old[r] and writes the VALUE that belongs to the pair, sorted[r] (L5: x[idx_new[r]] =
// sorted[r]), to the pair's own slab position in `valslab`.  gather_back_kernel then brings the values home along
// the records part1_kernel kept (loc, jrec), replacing the two-level rank scatter (bin + place).
struct B1Wb {
    const float* sorted;            // [B][N] the ERDF draw in rank order
    const uint32_t* idx_old;        // [B][N] permutation of the previous iteration
    unsigned long long* changed;    // [B]
    float* valslab;                 // [B][nb][kB1Cap]
    uint32_t* loc;                  // [B][N]
    unsigned short* jrec;           // [B][N]
    float* x_out;                   // [B][N]
};

// TAB: the slot of a key is its sub-bucket position on the sampled CDF (bs_of, the same table look-up part1_kernel
// did) instead of a linear map of the key onto the bucket's key interval.  For the few, wide buckets of a short curve
// (N < 2^20: a bucket is 1/4 .. 1/64 of the whole distribution, and float keys are logarithmic in the value) the
// linear map crowds most pairs into a few slots -- the rank among slot mates costs the square of a slot's population:
// 2.3 ms instead of 0.2 per 2^25 samples at N = 2^15 with C4's ERDF.  The table of such a curve is small (2^11 ..
// 2^15 bins) and stays in L1 / L2.
struct B1Tab {
    const uint2* tab;               // [B][2^bl]
    uint32_t M;
    int bl;
};

template <bool WB, bool TAB>
__global__ void __launch_bounds__(kB1SortThreads, 2) bucket1_sort_kernel(const uint2* __restrict__ slabs,
                                                                         const uint32_t* __restrict__ cursor,
                                                                         const uint32_t* __restrict__ base,
                                                                         const uint32_t* __restrict__ overflow,
                                                                         const uint32_t* __restrict__ klos,
                                                                         uint32_t* __restrict__ idx_out,
                                                                         float* __restrict__ sorted_out, uint32_t N,
                                                                         uint32_t nb, long long B, B1Wb wb, B1Tab tb) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    B1Smem& sm = *reinterpret_cast<B1Smem*>(smem_raw);
    const long long b = bidx();
    if (b >= B) return;
    if (overflow[b]) return;                       // this curve is sorted by the LSD passes instead
    const uint32_t bk = blockIdx.x;
    const uint32_t n = cursor[(size_t)b * nb + bk];          // <= kB1Cap (no overflow)
    if (n == 0) return;
    const uint32_t r0 = base[(size_t)b * nb + bk];
    const uint2* sl = slabs + ((size_t)b * nb + bk) * kB1Cap;
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
    const float scale = (float)kB1Slots / ((float)width + 1.0f);
    const uint2* ctab = TAB ? tb.tab + ((size_t)b << tb.bl) : nullptr;
    const uint32_t bs0 = bk << kB1SlotLog;
    auto slot_of = [&](uint32_t key) -> uint32_t {
        if (TAB) {
            const uint32_t bs = bs_of(key, ctab, tb.M, tb.bl);          // monotone in the key; equal keys, equal slots
            return bs > bs0 ? min(bs - bs0, (uint32_t)(kB1Slots - 1)) : 0u;
        }
        const uint32_t d = key > klo ? key - klo : 0u;
        return min((uint32_t)(__uint2float_rz(d) * scale), (uint32_t)(kB1Slots - 1));
    };
    constexpr int WPT = kB1Slots / 2 / kB1SortThreads;      // counter words per thread in the scan (4 = one uint4)
    static_assert(WPT == 4, "one uint4 of packed counters per thread");
    reinterpret_cast<uint4*>(sm.cw)[t] = make_uint4(0u, 0u, 0u, 0u);
    if (t == 0) sm.cwpad[3] = 0u;
    const unsigned short* send = reinterpret_cast<const unsigned short*>(sm.cw);       // after step 3: send[s] = end of slot s
    __syncthreads();
    // 1. slot populations (the slab stays in L2 for step 3).  (Two pairs per 128-bit load measured slower: 1.85 vs 1.69 ms.)
#pragma unroll 4
    for (uint32_t e = t; e < n; e += kB1SortThreads) {
        const uint32_t s = slot_of(__ldcg(&sl[e].x));
        atomicAdd(&sm.cw[s >> 1], 1u << ((s & 1u) << 4));
    }
    __syncthreads();
    // 2. exclusive scan of the slot populations (8 consecutive slots per thread)
    {
        const uint4 w4 = reinterpret_cast<const uint4*>(sm.cw)[t];
        const uint32_t w[4] = {w4.x, w4.y, w4.z, w4.w};
        uint32_t sum = 0;
#pragma unroll
        for (int i = 0; i < 4; ++i) sum += (w[i] & 0xffffu) + (w[i] >> 16);
        uint32_t inc = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t m = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += m;
        }
        if (lane == 31) sm.wsum[warp] = inc;
        __syncthreads();
        if (warp == 0) {
            // exclusive scan of the 32 warp totals
            const uint32_t wt = sm.wsum[lane];
            uint32_t wi = wt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t m = __shfl_up_sync(0xffffffffu, wi, o);
                if (lane >= o) wi += m;
            }
            sm.wsum[lane] = wi - wt;
        }
        __syncthreads();
        uint32_t run = inc - sum + sm.wsum[warp];
        uint32_t o[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const uint32_t lo = run; run += w[i] & 0xffffu;
            const uint32_t hi = run; run += w[i] >> 16;
            o[i] = lo | (hi << 16);
        }
        reinterpret_cast<uint4*>(sm.cw)[t] = make_uint4(o[0], o[1], o[2], o[3]);
    }
    __syncthreads();
    // 3. every pair into its slot's range (any order); the counter of slot s ends as the END of slot s
#pragma unroll 4
    for (uint32_t e = t; e < n; e += kB1SortThreads) {
        const uint2 kv = __ldcs(sl + e);
        const uint32_t s = slot_of(kv.x);
        const uint32_t sh = (s & 1u) << 4;
        const uint32_t q = (atomicAdd(&sm.cw[s >> 1], 1u << sh) >> sh) & 0xffffu;
        sm.pair[q] = ((unsigned long long)kv.x << 32) | kv.y;
        if (WB) reinterpret_cast<uint32_t*>(wb.valslab)[((size_t)b * nb + bk) * kB1Cap + e] = q;   // read back in step 4C
    }
    __syncthreads();
    // 4. exact rank of every pair among its slot mates (they are contiguous; the 64-bit (key, index) words are all
    //    distinct), one pair per thread at a time, and the index goes to that rank
    uint32_t* io = idx_out + (size_t)b * N + r0;
    if (WB) {
        // L4 + L5 for this bucket.  Nothing below touches global memory at a scattered address: the ranks of a bucket
        // are contiguous (r0 .. r0 + n), so idx_new, idx_old and sorted[] are accessed in RANK order (coalesced), the
        // value slab in SLAB order (coalesced), and the two orders meet in shared memory.  An index needs 26 bits
        // (N <= 2^26): the 6 spare bits of the low word at position r say where the pair of rank r sits, as a signed
        // offset inside the slot (slots of <= 31 pairs; a larger slot -- massive ties -- is marked and takes a slow,
        // still exact, path).
        constexpr uint32_t IDXM = 0x03ffffffu;
        constexpr unsigned long long CMPM = 0xffffffff03ffffffull;
        constexpr uint32_t BIG = 0x80000000u;                           // offset field = -32: "this slot is big"
        uint32_t* plo = reinterpret_cast<uint32_t*>(sm.pair);           // little endian: word 2 q = index, 2 q + 1 = key
        const uint32_t* iold = wb.idx_old + (size_t)b * N + r0;
        const float* srt = wb.sorted + (size_t)b * N + r0;
        uint32_t* vs = reinterpret_cast<uint32_t*>(wb.valslab) + ((size_t)b * nb + bk) * kB1Cap;
        uint32_t diff = 0;
        // (sorted[] and idx_old of this bucket's ranks are first touched in 4B: have them in L2 by then)
        if ((uint32_t)t * 32u < n) {
            asm volatile("prefetch.global.L2 [%0];" ::"l"(srt + t * 32));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(iold + t * 32));
        }
        // 4A. rank of every pair inside its slot; position r learns where its pair is
#pragma unroll 2
        for (uint32_t q = t; q < n; q += kB1SortThreads) {
            const unsigned long long v = sm.pair[q] & CMPM;             // (another pair's offset may already sit here)
            const int s = (int)slot_of((uint32_t)(v >> 32));
            const uint32_t a = send[s - 1], z = send[s];
            const uint32_t k = z - a;
            if (k == 1u) continue;
            uint32_t c;
            if (k == 2u) {
                c = ((sm.pair[q == a ? a + 1u : a] & CMPM) < v);
            } else {
                c = 0;
                uint32_t h = a;
                for (; h + 1u < z; h += 2u) {
                    const unsigned long long m0 = sm.pair[h] & CMPM, m1 = sm.pair[h + 1u] & CMPM;
                    c += (m0 < v);
                    c += (m1 < v);
                }
                if (h < z) c += ((sm.pair[h] & CMPM) < v);
            }
            const uint32_t r = a + c;
            if (k <= 31u) {
                plo[2 * r] = (plo[2 * r] & IDXM) | ((q - r) << 26);     // the index bits of position r never change
            } else {
                plo[2 * q] = (uint32_t)v | BIG;
                io[r] = (uint32_t)v;
                diff += (__ldg(iold + r) != (uint32_t)v);
            }
        }
        __syncthreads();
        // 4B. rank order: the pair of rank p gives its index and takes sorted[r0 + p] (into the key half of its word:
        //     keys are not needed any more)
#pragma unroll 2
        for (uint32_t p = t; p < n; p += kB1SortThreads) {
            const uint32_t lo = plo[2 * p];
            if ((lo & 0xfc000000u) == BIG) continue;                    // big slot: done in 4A / 4C
            const uint32_t h = p + (uint32_t)((int32_t)lo >> 26);
            const uint32_t idx = plo[2 * h] & IDXM;
            io[p] = idx;
            diff += (__ldcs(iold + p) != idx);
            plo[2 * h + 1] = __float_as_uint(__ldcs(srt + p));
        }
        __syncthreads();
        // 4C. slab order: the value of the pair that came from slab position e goes back to position e
        for (uint32_t e = t; e < n; e += kB1SortThreads) {
            const uint32_t q = vs[e];
            const uint32_t lo = plo[2 * q], hi = plo[2 * q + 1];
            uint32_t val = hi;
            if ((lo & 0xfc000000u) == BIG) {
                const int s = (int)slot_of(hi);
                const uint32_t a = send[s - 1], z = send[s];
                const unsigned long long v = ((unsigned long long)hi << 32) | (lo & IDXM);
                uint32_t r = a;
                for (uint32_t h = a; h < z; ++h) r += ((sm.pair[h] & CMPM) < v);
                val = __float_as_uint(__ldg(srt + r));
            }
            vs[e] = val;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) diff += __shfl_xor_sync(0xffffffffu, diff, o);
        if (lane == 0 && diff) atomicAdd(&wb.changed[b], (unsigned long long)diff);
        return;
    }
    float* so = sorted_out ? sorted_out + (size_t)b * N + r0 : nullptr;
#pragma unroll 2
    for (uint32_t q = t; q < n; q += kB1SortThreads) {
        const unsigned long long v = sm.pair[q];
        const uint32_t key = (uint32_t)(v >> 32);
        const int s = (int)slot_of(key);
        const uint32_t a = send[s - 1], z = send[s];
        uint32_t r = q;
        if (z - a > 1u) {
            r = a;
            for (uint32_t h = a; h < z; ++h) r += (sm.pair[h] < v);
        }
        io[r] = (uint32_t)v;
        if (so) so[r] = val_of(key);
    }
}

// L5 of the write-back mode: x[tile0 + jrec[s]] = valslab[loc[s]] for the stage positions s of one partition tile.
// loc / jrec are read in stage order (coalesced), the slab values along the runs part1_kernel wrote (consecutive s of
// a run are consecutive slab positions), and the tile is put into time order in shared memory before it is stored.
constexpr int kB1GatherThreads = 512;
__global__ void __launch_bounds__(kB1GatherThreads, 4) gather_back_kernel(const uint32_t* __restrict__ loc,
                                                                          const unsigned short* __restrict__ jrec,
                                                                          const float* __restrict__ valslab,
                                                                          const uint32_t* __restrict__ overflow,
                                                                          float* __restrict__ x, uint32_t N, uint32_t nb,
                                                                          long long B) {
    __shared__ __align__(16) float xs[kB1Tile];
    const long long b = bidx();
    if (b >= B) return;
    if (overflow[b]) return;                       // this curve takes the LSD sort and the plain rank scatter
    const int t = threadIdx.x;
    const size_t g0 = (size_t)b * N + (size_t)blockIdx.x * kB1Tile;
    const float* vs = valslab + (size_t)b * nb * kB1Cap;
    const uint4* l4 = reinterpret_cast<const uint4*>(loc + g0);
    const uint2* j4 = reinterpret_cast<const uint2*>(jrec + g0);
    constexpr int NV = kB1Tile / 4 / kB1GatherThreads;      // 4 vectors of 4 records per thread
    uint4 l[NV];
    uint2 j[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) { l[k] = __ldcs(l4 + k * kB1GatherThreads + t); j[k] = __ldcs(j4 + k * kB1GatherThreads + t); }
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        const float v0 = __ldcs(vs + l[k].x), v1 = __ldcs(vs + l[k].y), v2 = __ldcs(vs + l[k].z), v3 = __ldcs(vs + l[k].w);
        xs[j[k].x & 0xffffu] = v0; xs[j[k].x >> 16] = v1; xs[j[k].y & 0xffffu] = v2; xs[j[k].y >> 16] = v3;
    }
    __syncthreads();
    float4* xo = reinterpret_cast<float4*>(x + g0);
#pragma unroll
    for (int k = 0; k < NV; ++k) __stcs(xo + k * kB1GatherThreads + t, reinterpret_cast<const float4*>(xs)[k * kB1GatherThreads + t]);
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
inline cudaError_t bucket1_set_attrs() {
    cudaFuncSetAttribute(part1_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaFuncSetAttribute(bucket1_sort_kernel<false, false>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaFuncSetAttribute(bucket1_sort_kernel<false, true>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaFuncSetAttribute(bucket1_sort_kernel<true, false>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaError_t e = cudaFuncSetAttribute(part1_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)part1_smem(kB1MaxBuckets));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bucket1_sort_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(B1Smem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bucket1_sort_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(B1Smem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(bucket1_sort_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(B1Smem));
    return e;
}

// pair scratch (uint2 units): slabs [B][nb][kB1Cap]
inline size_t bucket1_pair_elems(long long B, long long N) { return (size_t)B * (size_t)(N >> kB1MeanLog) * kB1Cap; }

// The write-back mode pays where the plain rank scatter needs two levels (N >= 2^22: bin + place, 2.5 ms per C4
// iteration, against 0.94 for gather_back + 1.05 more in the finish kernel + 0.23 in part1: C4 470 -> 464 ms per step);
// for shorter curves the one-kernel scatter inside an L2-resident window is cheaper (C3: 750 vs 835 ms per step).
inline bool bucket1_wb_applicable(size_t elem_size, long long N) { return bucket1_applicable(elem_size, N) && N >= (1ll << 22); }

// write-back scratch of the E13 loop: loc u32 [B][N] | jrec u16 [B][N] | valslab f32 [B][nb][kB1Cap]
inline size_t bucket1_wb_bytes(long long B, long long N) {
    return align_up((size_t)B * N * 4, 256) + align_up((size_t)B * N * 2, 256) + align_up(bucket1_pair_elems(B, N) * 4, 256);
}
inline void bucket1_wb_carve(void* p, long long B, long long N, B1Wb* wb) {
    unsigned char* w = (unsigned char*)p;
    wb->loc = (uint32_t*)w; w += align_up((size_t)B * N * 4, 256);
    wb->jrec = (unsigned short*)w; w += align_up((size_t)B * N * 2, 256);
    wb->valslab = (float*)w;
}


// control words: hist [B][65536] u32 | cursor [B][nb] | overflow [B] (zeroed per call) | tab [B][65536] uint2 |
//                base [B][nb] | klo [B][nb+1]
inline size_t bucket1_zero_bytes(long long B, long long N) {
    const size_t nb = (size_t)(N >> kB1MeanLog);
    return (((size_t)B * 4) << bk_binlog(N)) + (size_t)B * nb * 4 + (size_t)B * 4;
}
inline size_t bucket1_ctl_bytes(long long B, long long N) {
    const size_t nb = (size_t)(N >> kB1MeanLog);
    return align_up(bucket1_zero_bytes(B, N), 256) + align_up(((size_t)B * 8) << bk_binlog(N), 256) + align_up((size_t)B * nb * 4, 256) +
           align_up((size_t)B * (nb + 1) * 4, 256);
}

// vals [B][N] -> idx_out (and optionally the sorted values) for the curves whose buckets all fit; *overflow_out points
// at the per-curve flags (1 = not sorted here).  pairs: bucket1_pair_elems(B, N) (key, index) pairs of scratch.
// wb != null: write-back mode (see B1Wb): also x_out[idx_out[r]] = sorted[r] and the rank-change count, for the curves
// whose buckets all fit.
inline cudaError_t bucket1_sort(const float* vals, uint32_t* idx_out, float* sorted_out, long long B, long long N,
                                uint2* pairs, void* ctl, const uint32_t** overflow_out, cudaStream_t st,
                                const B1Wb* wb = nullptr) {
    const uint32_t nb = (uint32_t)(N >> kB1MeanLog);
    unsigned char* w = (unsigned char*)ctl;
    uint32_t* hist = (uint32_t*)w;
    const int bl = bk_binlog(N);
    uint32_t* cursor = hist + ((size_t)B << bl);
    uint32_t* overflow = cursor + (size_t)B * nb;
    const size_t zero_bytes = bucket1_zero_bytes(B, N);
    w += align_up(zero_bytes, 256);
    uint2* tab = (uint2*)w; w += align_up(((size_t)B * 8) << bl, 256);
    uint32_t* base = (uint32_t*)w; w += align_up((size_t)B * nb * 4, 256);
    uint32_t* klo = (uint32_t*)w;
    cudaError_t e = cudaMemsetAsync(hist, 0, zero_bytes, st);
    if (e != cudaSuccess) return e;
    const uint32_t nsamp = (uint32_t)(N >> kBkSampleLog);
    const uint32_t M = bucket1_magic(nb, bl);
    const unsigned chunks = cdf_chunks(bl);
    AGN_LAUNCH(K_SORT_CDF, st, (cdf_sample_kernel<<<bgrid(cdf_sample_grid(nsamp), B), 256, 0, st>>>(vals, hist, (uint32_t)N, B, bl)));
    AGN_LAUNCH(K_SORT_CDF, st, (cdf_table_kernel<<<(unsigned)(B * chunks), 1024, 0, st>>>(hist, tab, 24 - (ilog2_u64((uint64_t)N) - kBkSampleLog), bl, chunks)));
    AGN_LAUNCH(K_SORT_CDF, st, (bucket_bounds_kernel<<<bgrid((nb + 256) / 256, B), 256, 0, st>>>(tab, klo, nb, M, kB1SlotLog, B, bl)));
    Part1Args a;
    a.vals = vals; a.out = pairs; a.cursor = cursor; a.overflow = overflow; a.tab = tab;
    a.N = (uint32_t)N; a.nb = nb; a.M = M; a.B = B; a.bl = bl;
    a.loc = wb ? wb->loc : nullptr; a.jrec = wb ? wb->jrec : nullptr;
    AGN_LAUNCH(wb ? K_SORT_PART_ONE_WB : K_SORT_PART_ONE, st, (part1_kernel<<<bgrid((unsigned)(N / kB1Tile), B), kB1PartThreads, part1_smem(nb), st>>>(a)));
    const uint32_t bchunks = nb >= 1024 ? nb / 1024 : 1u;
    AGN_LAUNCH(K_SORT_CDF, st, (bucket_base_kernel<<<(unsigned)(B * bchunks), 1024, 0, st>>>(cursor, base, nb, bchunks, (uint32_t)kB1Cap)));
    if (wb) {
        AGN_LAUNCH(K_SORT_BUCKET_WB, st, (bucket1_sort_kernel<true, false><<<bgrid(nb, B), kB1SortThreads, sizeof(B1Smem), st>>>(
            pairs, cursor, base, overflow, klo, idx_out, sorted_out, (uint32_t)N, nb, B, *wb, B1Tab())));
        AGN_LAUNCH(K_GATHER_BACK, st, (gather_back_kernel<<<bgrid((unsigned)(N / kB1Tile), B), kB1GatherThreads, 0, st>>>(
            wb->loc, wb->jrec, wb->valslab, overflow, wb->x_out, (uint32_t)N, nb, B)));
    } else {
        B1Tab tb;
        tb.tab = tab; tb.M = M; tb.bl = bl;
        if (N < (1ll << 20))
            AGN_LAUNCH(K_SORT_BUCKET, st, (bucket1_sort_kernel<false, true><<<bgrid(nb, B), kB1SortThreads, sizeof(B1Smem), st>>>(
                pairs, cursor, base, overflow, klo, idx_out, sorted_out, (uint32_t)N, nb, B, B1Wb(), tb)));
        else
            AGN_LAUNCH(K_SORT_BUCKET, st, (bucket1_sort_kernel<false, false><<<bgrid(nb, B), kB1SortThreads, sizeof(B1Smem), st>>>(
                pairs, cursor, base, overflow, klo, idx_out, sorted_out, (uint32_t)N, nb, B, B1Wb(), tb)));
    }
    *overflow_out = overflow;
    return cudaGetLastError();
}

}  // namespace agn

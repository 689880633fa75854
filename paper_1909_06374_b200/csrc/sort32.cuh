// sort32.cuh -- the fp32 hot-path versions of L4 (segmented stable LSD radix argsort, N > 2^14) and L5
// (two-level rank scatter + change count).  Same algorithms as sort.cuh, re-engineered for throughput on B200:
//   * (key, index) travel as one 8-byte pair (array of uint2): one 64-bit load/store and one shared-memory
//     access per element instead of two, and digit runs in HBM are twice as long;
//   * tiles of 4096 keys, 256 threads, <= 64 registers: four resident CTAs per SM overlap the load, rank,
//     look-back and write phases of different tiles; every thread owns one digit in the scan / look-back phase;
//   * ranking without MATCH.ANY (see rank_keys in sort.cuh), look-back inspects kLookBatch predecessors per
//     round trip, all in-segment indices are 32-bit.
// Segments are power-of-two lengths >= 2^15, so every tile is full.
#pragma once
#include "common.cuh"
#include "sort.cuh"

namespace agn {

constexpr int kS32Threads = 256;
constexpr int kS32Kpt = 16;
constexpr int kS32Tile = kS32Threads * kS32Kpt;      // 4096
constexpr int kS32Warps = kS32Threads / 32;

struct S32Smem {
    uint2 stage[kS32Tile];
    uint2 cm[kS32Warps * kRadix];       // {lane mask of the current round, running count} per (warp, digit)
    uint32_t tile_off[kRadix];
    uint32_t goff[kRadix];
    uint32_t wsum[kS32Warps];
    uint32_t tile;
    uint32_t diff;
};

// ranks the 16 warp-striped keys of every thread by `digit`; returns local positions and leaves
// sm.tile_off[d] (exclusive digit offsets in the tile); returns this thread's digit count (thread == digit)
__device__ __forceinline__ uint32_t s32_rank(const uint32_t (&dig)[kS32Kpt], uint32_t (&pos)[kS32Kpt], S32Smem& sm) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
    for (int i = 0; i < kS32Warps; ++i) sm.cm[i * kRadix + threadIdx.x] = make_uint2(0u, 0u);
    __syncthreads();
    const uint32_t lt = lanemask_lt(), bit = 1u << lane;
    uint2* cw = sm.cm + warp * kRadix;
    uint32_t r[kS32Kpt];
#pragma unroll
    for (int j = 0; j < kS32Kpt; ++j) {
        const uint32_t d = dig[j];
        atomicOr(&cw[d].x, bit);
        __syncwarp();
        const uint2 mc = cw[d];
        r[j] = mc.y + __popc(mc.x & lt);
        __syncwarp();
        if ((mc.x & lt) == 0u) cw[d] = make_uint2(0u, mc.y + __popc(mc.x));
        __syncwarp();
    }
    __syncthreads();
    // thread == digit: exclusive scan over the warps, then over the digits
    uint32_t run = 0;
#pragma unroll
    for (int w = 0; w < kS32Warps; ++w) {
        const uint32_t t = sm.cm[w * kRadix + threadIdx.x].y;
        sm.cm[w * kRadix + threadIdx.x].y = run;
        run += t;
    }
    uint32_t inc = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t n = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += n;
    }
    if (lane == 31) sm.wsum[warp] = inc;
    __syncthreads();
    uint32_t add = 0;
#pragma unroll
    for (int w = 0; w < kS32Warps; ++w) add += (w < warp) ? sm.wsum[w] : 0u;
    sm.tile_off[threadIdx.x] = inc - run + add;
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kS32Kpt; ++j) pos[j] = sm.tile_off[dig[j]] + cw[dig[j]].y + r[j];
    return run;
}

struct Sweep32Args {
    const float* vals;          // FIRST: raw values [B][N]
    const uint2* in;            // later passes: (key, idx) pairs
    uint2* out;                 // FIRST/MIDDLE
    uint32_t* idx_out;          // LAST
    float* sorted_out;          // LAST, may be NULL
    uint32_t N;
    int shift;
    const uint32_t* dstart;     // [B][NP][256] exclusive digit starts (scanned histogram)
    int pass, npass;
    uint32_t* status;           // [B][ntiles][256] zero-initialised
    uint32_t* ticket;           // [B] zero-initialised
    uint32_t ntiles;
    long long B;
};

// exclusive scan of every 256-bin histogram, in place (one warp-scan CTA per histogram)
__global__ void __launch_bounds__(kRadix) digit_scan_kernel(uint32_t* __restrict__ hist) {
    __shared__ uint32_t ws[8];
    uint32_t* h = hist + (size_t)blockIdx.x * kRadix;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t c = h[threadIdx.x];
    uint32_t inc = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t n = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += n;
    }
    if (lane == 31) ws[warp] = inc;
    __syncthreads();
    uint32_t add = 0;
    for (int w = 0; w < warp; ++w) add += ws[w];
    h[threadIdx.x] = inc - c + add;
}

// KIND 0: first pass (raw values in, pairs out); 1: middle (pairs in, pairs out); 2: last (pairs in, indices out)
template <int KIND>
__global__ void __launch_bounds__(kS32Threads, 4) sweep32_kernel(Sweep32Args a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    S32Smem& sm = *reinterpret_cast<S32Smem*>(smem_raw);
    const long long b = bidx();
    if (b >= a.B) return;
    if (threadIdx.x == 0) sm.tile = atomicAdd(&a.ticket[b], 1u);
    __syncthreads();
    const uint32_t tile = sm.tile;
    const uint32_t base = tile * kS32Tile;
    const size_t seg = (size_t)b * a.N;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint2 kv[kS32Kpt];
    uint32_t dig[kS32Kpt], pos[kS32Kpt];
    const uint32_t e0 = base + warp * (32 * kS32Kpt) + lane;
    if (KIND == 0) {
        const float* v = a.vals + seg + e0;
#pragma unroll
        for (int j = 0; j < kS32Kpt; ++j) kv[j] = make_uint2(key_of(__ldcs(v + j * 32)), e0 + j * 32);
    } else {
        const uint2* v = a.in + seg + e0;
#pragma unroll
        for (int j = 0; j < kS32Kpt; ++j) kv[j] = __ldcs(v + j * 32);
    }
#pragma unroll
    for (int j = 0; j < kS32Kpt; ++j) dig[j] = (kv[j].x >> a.shift) & (kRadix - 1);
    const uint32_t agg = s32_rank(dig, pos, sm);
    // thread == digit: publish the tile aggregate, look back over earlier tiles of the segment
    {
        const int d = threadIdx.x;
        volatile uint32_t* st = a.status + (size_t)b * a.ntiles * kRadix + d;
        uint32_t excl = 0;
        if (tile == 0) {
            st[0] = kFlagInc | agg;
        } else {
            st[(size_t)tile * kRadix] = kFlagAgg | agg;
            int t = (int)tile - 1;
            bool done = false;
            while (!done) {
                uint32_t sv[kLookBatch];
#pragma unroll
                for (int i = 0; i < kLookBatch; ++i) sv[i] = (t - i >= 0) ? st[(size_t)(t - i) * kRadix] : (2u << 30);
                int used = kLookBatch;
#pragma unroll
                for (int i = 0; i < kLookBatch; ++i) {
                    if (!done && used == kLookBatch) {
                        const uint32_t f = sv[i] & kFlagMask;
                        if (f == 0) used = i;
                        else {
                            excl += sv[i] & ~kFlagMask;
                            if (f == kFlagInc) done = true;
                        }
                    }
                }
                t -= used;
            }
            st[(size_t)tile * kRadix] = kFlagInc | (excl + agg);
        }
        sm.goff[d] = a.dstart[((size_t)b * a.npass + a.pass) * kRadix + d] + excl - sm.tile_off[d];
    }
#pragma unroll
    for (int j = 0; j < kS32Kpt; ++j) sm.stage[pos[j]] = kv[j];
    __syncthreads();
#pragma unroll 4
    for (int s = threadIdx.x; s < kS32Tile; s += kS32Threads) {
        const uint2 p = sm.stage[s];
        const uint32_t g = sm.goff[(p.x >> a.shift) & (kRadix - 1)] + (uint32_t)s;
        if (KIND == 2) {
            a.idx_out[seg + g] = p.y;
            if (a.sorted_out) a.sorted_out[seg + g] = val_of(p.x);
        } else {
            a.out[seg + g] = p;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// L5 two-level: bin (value, dst) pairs by the top 8 bits of dst, then place
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kS32Threads, 4) scatter_bin32_kernel(const uint32_t* __restrict__ idx_new,
                                                                       const uint32_t* __restrict__ idx_old,
                                                                       const float* __restrict__ sorted,
                                                                       uint2* __restrict__ pairs, uint32_t N, int shift,
                                                                       uint32_t* __restrict__ cursor,
                                                                       unsigned long long* __restrict__ changed,
                                                                       long long B) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    S32Smem& sm = *reinterpret_cast<S32Smem*>(smem_raw);
    const long long b = bidx();
    if (b >= B) return;
    const uint32_t base = blockIdx.x * kS32Tile;
    const size_t seg = (size_t)b * N;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint2 kv[kS32Kpt];                  // x = value bits, y = dst
    uint32_t dig[kS32Kpt], pos[kS32Kpt];
    const size_t e0 = seg + base + warp * (32 * kS32Kpt) + lane;
    unsigned int diff = 0;
    if (threadIdx.x == 0) sm.diff = 0u;
#pragma unroll
    for (int j = 0; j < kS32Kpt; ++j) {
        const uint32_t dst = __ldcs(idx_new + e0 + j * 32);
        diff += (dst != __ldcs(idx_old + e0 + j * 32));
        kv[j] = make_uint2(__float_as_uint(__ldcs(sorted + e0 + j * 32)), dst);
        dig[j] = (dst >> shift) & (kRadix - 1);
    }
    const uint32_t cnt = s32_rank(dig, pos, sm);
    {
        const int d = threadIdx.x;
        const uint32_t start = cnt ? atomicAdd(&cursor[b * kRadix + d], cnt) : 0u;
        sm.goff[d] = ((uint32_t)d << shift) + start - sm.tile_off[d];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) diff += __shfl_xor_sync(0xffffffffu, diff, o);
    if (lane == 0 && diff) atomicAdd(&sm.diff, diff);        // sm.diff was zeroed before the barriers of s32_rank
#pragma unroll
    for (int j = 0; j < kS32Kpt; ++j) sm.stage[pos[j]] = kv[j];
    __syncthreads();
    if (threadIdx.x == 0 && sm.diff) atomicAdd(&changed[b], (unsigned long long)sm.diff);
#pragma unroll 4
    for (int s = threadIdx.x; s < kS32Tile; s += kS32Threads) {
        const uint2 p = sm.stage[s];
        pairs[seg + sm.goff[(p.y >> shift) & (kRadix - 1)] + (uint32_t)s] = p;
    }
}

__global__ void __launch_bounds__(256) scatter_place32_kernel(const uint4* __restrict__ pairs2, float* __restrict__ x,
                                                              uint32_t N, uint32_t* __restrict__ cursor, long long B) {
    const long long b = bidx();
    if (b >= B) return;
    if (blockIdx.x == 0) cursor[b * kRadix + threadIdx.x] = 0u;      // ready for the next iteration's bin pass
    const size_t seg = (size_t)b * N;
    float* xs = x + seg;
    const uint4* p = pairs2 + (seg >> 1) + (size_t)blockIdx.x * 1024 + threadIdx.x;     // 2 pairs per uint4
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint4 q = __ldcs(p + i * 256);
        xs[q.y] = __uint_as_float(q.x);
        xs[q.w] = __uint_as_float(q.z);
    }
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
inline cudaError_t sort32_set_attrs() {
    const int sm = (int)sizeof(S32Smem);
    cudaError_t e = cudaFuncSetAttribute(sweep32_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sweep32_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(sweep32_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(scatter_bin32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    cudaFuncSetAttribute(sweep32_kernel<0>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaFuncSetAttribute(sweep32_kernel<1>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaFuncSetAttribute(sweep32_kernel<2>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaFuncSetAttribute(scatter_bin32_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    return e;
}

inline bool sort32_applicable(size_t elem_size, long long N) {
    return elem_size == 4 && N > SortCfg<float>::ctaMax && N <= (1ll << 27);
}

// workspace (bytes): two pair buffers + control (hist, tickets, status)
inline size_t sort32_ws_bytes(long long B, long long N) {
    const size_t ntiles = (size_t)(N / kS32Tile);
    size_t s = 2 * align_up((size_t)B * N * sizeof(uint2), 256);
    s += align_up((size_t)B * 4 * kRadix * 4 + (size_t)B * 4 * 4 + (size_t)B * 4 * ntiles * kRadix * 4, 256);
    return s;
}

// vals [B][N] -> idx_out [B][N]; optionally the sorted values.  Returns the free pair buffer (for the scatter) in *spare.
inline cudaError_t seg_argsort32(const float* vals, uint32_t* idx_out, float* sorted_out, long long B, long long N,
                                 void* ws, uint2** spare, cudaStream_t st) {
    constexpr int NP = 4;
    unsigned char* w = (unsigned char*)ws;
    uint2* pa = (uint2*)w; w += align_up((size_t)B * N * sizeof(uint2), 256);
    uint2* pb = (uint2*)w; w += align_up((size_t)B * N * sizeof(uint2), 256);
    const size_t ntiles = (size_t)(N / kS32Tile);
    uint32_t* hist = (uint32_t*)w;
    uint32_t* ticket = hist + (size_t)B * NP * kRadix;
    uint32_t* status = ticket + (size_t)B * NP;
    const size_t ctl = (size_t)B * NP * kRadix * 4 + (size_t)B * NP * 4 + (size_t)B * NP * ntiles * kRadix * 4;
    cudaError_t e = cudaMemsetAsync(hist, 0, ctl, st);
    if (e != cudaSuccess) return e;
    const int chunk = 1 << 16;
    AGN_LAUNCH(K_SORT_HIST, st, (digit_hist_kernel<float, 512><<<bgrid((unsigned)((N + chunk - 1) / chunk), B), 512, 0, st>>>(vals, hist, N, N, chunk, B)));
    AGN_LAUNCH(K_SORT_HIST, st, (digit_scan_kernel<<<(unsigned)(B * NP), kRadix, 0, st>>>(hist)));
    const dim3 grid = bgrid((unsigned)ntiles, B);
    for (int p = 0; p < NP; ++p) {
        Sweep32Args a;
        a.vals = vals;
        a.in = (p == 2) ? pb : pa;                // pass 0: vals -> pa; 1: pa -> pb; 2: pb -> pa; 3: pa -> idx
        a.out = (p == 1) ? pb : pa;
        a.idx_out = idx_out; a.sorted_out = sorted_out;
        a.N = (uint32_t)N; a.shift = p * kRadixBits;
        a.dstart = hist; a.pass = p; a.npass = NP;
        a.status = status + (size_t)p * B * ntiles * kRadix;
        a.ticket = ticket + (size_t)p * B;
        a.ntiles = (uint32_t)ntiles; a.B = B;
        if (p == 0) AGN_LAUNCH(K_SORT_SWEEP, st, (sweep32_kernel<0><<<grid, kS32Threads, sizeof(S32Smem), st>>>(a)));
        else if (p == NP - 1) AGN_LAUNCH(K_SORT_SWEEP, st, (sweep32_kernel<2><<<grid, kS32Threads, sizeof(S32Smem), st>>>(a)));
        else AGN_LAUNCH(K_SORT_SWEEP, st, (sweep32_kernel<1><<<grid, kS32Threads, sizeof(S32Smem), st>>>(a)));
    }
    if (spare) *spare = pb;
    return cudaGetLastError();
}

// L5 two-level for fp32 (N >= 2^kTwoLevelScatterLog).  cursor: [B][256] u32, zero on entry (left zero again).
inline cudaError_t rank_scatter_two_level32(const uint32_t* idx_new, const uint32_t* idx_old, const float* sorted, float* x,
                                            long long B, long long N, uint2* pairs, uint32_t* cursor,
                                            unsigned long long* changed, cudaStream_t st) {
    const int shift = ilog2_u64((uint64_t)N) - kRadixBits;
    AGN_LAUNCH(K_SCATTER_BIN, st, (scatter_bin32_kernel<<<bgrid((unsigned)(N / kS32Tile), B), kS32Threads, sizeof(S32Smem), st>>>(
        idx_new, idx_old, sorted, pairs, (uint32_t)N, shift, cursor, changed, B)));
    AGN_LAUNCH(K_SCATTER_PLACE, st, (scatter_place32_kernel<<<bgrid((unsigned)(N / 2048), B), 256, 0, st>>>(
        (const uint4*)pairs, x, (uint32_t)N, cursor, B)));
    return cudaGetLastError();
}

}  // namespace agn

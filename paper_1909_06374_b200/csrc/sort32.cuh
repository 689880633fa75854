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
#include <cstring>
#include "common.cuh"
#include "sort.cuh"
#include "bucket32.cuh"
#include "bucket1.cuh"

namespace agn {

constexpr int kS32Threads = 256;
constexpr int kS32Kpt = 16;
constexpr int kS32Tile = kS32Threads * kS32Kpt;      // 4096
constexpr int kS32Warps = kS32Threads / 32;
constexpr int kS32Chunk = 4;                         // tiles per look-back unit of the sweep kernel

struct S32Smem {
    uint2 stage[kS32Tile];
    uint32_t cm[2 * kS32Warps * kRadix]; // per (half-warp, digit): running count << 16 | lane mask of the current round;
                                         // after the scan: start of the (half-warp, digit) run inside the tile
    uint32_t tile_off[kRadix];
    uint32_t goff[kRadix];
    uint32_t wsum[kS32Warps];
    uint32_t hist[kRadix];              // sweep: digit counts of the whole chunk
    uint32_t gbase[kRadix];             // sweep: running global start of every digit inside the chunk
    uint32_t tile;
    uint32_t diff;
};

// Element arrangement inside a tile: half-warp v = 2*warp + (lane >> 4) owns the 256 consecutive elements
// v*256 .. v*256+255; item j of sub-lane sl = lane & 15 is element v*256 + j*16 + sl (a half-warp reads 16
// consecutive elements per item: full 128-byte lines for pairs).  Ranking is per half-warp so that the mask of a
// round and the running count share ONE 32-bit shared-memory word (a random 32-bit access costs ~3.4 wavefronts,
// a random 64-bit one ~6): per key one ATOMS.OR, one LDS and one predicated STS.
// Returns local positions; leaves sm.tile_off[d]; returns this thread's digit count (thread == digit).
__device__ __forceinline__ uint32_t s32_elem0() {
    const int v = threadIdx.x >> 4, sl = threadIdx.x & 15;
    return (uint32_t)(v * 256 + sl);
}
constexpr int kS32ItemStride = 16;

__device__ __forceinline__ uint32_t s32_rank(const uint32_t (&dig)[kS32Kpt], uint32_t (&pos)[kS32Kpt], S32Smem& sm) {
    constexpr int V = 2 * kS32Warps;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int v = threadIdx.x >> 4, sl = threadIdx.x & 15;
#pragma unroll
    for (int i = 0; i < V; ++i) sm.cm[i * kRadix + threadIdx.x] = 0u;
    __syncthreads();
    const uint32_t lt = (1u << sl) - 1u, bit = 1u << sl;
    uint32_t* cw = sm.cm + v * kRadix;
    uint32_t r[kS32Kpt];
#pragma unroll
    for (int j = 0; j < kS32Kpt; ++j) {
        const uint32_t d = dig[j];
        atomicOr(&cw[d], bit);
        __syncwarp();
        const uint32_t mc = cw[d];
        const uint32_t mask = mc & 0xffffu;
        r[j] = (mc >> 16) + __popc(mask & lt);
        __syncwarp();
        if ((mask & lt) == 0u) cw[d] = (mc & 0xffff0000u) + ((uint32_t)__popc(mask) << 16);
        __syncwarp();
    }
    __syncthreads();
    // thread == digit: totals over the half-warps, exclusive scan over the digits, then the run starts
    uint32_t run = 0;
#pragma unroll
    for (int i = 0; i < V; ++i) run += sm.cm[i * kRadix + threadIdx.x] >> 16;
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
    const uint32_t toff = inc - run + add;
    sm.tile_off[threadIdx.x] = toff;
    uint32_t acc = toff;
#pragma unroll
    for (int i = 0; i < V; ++i) {
        const uint32_t c = sm.cm[i * kRadix + threadIdx.x] >> 16;
        sm.cm[i * kRadix + threadIdx.x] = acc;
        acc += c;
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kS32Kpt; ++j) pos[j] = cw[dig[j]] + r[j];
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
    uint32_t* status;           // [B][nchunks][256] zero-initialised
    uint32_t* ticket;           // [B] zero-initialised
    uint32_t ntiles, nchunks;
    long long B;
    const uint32_t* gate;       // NULL, or [B]: the curve is sorted here only if its word is non-zero
};

// exclusive scan of every 256-bin histogram, in place (one warp-scan CTA per histogram)
__global__ void __launch_bounds__(kRadix) digit_scan_kernel(uint32_t* __restrict__ hist, const uint32_t* __restrict__ gate,
                                                            int per_curve) {
    __shared__ uint32_t ws[8];
    if (gate && gate[blockIdx.x / per_curve] == 0u) return;
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
// One CTA handles a CHUNK of kS32Chunk consecutive tiles.  Phase A counts the chunk's digits (one streaming read),
// publishes the chunk aggregate and looks back over earlier chunks; phase B re-reads the tiles (they are still in
// L2), ranks each one and writes it out with a running per-digit offset.  The decoupled look-back window is
// (chunks started per microsecond) x (look-back latency): per-tile look-back at ~90 tiles/us made every tile sum
// ~50 predecessor aggregates; per-chunk it is a handful.
template <int KIND>
__device__ __forceinline__ void s32_load_tile(const Sweep32Args& a, size_t seg, uint32_t e0, uint2 (&kv)[kS32Kpt]) {
    if (KIND == 0) {
        const float* v = a.vals + seg + e0;
#pragma unroll
        for (int j = 0; j < kS32Kpt; ++j) kv[j] = make_uint2(key_of(v[j * kS32ItemStride]), e0 + j * kS32ItemStride);
    } else {
        const uint2* v = a.in + seg + e0;
#pragma unroll
        for (int j = 0; j < kS32Kpt; ++j) kv[j] = v[j * kS32ItemStride];
    }
}

template <int KIND>
__global__ void __launch_bounds__(kS32Threads, 4) sweep32_kernel(Sweep32Args a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    S32Smem& sm = *reinterpret_cast<S32Smem*>(smem_raw);
    const long long b = bidx();
    if (b >= a.B) return;
    if (a.gate && a.gate[b] == 0u) return;
    // persistent: a CTA takes chunk tickets until none is left (a gated-off launch then costs a few hundred CTAs, not
    // one per chunk); a CTA only ever waits for chunks with smaller tickets, which are held by running CTAs
    for (;;) {
    __syncthreads();
    if (threadIdx.x == 0) sm.tile = atomicAdd(&a.ticket[b], 1u);
    sm.hist[threadIdx.x] = 0u;
    __syncthreads();
    const uint32_t chunk = sm.tile;
    if (chunk >= a.nchunks) break;
    const uint32_t tiles_here = min((uint32_t)kS32Chunk, a.ntiles - chunk * kS32Chunk);
    const size_t seg = (size_t)b * a.N;
    const uint32_t e00 = chunk * (kS32Chunk * kS32Tile) + s32_elem0();
    uint2 kv[kS32Kpt];
    uint32_t dig[kS32Kpt], pos[kS32Kpt];
    // ---- phase A: digit counts of the chunk
    for (uint32_t c = 0; c < tiles_here; ++c) {
        s32_load_tile<KIND>(a, seg, e00 + c * kS32Tile, kv);
#pragma unroll
        for (int j = 0; j < kS32Kpt; ++j) atomicAdd(&sm.hist[(kv[j].x >> a.shift) & (kRadix - 1)], 1u);
    }
    __syncthreads();
    // ---- thread == digit: publish the chunk aggregate, look back over earlier chunks of the segment
    {
        const int d = threadIdx.x;
        const uint32_t agg = sm.hist[d];
        volatile uint32_t* st = a.status + (size_t)b * a.nchunks * kRadix + d;
        uint32_t excl = 0;
        if (chunk == 0) {
            st[0] = kFlagInc | agg;
        } else {
            st[(size_t)chunk * kRadix] = kFlagAgg | agg;
            int t = (int)chunk - 1;
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
            st[(size_t)chunk * kRadix] = kFlagInc | (excl + agg);
        }
        sm.gbase[d] = a.dstart[((size_t)b * a.npass + a.pass) * kRadix + d] + excl;
    }
    // ---- phase B: rank and write every tile of the chunk (re-read through L2)
    for (uint32_t c = 0; c < tiles_here; ++c) {
        s32_load_tile<KIND>(a, seg, e00 + c * kS32Tile, kv);
#pragma unroll
        for (int j = 0; j < kS32Kpt; ++j) dig[j] = (kv[j].x >> a.shift) & (kRadix - 1);
        const uint32_t cnt = s32_rank(dig, pos, sm);          // has barriers: the previous tile's stage reads are done
        {
            const uint32_t g = sm.gbase[threadIdx.x];
            sm.goff[threadIdx.x] = g - sm.tile_off[threadIdx.x];
            sm.gbase[threadIdx.x] = g + cnt;
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
        __syncthreads();      // stage and goff are rewritten by the next tile
    }
    }   // ticket loop
}

// ------------------------------------------------------------------------------------------------
// L5 two-level: place step (the bin step is bucket_part_kernel<2> of bucket32.cuh)
// ------------------------------------------------------------------------------------------------
template <int kPlaceElems>
__global__ void __launch_bounds__(256) scatter_place32_kernel(const uint4* __restrict__ pairs2, float* __restrict__ x,
                                                              uint32_t N, uint32_t* __restrict__ cursor, long long B,
                                                              const uint32_t* __restrict__ gate) {
    const long long b = bidx();
    if (b >= B) return;
    if (gate && gate[b] == 0u) return;
    if (blockIdx.x == 0) cursor[b * kRadix + threadIdx.x] = 0u;      // ready for the next iteration's bin pass
    const size_t seg = (size_t)b * N;
    float* xs = x + seg;
    // kPlaceElems pairs per CTA (2 per uint4): 2048 where the kernel does the work (1.45 ms per 2^28 pairs; 8192 measured
    // 1.99 ms), 8192 where it is the gated fallback of the write-back sort and normally exits at once -- its cost is then
    // the number of CTAs (131072 CTAs of 2048 pairs took 70 us per C4 iteration doing nothing).
    const uint4* p = pairs2 + (seg >> 1) + (size_t)blockIdx.x * (kPlaceElems / 2) + threadIdx.x;
#pragma unroll 4
    for (int i = 0; i < kPlaceElems / 512; ++i) {
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
    cudaFuncSetAttribute(sweep32_kernel<0>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaFuncSetAttribute(sweep32_kernel<1>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    cudaFuncSetAttribute(sweep32_kernel<2>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    if (e == cudaSuccess) e = bucket32_set_attrs();
    if (e == cudaSuccess) e = bucket1_set_attrs();
    return e;
}

inline bool sort32_applicable(size_t elem_size, long long N) {
    return elem_size == 4 && N > SortCfg<float>::ctaMax && N <= (1ll << 27);
}

// workspace (bytes): two pair buffers + control (hist, tickets, status)
inline size_t sort32_ws_bytes(long long B, long long N) {
    const size_t ntiles = (size_t)(N / kS32Tile);
    size_t s = 2 * align_up((size_t)B * N * sizeof(uint2), 256);
    if (bucket1_applicable(4, N)) s = std::max(s, align_up(bucket1_pair_elems(B, N) * sizeof(uint2), 256));
    else if (bucket32_applicable(4, N)) s = std::max(s, align_up(bucket32_pair_elems(B, N) * sizeof(uint2), 256));
    s += align_up((size_t)B * 4 * kRadix * 4 + (size_t)B * 4 * 4 + (size_t)B * 4 * ntiles * kRadix * 4, 256);
    if (bucket1_applicable(4, N)) s += bucket1_ctl_bytes(B, N);
    else if (bucket32_applicable(4, N)) s += bucket32_ctl_bytes(B, N);
    return s;
}

// Control words of the LSD passes for the curves that take them (gate[b] != 0): digit histograms [B][4][256], tickets
// [4][B], look-back status [4][B][nchunks][256] (pass stride B * ntiles * 256).  Exits at once for the other curves,
// which is every curve of a normal run: the bucket sort has already sorted them.
__global__ void __launch_bounds__(kRadix) lsd_clear_kernel(uint32_t* __restrict__ hist, uint32_t* __restrict__ ticket,
                                                           uint32_t* __restrict__ status, const uint32_t* __restrict__ gate,
                                                           uint32_t nchunks, size_t pass_stride, long long B) {
    const long long b = bidx();
    if (b >= B || gate[b] == 0u) return;
    for (uint32_t u = blockIdx.x; u < 4u * nchunks; u += gridDim.x) {
        const uint32_t p = u / nchunks, c = u - p * nchunks;
        status[(size_t)p * pass_stride + ((size_t)b * nchunks + c) * kRadix + threadIdx.x] = 0u;
        if (c == 0) {
            hist[((size_t)b * 4 + p) * kRadix + threadIdx.x] = 0u;
            if (threadIdx.x == 0) ticket[(size_t)p * B + b] = 0u;
        }
    }
}

// vals [B][N] -> idx_out [B][N]; optionally the sorted values.  Returns the free pair buffer (for the scatter) in *spare.
// wb (one-level distribution sort only): write-back mode, see B1Wb in bucket1.cuh.
inline cudaError_t seg_argsort32(const float* vals, uint32_t* idx_out, float* sorted_out, long long B, long long N,
                                 void* ws, uint2** spare, cudaStream_t st, const uint32_t** gate_out = nullptr,
                                 const B1Wb* wb = nullptr) {
    constexpr int NP = 4;
    unsigned char* w = (unsigned char*)ws;
    uint2* pa = (uint2*)w; w += align_up((size_t)B * N * sizeof(uint2), 256);
    uint2* pb = (uint2*)w; w += align_up((size_t)B * N * sizeof(uint2), 256);
    const bool one_level = bucket1_applicable(4, N);
    if (one_level) w = (unsigned char*)ws + std::max((size_t)(w - (unsigned char*)ws), align_up(bucket1_pair_elems(B, N) * sizeof(uint2), 256));
    else if (bucket32_applicable(4, N)) w = (unsigned char*)ws + std::max((size_t)(w - (unsigned char*)ws), align_up(bucket32_pair_elems(B, N) * sizeof(uint2), 256));
    const size_t ntiles = (size_t)(N / kS32Tile);
    uint32_t* hist = (uint32_t*)w;
    uint32_t* ticket = hist + (size_t)B * NP * kRadix;
    uint32_t* status = ticket + (size_t)B * NP;
    const size_t ctl = (size_t)B * NP * kRadix * 4 + (size_t)B * NP * 4 + (size_t)B * NP * ntiles * kRadix * 4;
    cudaError_t e;
    // long curves: distribution sort, one partition level (bucket1.cuh; N <= 2^26) or two (bucket32.cuh; N = 2^27); the
    // LSD passes below then only run for curves it gave up on
    const uint32_t* gate = nullptr;
    if (one_level) {
        e = bucket1_sort(vals, idx_out, sorted_out, B, N, pa, w + align_up(ctl, 256), &gate, st, wb);
        if (e != cudaSuccess) return e;
    } else if (bucket32_applicable(4, N)) {
        e = bucket32_sort(vals, idx_out, sorted_out, B, N, pa, w + align_up(ctl, 256), &gate, st);
        if (e != cudaSuccess) return e;
    }
    const size_t nchunks = (ntiles + kS32Chunk - 1) / kS32Chunk;
    if (gate) {
        AGN_LAUNCH(K_SORT_FALLBACK, st, (lsd_clear_kernel<<<bgrid((unsigned)std::min<size_t>(NP * nchunks, 512), B), kRadix, 0, st>>>(
            hist, ticket, status, gate, (uint32_t)nchunks, (size_t)B * ntiles * kRadix, B)));
    } else {
        e = cudaMemsetAsync(hist, 0, ctl, st);
        if (e != cudaSuccess) return e;
    }
    const int chunk = 1 << 16;
    // with a gate these launches are the fallback of the distribution sort: they exit at once unless a slab overflowed
    const int id_hist = gate ? K_SORT_FALLBACK : K_SORT_HIST, id_sweep = gate ? K_SORT_FALLBACK : K_SORT_SWEEP;
    AGN_LAUNCH(id_hist, st, (digit_hist_kernel<float, 512><<<bgrid((unsigned)((N + chunk - 1) / chunk), B), 512, 0, st>>>(vals, hist, N, N, chunk, B, gate)));
    AGN_LAUNCH(id_hist, st, (digit_scan_kernel<<<(unsigned)(B * NP), kRadix, 0, st>>>(hist, gate, NP)));
    const dim3 grid = bgrid((unsigned)std::min<size_t>(nchunks, 592), B);
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
        a.ntiles = (uint32_t)ntiles; a.nchunks = (uint32_t)nchunks; a.B = B; a.gate = gate;
        if (p == 0) AGN_LAUNCH(id_sweep, st, (sweep32_kernel<0><<<grid, kS32Threads, sizeof(S32Smem), st>>>(a)));
        else if (p == NP - 1) AGN_LAUNCH(id_sweep, st, (sweep32_kernel<2><<<grid, kS32Threads, sizeof(S32Smem), st>>>(a)));
        else AGN_LAUNCH(id_sweep, st, (sweep32_kernel<1><<<grid, kS32Threads, sizeof(S32Smem), st>>>(a)));
    }
    if (spare) *spare = pb;
    if (gate_out) *gate_out = gate;
    return cudaGetLastError();
}

// L5 two-level for fp32 (N >= 2^kTwoLevelScatterLog).  cursor: [B][256] u32, zero on entry (left zero again).
inline cudaError_t rank_scatter_two_level32(const uint32_t* idx_new, const uint32_t* idx_old, const float* sorted, float* x,
                                            long long B, long long N, uint2* pairs, uint32_t* cursor,
                                            unsigned long long* changed, cudaStream_t st, const uint32_t* gate = nullptr) {
    const int shift = ilog2_u64((uint64_t)N) - kRadixBits;
    // bin step: the tile kernel of bucket32.cuh in its LEVEL 2 form (no order is needed inside a window)
    PartArgs a;
    memset(&a, 0, sizeof(a));
    a.vals = sorted; a.idx_new = idx_new; a.idx_old = idx_old; a.changed = changed;
    a.out = pairs; a.cursor = cursor; a.N = (uint32_t)N; a.lb = (uint32_t)shift; a.nc = kRadix; a.nb = kRadix;
    a.cap_out = (uint32_t)(N >> kRadixBits); a.B = B; a.gate = gate;
    // with a gate these two launches are the fallback of the write-back sort: they exit at once for every other curve
    AGN_LAUNCH(gate ? K_SORT_FALLBACK : K_SCATTER_BIN, st, (bucket_part_kernel<2><<<bgrid((unsigned)(N / bk_part_tile(2)), B), kBkPartThreads, sizeof(PartSmem<2>), st>>>(a)));
    if (gate)
        AGN_LAUNCH(K_SORT_FALLBACK, st, (scatter_place32_kernel<8192><<<bgrid((unsigned)(N / 8192), B), 256, 0, st>>>(
            (const uint4*)pairs, x, (uint32_t)N, cursor, B, gate)));
    else
        AGN_LAUNCH(K_SCATTER_PLACE, st, (scatter_place32_kernel<2048><<<bgrid((unsigned)(N / 2048), B), 256, 0, st>>>(
            (const uint4*)pairs, x, (uint32_t)N, cursor, B, gate)));
    return cudaGetLastError();
}

}  // namespace agn

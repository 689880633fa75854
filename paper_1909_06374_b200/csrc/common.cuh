// common.cuh -- shared device helpers of the agnvar CUDA library (sm_100a).
// Nothing here is shared with oracle/ (the CPU oracle is independent test infrastructure).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <stdlib.h>
#include <mutex>

namespace agn {

// ------------------------------------------------------------------------------------------------
// complex numbers on float2 / double2
// ------------------------------------------------------------------------------------------------
template <typename T> struct Cx;
template <> struct Cx<float> { typedef float2 type; };
template <> struct Cx<double> { typedef double2 type; };

template <typename T> __host__ __device__ __forceinline__ typename Cx<T>::type mk(T a, T b) {
    typename Cx<T>::type r; r.x = a; r.y = b; return r;
}
template <typename C> __device__ __forceinline__ C cadd(C a, C b) { a.x += b.x; a.y += b.y; return a; }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { a.x -= b.x; a.y -= b.y; return a; }
template <typename C> __device__ __forceinline__ C cmul(C a, C b) {
    C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r;
}
// a * conj(b)
template <typename C> __device__ __forceinline__ C cmulc(C a, C b) {
    C r; r.x = a.x * b.x + a.y * b.y; r.y = a.y * b.x - a.x * b.y; return r;
}
template <typename C> __device__ __forceinline__ C cconj(C a) { a.y = -a.y; return a; }
template <typename C> __device__ __forceinline__ C cswap(C a) { C r; r.x = a.y; r.y = a.x; return r; }
// multiply by -i (forward radix-4 rotation) : (x, y) -> (y, -x)
template <typename C> __device__ __forceinline__ C cmul_mi(C a) { C r; r.x = a.y; r.y = -a.x; return r; }

__host__ __device__ __forceinline__ int ilog2_u64(uint64_t v) {
    int l = 0;
    while (v > 1) { v >>= 1; ++l; }
    return l;
}

// ------------------------------------------------------------------------------------------------
// Philox4x32-10 (O1).  Round: p0 = 0xD2511F53*c0, p1 = 0xCD9E8D57*c2;
// c <- (hi(p1)^c1^k0, lo(p1), hi(p0)^c3^k1, lo(p0)); key += (0x9E3779B9, 0xBB67AE85).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        uint4 n;
        n.x = hi1 ^ c.y ^ k.x;
        n.y = lo1;
        n.z = hi0 ^ c.w ^ k.y;
        n.w = lo0;
        c = n;
        k.x += 0x9E3779B9u;
        k.y += 0xBB67AE85u;
    }
    return c;
}

// counter = (i lo, i hi, curve b, tag), key = (seed lo, seed hi)
__device__ __forceinline__ uint4 philox_stream(uint64_t seed, uint64_t i, uint32_t b, uint32_t tag) {
    uint4 c = make_uint4((uint32_t)i, (uint32_t)(i >> 32), b, tag);
    uint2 k = make_uint2((uint32_t)seed, (uint32_t)(seed >> 32));
    return philox4x32_10(c, k);
}

// u = (2*(wa*2^20 + (wb>>12)) + 1) * 2^-53, exact in fp64, in (0,1)
__device__ __forceinline__ double u53(uint32_t wa, uint32_t wb) {
    uint64_t m = ((uint64_t)wa << 20) + (uint64_t)(wb >> 12);
    return (double)(2 * m + 1) * (1.0 / 9007199254740992.0);
}

// ------------------------------------------------------------------------------------------------
// order-preserving radix keys; -0 is canonicalised to +0 (Q13) so that bitwise order == '<' order
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t key_of(float v) {
    uint32_t u = __float_as_uint(v);
    if (u == 0x80000000u) u = 0u;
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ uint64_t key_of(double v) {
    uint64_t u = (uint64_t)__double_as_longlong(v);
    if (u == 0x8000000000000000ull) u = 0ull;
    return (u & 0x8000000000000000ull) ? ~u : (u | 0x8000000000000000ull);
}
__device__ __forceinline__ float val_of(uint32_t k) {
    uint32_t u = (k & 0x80000000u) ? (k & 0x7FFFFFFFu) : ~k;
    return __uint_as_float(u);
}
__device__ __forceinline__ double val_of(uint64_t k) {
    uint64_t u = (k & 0x8000000000000000ull) ? (k & 0x7FFFFFFFFFFFFFFFull) : ~k;
    return __longlong_as_double((long long)u);
}

template <typename T> struct KeyT;
template <> struct KeyT<float> { typedef uint32_t type; static constexpr int bits = 32; };
template <> struct KeyT<double> { typedef uint64_t type; static constexpr int bits = 64; };

// ------------------------------------------------------------------------------------------------
// accurate sin/cos of 2*pi*num/den for integer num in [0, den), den a power of two (exact argument)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void sincos_2pi_frac(uint64_t num, int log_den, double* s, double* c) {
    // 2*num/den is exact in fp64 (num < 2^53)
    double a = ldexp((double)num, 1 - log_den);
    sincospi(a, s, c);
}

// batch index spread over grid y and z (gridDim.y is limited to 65535)
__device__ __forceinline__ long long bidx() { return (long long)blockIdx.z * gridDim.y + blockIdx.y; }
static inline dim3 bgrid(unsigned x, long long nb) {
    unsigned gy = nb > 32768 ? 32768u : (unsigned)nb;
    unsigned gz = (unsigned)((nb + gy - 1) / gy);
    return dim3(x, gy, gz);
}

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// ------------------------------------------------------------------------------------------------
// per-device host-side state (function attributes set, SM count, occupancy-derived grid sizes): keyed by the real
// device ordinal, so that one process may drive several devices
// ------------------------------------------------------------------------------------------------
struct DevCache {
    int dev = -1;
    bool attrs[2] = {false, false};     // by element size (4, 8)
    int sms = 0;
    int grid[32] = {0};                 // persistent-kernel grid sizes, by kernel slot
};
// Threading contract (include/agnvar.h, "Threads"): the slot's first-use initialisation is serialised here, but the
// entries (attrs, grid) are then read and written without locks -- host threads that drive the SAME device must not
// be inside the library at the same time; threads on different devices are independent.
inline DevCache& dev_cache() {
    static DevCache tab[64];
    static std::mutex mu;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0) dev = 0;   // no usable device: the first launch reports the error
    DevCache& c = tab[dev & 63];
    std::lock_guard<std::mutex> lock(mu);
    if (c.dev != dev) {                 // first use of this ordinal (or an ordinal >= 64 aliasing a slot): start over
        c = DevCache();
        c.dev = dev;
        if (cudaDeviceGetAttribute(&c.sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || c.sms < 1) c.sms = 1;
    }
    return c;
}

// ------------------------------------------------------------------------------------------------
// launch trace (agnvar_trace_start / agnvar_trace_stop): when enabled, every kernel launch of the
// library is bracketed by two CUDA events on its stream, so that a caller can read per-kernel device
// time and launch counts of exactly the launches it timed.  Off by default (zero cost).
// ------------------------------------------------------------------------------------------------
enum KernelId {
    K_FFT_STRIDED = 0, K_FFT_CONTIG, K_REPLACE, K_SORT_CTA, K_SORT_HIST, K_SORT_SWEEP, K_SCATTER, K_ITER_POST,
    K_PERM_ANORM, K_TK_FILL, K_TK_COMBINE, K_UNTANGLE_OUT, K_PSD, K_ERDF_TABLE, K_ERDF_SAMPLE, K_PGRAM, K_TABLES,
    K_COPY, K_PHILOX, K_SCATTER_BIN, K_SCATTER_PLACE, K_FFT_COL, K_FFT_MID, K_SORT_CDF, K_SORT_PART0, K_SORT_BUCKET, K_DELTA, K_SORT_PART1, K_SORT_PART_ONE, K_E13_ONCHIP, K_SF, K_SORT_FALLBACK, K_SORT_PART_ONE_WB, K_SORT_BUCKET_WB, K_GATHER_BACK, K_SLICE_SAMPLE, K_NIDS
};
static const char* const kKernelNames[K_NIDS] = {
    "fft_pass_strided", "fft_pass_contiguous", "amplitude_replace", "cta_argsort", "sort_digit_hist",
    "sort_onesweep", "rank_scatter_count", "iter_bookkeeping", "perm_anorm", "tk_fill", "tk_combine5_crop",
    "untangle_out", "psd", "erdf_table", "erdf_sample", "periodogram_scale_bin", "twiddle_tables", "copy", "philox",
    "scatter_bin", "scatter_place", "fft_columns", "fft_mid_fused", "sort_cdf_tables", "sort_part_level0",
    "sort_bucket_finish", "delta_rms", "sort_part_level1", "sort_part_onelevel", "e13_onchip_loop", "structure_function", "sort_lsd_fallback_gated",
    "sort_part_onelevel_rec", "sort_finish_writeback", "scatter_gather_back", "slice_sample"};

struct TraceRec { int id; cudaEvent_t e0, e1; };
struct TraceState {
    bool on = false;
    unsigned long long launches = 0;   // every kernel launch of the library, traced or not
    TraceRec* recs = nullptr;
    size_t n = 0, cap = 0;
    cudaEvent_t* pool = nullptr;
    size_t pool_n = 0, pool_used = 0;
};
inline TraceState& trace_state() { static TraceState s; return s; }
inline cudaEvent_t trace_event() {
    TraceState& t = trace_state();
    if (t.pool_used == t.pool_n) {
        size_t nn = t.pool_n ? t.pool_n * 2 : 1024;
        t.pool = (cudaEvent_t*)realloc(t.pool, nn * sizeof(cudaEvent_t));
        for (size_t i = t.pool_n; i < nn; ++i) cudaEventCreate(&t.pool[i]);
        t.pool_n = nn;
    }
    return t.pool[t.pool_used++];
}
struct TraceScope {
    cudaStream_t st; bool on;
    TraceScope(int id, cudaStream_t s) : st(s), on(trace_state().on) {
        TraceState& t = trace_state();
        ++t.launches;
        if (!on) return;
        if (t.n == t.cap) { t.cap = t.cap ? t.cap * 2 : 1024; t.recs = (TraceRec*)realloc(t.recs, t.cap * sizeof(TraceRec)); }
        TraceRec& r = t.recs[t.n++];
        r.id = id; r.e0 = trace_event(); r.e1 = trace_event();
        cudaEventRecord(r.e0, st);
    }
    ~TraceScope() { if (on) cudaEventRecord(trace_state().recs[trace_state().n - 1].e1, st); }
};
#define AGN_TRACE(id, st) ::agn::TraceScope _agn_trace_scope_((id), (st))
// one kernel launch, counted and (when tracing) timed
#define AGN_LAUNCH(id, st, ...) do { ::agn::TraceScope _agn_ts_((id), (st)); __VA_ARGS__; } while (0)

}  // namespace agn

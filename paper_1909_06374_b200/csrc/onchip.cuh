// onchip.cuh -- the whole E13 loop (L1-L6) of one short light curve inside ONE CTA (fp32: 256 <= N <= 2^14; fp64:
// 256 <= N <= 2^13): x_sim, the spectrum, the sort's (key, index) pairs, the slot counters and the previous permutation
// all live in shared memory (fp32: 12 N bytes, 12 KB at N = 1024, 192 KB at N = 2^14; fp64: 20 N bytes, 80 KB at
// N = 4096); HBM sees perm0 and the result once per call, and per iteration only A_norm (half a value per sample) and
// sorted[] (one value per sample), both re-read through L1/L2.  A curve leaves the
// loop at its own first k with changed = 0 (L6 decided on chip; no other curve waits for it), CTAs take curves from a
// ticket counter.  This is SURVEY section 7 steps 4-5 / 8(d): "one curve per CTA: on-chip loop".
//
// Per iteration:
//   L1  forward FFT of z[n] = x[2n] + i x[2n+1] (L = N/2 points): Stockham radix-8/4/2 stages in shared memory
//   L2  real-FFT untangle + amplitude replace + re-tangle on the pairs (k, L - k), natural order
//   L3  inverse FFT (swap trick), 1/L; x_adj + 0.0 (Q13)
//   L4  stable argsort of x_adj as an interpolation counting sort: slot = monotone linear map of the VALUE onto
//       [mean - 4 sigma, mean + 4 sigma] (N slots, clamped; any monotone map gives the same result, this one keeps the
//       slots about equally full for the near-Gaussian x_adj), 16-bit slot counters packed two per word, pairs grouped
//       by slot, then the exact rank of every pair among its slot mates by the 64-bit (key, index) comparison: ties come
//       out by ascending time index (O6 step 4), bit-identical to std::stable_sort.  Cost grows with the square of a
//       slot's population: an input with massive ties (all keys equal) is still sorted exactly, slowly.
//   L5  changed += (idx_new[r] != idx_old[r]);  x_sim[idx_new[r]] = sorted[r]
//   L6  changed = 0 -> converged (iters_used = k); with the paper's delta_i rule (Eq. 4) switched on, also
//       delta_k <= threshold.  delta_k costs one more pass over the curve per iteration: x_sim,k goes to the curve's
//       output row in global memory at the start of the iteration (L2-resident) and is compared with x_sim,k+1 at the end.
#pragma once
#include "common.cuh"
#include "fft.cuh"
#include "kernels.cuh"

namespace agn {

// (key, time index) of the in-CTA sort: fp32 packs both into one 64-bit word; fp64 keys are 64 bits wide themselves
template <typename T> struct OcPair;
template <> struct OcPair<float> {
    typedef unsigned long long type;
    static __device__ __forceinline__ type make(float v, uint32_t idx) { return ((unsigned long long)key_of(v) << 32) | idx; }
    static __device__ __forceinline__ bool less(const type& a, const type& b) { return a < b; }
    static __device__ __forceinline__ uint32_t idx(const type& a) { return (uint32_t)a; }
    static __device__ __forceinline__ float val(const type& a) { return val_of((uint32_t)(a >> 32)); }
};
template <> struct OcPair<double> {
    typedef ulonglong2 type;            // x = key, y = index
    static __device__ __forceinline__ type make(double v, uint32_t idx) { return make_ulonglong2(key_of(v), (unsigned long long)idx); }
    static __device__ __forceinline__ bool less(const type& a, const type& b) { return a.x < b.x || (a.x == b.x && a.y < b.y); }
    static __device__ __forceinline__ uint32_t idx(const type& a) { return (uint32_t)a.y; }
    static __device__ __forceinline__ double val(const type& a) { return val_of((uint64_t)a.x); }
};

template <typename T, int LOGN> struct OnchipCfg {
    static constexpr int N = 1 << LOGN, L = N / 2;
    static constexpr int THREADS = (N / 8 > 1024) ? 1024 : N / 8;
    static constexpr int KPT = N / THREADS;             // keys per thread (8 or 16)
    static constexpr int EPT = L / THREADS;             // complex points per thread in an FFT stage (4 or 8)
    static constexpr int RP = L + (L >> 4);             // padded row
    static constexpr int WARPS = THREADS / 32;
    // region A: spectrum / x_sim (complex RP) in the FFT half of an iteration, (key, index) pairs in the sort half
    static constexpr size_t bytesA = (size_t)N * sizeof(typename OcPair<T>::type) > (size_t)RP * 2 * sizeof(T)
                                         ? (size_t)N * sizeof(typename OcPair<T>::type) : (size_t)RP * 2 * sizeof(T);
    static constexpr size_t smem = bytesA + (size_t)N * 2 /* packed slot counters */ + (size_t)N * 2 /* idx_old u16 */ +
                                   (size_t)(2 * 32 + 32) * 8 /* reduction scratch */;
};

template <typename T> struct OnchipArgs {
    const T* anorm;             // [B][L+1] natural order
    const T* sorted;            // [B][N]
    uint32_t* perm;             // [B][N] in: perm0, out: final permutation
    T* x;                       // [B][N] out
    T* xadj_dbg;                // [B][N] or NULL: x_adj of the last executed iteration
    int32_t* iters_used;        // [B] or NULL
    long long* hist;            // [B][max_iter] or NULL (zeroed by the host)
    const typename Cx<T>::type* tw14;   // exp(-2 pi i m / 2^14)
    unsigned int* ticket;       // zero on entry
    int max_iter;
    long long B;
    // the paper's stopping rule (Eq. 4; NEXT-1), off when both are unset: delta_k = rms over the
    // samples of log10(x_sim,k+1 / x_sim,k); a curve also stops at the first k with delta_k <= delta_threshold
    double delta_threshold;     // <= 0: exact rank-change rule only
    double* delta_hist;         // [B][max_iter] or NULL (zeroed by the host)
};

// float index of time sample j inside the padded complex row
__device__ __forceinline__ int xpos(int j) { const int n = j >> 1; return 2 * (n + (n >> 4)) + (j & 1); }

// all Stockham stages of one row of L = 2^logL points (natural in -> natural out, forward sign)
template <typename T, int THREADS, int EPT>
__device__ __forceinline__ void onchip_fft(typename Cx<T>::type* s, int logL, int Rp, const typename Cx<T>::type* __restrict__ tw14) {
    constexpr int RAD = EPT >= 8 ? 8 : EPT;
    constexpr int LOGRAD = RAD == 8 ? 3 : (RAD == 4 ? 2 : 1);
    int logNs = 0;
    while (logL - logNs >= LOGRAD) {
        fft_stage<T, RAD, THREADS, EPT, true>(s, logL, logNs, 0, Rp, tw14);
        logNs += LOGRAD;
    }
    if (logL - logNs == 2) fft_stage<T, 4, THREADS, EPT, true>(s, logL, logNs, 0, Rp, tw14);
    else if (logL - logNs == 1) fft_stage<T, 2, THREADS, EPT, true>(s, logL, logNs, 0, Rp, tw14);
}

// DM: with the delta_i rule (a separate instantiation, so that the plain loop's code and register use stay as they were)
template <typename T, int LOGN, bool DM>
__global__ void __launch_bounds__(OnchipCfg<T, LOGN>::THREADS) e13_onchip_kernel(OnchipArgs<T> a) {
    typedef OnchipCfg<T, LOGN> Cfg;
    typedef typename Cx<T>::type C;
    typedef OcPair<T> PR;
    typedef typename PR::type Pair;
    constexpr int N = Cfg::N, L = Cfg::L, THREADS = Cfg::THREADS, KPT = Cfg::KPT, RP = Cfg::RP, WARPS = Cfg::WARPS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* Z = reinterpret_cast<C*>(smem_raw);
    T* Zf = reinterpret_cast<T*>(smem_raw);
    Pair* pair = reinterpret_cast<Pair*>(smem_raw);
    uint32_t* cw = reinterpret_cast<uint32_t*>(smem_raw + Cfg::bytesA);                  // [N/2]
    unsigned short* perm_s = reinterpret_cast<unsigned short*>(smem_raw + Cfg::bytesA + (size_t)N * 2);      // [N]
    double* red = reinterpret_cast<double*>(smem_raw + Cfg::bytesA + (size_t)N * 4);     // [64] + [32]
    __shared__ unsigned int s_curve;
    __shared__ T s_lo, s_scale;
    __shared__ unsigned int s_changed;
    __shared__ int s_stop;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    // delta_k wanted: x_sim,k is parked in the curve's output row a.x (every thread stores and later re-reads its own
    // samples, so no ordering between threads is involved), and compared with x_sim,k+1 once that sits in region A
    constexpr bool dm = DM;

    for (;;) {
    __syncthreads();
    if (t == 0) s_curve = atomicAdd(a.ticket, 1u);
    __syncthreads();
    const long long b = s_curve;
    if (b >= a.B) break;
    const T* An = a.anorm + b * (L + 1);
    const T* srt = a.sorted + b * N;
    uint32_t* pg = a.perm + b * N;
    // x_sim,1: the draw in draw order (Q15); idx_old = perm0
    for (int r = t; r < N; r += THREADS) {
        const uint32_t i = pg[r];
        perm_s[r] = (unsigned short)i;
        Zf[xpos((int)i)] = srt[r];
    }
    int used = a.max_iter;
    for (int k = 1; k <= a.max_iter; ++k) {
        __syncthreads();
        if (dm) {
            T* xo = a.x + b * N;
#pragma unroll
            for (int i = 0; i < KPT; ++i) { const int j = i * THREADS + t; xo[j] = Zf[xpos(j)]; }
        }
        // ---- L1 forward FFT (a stage reads, synchronises, then writes: the reads above are done before any write)
        onchip_fft<T, THREADS, Cfg::EPT>(Z, LOGN - 1, RP, a.tw14);
        // ---- L2 untangle + amplitude replace + re-tangle (the stage's trailing barrier has been passed)
        for (int kk = t; kk <= L / 2; kk += THREADS) {
            if (kk == 0) {
                const C z0 = Z[0];
                const T x0 = z0.x + z0.y, xl = z0.x - z0.y;
                const T a0 = An[0], al = An[L];
                const T y0 = (x0 != (T)0) ? (x0 > (T)0 ? a0 : -a0) : a0;
                const T yl = (xl != (T)0) ? (xl > (T)0 ? al : -al) : al;
                Z[0] = mk<T>((T)0.5 * (y0 + yl), (T)0.5 * (y0 - yl));
            } else {
                const int k2 = L - kk;
                const int p1 = kk + (kk >> 4), p2 = k2 + (k2 >> 4);
                C z1 = Z[p1], z2 = Z[p2];
                replace_pair<T>(z1, z2, a.tw14[kk << (kLogTw - LOGN)], An[kk], An[k2]);      // w_N^k
                Z[p1] = z1;
                if (k2 != kk) Z[p2] = z2;
            }
        }
        __syncthreads();
        // ---- L3 inverse FFT: swap, forward stages, swap and 1/L (folded into the key read below)
        for (int n = t; n < L; n += THREADS) { const int p = n + (n >> 4); Z[p] = cswap(Z[p]); }
        __syncthreads();
        onchip_fft<T, THREADS, Cfg::EPT>(Z, LOGN - 1, RP, a.tw14);
        // ---- L4 keys into registers: x_adj[j] = (1/L) * swapped component, + 0.0 (Q13)
        T v[KPT];
        const T invL = (T)1 / (T)L;
        T sum = 0, sq = 0;
#pragma unroll
        for (int i = 0; i < KPT; ++i) {
            const int j = i * THREADS + t;
            const int n = j >> 1;
            // element j of the real series is the (j & 1) component of the UNSWAPPED result = the other one of Z
            v[i] = Zf[2 * (n + (n >> 4)) + ((j & 1) ^ 1)] * invL + (T)0;
            sum += v[i];
            sq = fma(v[i], v[i], sq);
        }
        if (a.xadj_dbg) {
#pragma unroll
            for (int i = 0; i < KPT; ++i) a.xadj_dbg[b * N + i * THREADS + t] = v[i];
        }
        // mean and sigma of x_adj (any values give a correct sort: they only place the slots)
        {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) { sum += __shfl_xor_sync(0xffffffffu, sum, o); sq += __shfl_xor_sync(0xffffffffu, sq, o); }
            if (lane == 0) { red[warp] = (double)sum; red[32 + warp] = (double)sq; }
            if (t == 0) s_changed = 0u;
            __syncthreads();            // also: every thread has read its keys out of region A
            if (warp == 0) {
                double s1 = lane < WARPS ? red[lane] : 0.0, s2 = lane < WARPS ? red[32 + lane] : 0.0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) { s1 += __shfl_xor_sync(0xffffffffu, s1, o); s2 += __shfl_xor_sync(0xffffffffu, s2, o); }
                if (lane == 0) {
                    const double mu = s1 / (double)N;
                    double var = s2 / (double)N - mu * mu;
                    if (!(var > 0.0)) var = 0.0;
                    const double sg = sqrt(var);
                    const double lo = mu - 4.0 * sg, width = 8.0 * sg;
                    s_lo = (T)lo;
                    s_scale = (width > 0.0 && isfinite(width)) ? (T)((double)N / width) : (T)0;
                }
            }
            for (int i = t; i < N / 2; i += THREADS) cw[i] = 0u;
            __syncthreads();
        }
        const T lo = s_lo, scale = s_scale;
        auto slot_of = [&](T x) -> uint32_t {
            const T f = (x - lo) * scale;                          // monotone in x; NaN / negative -> slot 0
            return (f >= (T)1) ? min((uint32_t)f, (uint32_t)(N - 1)) : 0u;     // (the conversion saturates)
        };
        // slot populations
#pragma unroll
        for (int i = 0; i < KPT; ++i) {
            const uint32_t s = slot_of(v[i]);
            atomicAdd(&cw[s >> 1], 1u << ((s & 1u) << 4));
        }
        __syncthreads();
        // exclusive scan of the N slot populations: thread t owns the WPT consecutive words [t * WPT, (t + 1) * WPT)
        {
            constexpr int WPT = N / 2 / THREADS;        // 4 or 8 words = 8 or 16 slots
            uint32_t w[WPT];
            uint32_t tot = 0;
#pragma unroll
            for (int i = 0; i < WPT / 4; ++i) {
                const uint4 q = reinterpret_cast<const uint4*>(cw)[t * (WPT / 4) + i];
                w[4 * i] = q.x; w[4 * i + 1] = q.y; w[4 * i + 2] = q.z; w[4 * i + 3] = q.w;
            }
#pragma unroll
            for (int i = 0; i < WPT; ++i) tot += (w[i] & 0xffffu) + (w[i] >> 16);
            uint32_t inc = tot;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t m = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += m;
            }
            uint32_t* wsum = reinterpret_cast<uint32_t*>(red + 64);
            if (lane == 31) wsum[warp] = inc;
            __syncthreads();
            uint32_t run = inc - tot;
#pragma unroll
            for (int wv = 0; wv < WARPS; ++wv) run += (wv < warp) ? wsum[wv] : 0u;
#pragma unroll
            for (int i = 0; i < WPT; ++i) {
                const uint32_t l0 = run; run += w[i] & 0xffffu;
                const uint32_t h0 = run; run += w[i] >> 16;
                w[i] = l0 | (h0 << 16);
            }
#pragma unroll
            for (int i = 0; i < WPT / 4; ++i)
                reinterpret_cast<uint4*>(cw)[t * (WPT / 4) + i] = make_uint4(w[4 * i], w[4 * i + 1], w[4 * i + 2], w[4 * i + 3]);
        }
        __syncthreads();
        // pairs grouped by slot (any order inside a slot); counters end as the END of each slot
#pragma unroll
        for (int i = 0; i < KPT; ++i) {
            const uint32_t s = slot_of(v[i]), sh = (s & 1u) << 4;
            const uint32_t q = (atomicAdd(&cw[s >> 1], 1u << sh) >> sh) & 0xffffu;
            pair[q] = PR::make(v[i], (uint32_t)(i * THREADS + t));
        }
        __syncthreads();
        // exact rank among the slot mates; L5 on the fly: change count, idx_old <- idx_new, value for x_sim
        uint32_t oidx[KPT];
        T oval[KPT];
        uint32_t diff = 0;
#pragma unroll
        for (int i = 0; i < KPT; ++i) {
            const int q = i * THREADS + t;
            const Pair pv = pair[q];
            const uint32_t s = slot_of(PR::val(pv));
            const uint32_t w = cw[s >> 1];
            uint32_t z, st0;
            if (s & 1u) { z = w >> 16; st0 = w & 0xffffu; }
            else { z = w & 0xffffu; st0 = s ? (cw[(s >> 1) - 1] >> 16) : 0u; }
            uint32_t r = (uint32_t)q;
            if (z - st0 > 1u) {
                r = st0;
                for (uint32_t h = st0; h < z; ++h) r += PR::less(pair[h], pv);
            }
            const uint32_t idx = PR::idx(pv);
            diff += ((uint32_t)perm_s[r] != idx);
            perm_s[r] = (unsigned short)idx;
            oidx[i] = idx;
            oval[i] = srt[r];
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) diff += __shfl_xor_sync(0xffffffffu, diff, o);
        if (lane == 0 && diff) atomicAdd(&s_changed, diff);
        __syncthreads();                // every pair has been read: region A becomes x_sim again
#pragma unroll
        for (int i = 0; i < KPT; ++i) Zf[xpos((int)oidx[i])] = oval[i];
        const uint32_t changed = s_changed;
        if (t == 0 && a.hist) a.hist[b * a.max_iter + (k - 1)] = (long long)changed;
        // ---- L6
        bool stop = changed == 0u;
        if (dm) {
            // Eq. 4 on chip: sum of squares in fp64, fixed order (per thread by ascending sample, warp tree, warps in order)
            __syncthreads();                    // x_sim,k+1 is complete in region A
            const T* xo = a.x + b * N;
            double acc = 0.0;
#pragma unroll
            for (int i = 0; i < KPT; ++i) {
                const int j = i * THREADS + t;
                const T xn = Zf[xpos(j)], xp = xo[j];
                if (xn != xp) {                 // an unchanged sample contributes log10(1) = 0 exactly: skip the division and the log
                    const double d = log10_ratio(xn, xp);
                    acc = fma(d, d, acc);
                }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
            if (lane == 0) red[warp] = acc;
            __syncthreads();
            if (t == 0) {
                double tot = 0.0;
                for (int w = 0; w < WARPS; ++w) tot += red[w];
                const double delta = sqrt(tot / (double)N);
                if (a.delta_hist) a.delta_hist[b * a.max_iter + (k - 1)] = delta;
                s_stop = (a.delta_threshold > 0.0 && delta <= a.delta_threshold) ? 1 : 0;
            }
            __syncthreads();
            stop = stop || s_stop != 0;
        }
        if (stop) { used = k; break; }
    }
    __syncthreads();
    // results: x_sim and the final permutation
    for (int j = t; j < N; j += THREADS) {
        a.x[b * N + j] = Zf[xpos(j)];
        pg[j] = (uint32_t)perm_s[j];
    }
    if (t == 0 && a.iters_used) a.iters_used[b] = used;
    }   // curve loop
}

inline bool onchip_applicable(size_t elem_size, long long N) {
    return N >= 256 && ((elem_size == 4 && N <= 16384) || (elem_size == 8 && N <= 8192));
}

template <typename T, int LOGN, bool DM> inline cudaError_t onchip_launch_dm(const OnchipArgs<T>& a, int slot, cudaStream_t st) {
    typedef OnchipCfg<T, LOGN> Cfg;
    int& grid = dev_cache().grid[slot];
    if (!grid) {
        cudaError_t e = cudaFuncSetAttribute(e13_onchip_kernel<T, LOGN, DM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::smem);
        if (e != cudaSuccess) return e;
        cudaFuncSetAttribute(e13_onchip_kernel<T, LOGN, DM>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        int per = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, e13_onchip_kernel<T, LOGN, DM>, Cfg::THREADS, Cfg::smem);
        if (e != cudaSuccess) return e;
        if (per < 1) return cudaErrorInvalidConfiguration;
        grid = dev_cache().sms * per;
    }
    const unsigned g = (unsigned)std::min<long long>(a.B, grid);
    AGN_LAUNCH(K_E13_ONCHIP, st, (e13_onchip_kernel<T, LOGN, DM><<<g, Cfg::THREADS, Cfg::smem, st>>>(a)));
    return cudaGetLastError();
}
// slot: dev_cache().grid index of the plain instantiation (3 .. 15); the delta instantiation keeps its own 13 slots above
template <typename T, int LOGN> inline cudaError_t onchip_launch(const OnchipArgs<T>& a, int slot, cudaStream_t st) {
    if (a.delta_hist != nullptr || a.delta_threshold > 0.0) return onchip_launch_dm<T, LOGN, true>(a, slot + 13, st);
    return onchip_launch_dm<T, LOGN, false>(a, slot, st);
}

template <typename T> inline cudaError_t onchip_run(int logN, const OnchipArgs<T>& a, cudaStream_t st) {
    constexpr int s0 = sizeof(T) == 4 ? 3 : 10;         // dev_cache().grid slots 3..9 (fp32), 10..15 (fp64)
    switch (logN) {
        case 8: return onchip_launch<T, 8>(a, s0, st);
        case 9: return onchip_launch<T, 9>(a, s0 + 1, st);
        case 10: return onchip_launch<T, 10>(a, s0 + 2, st);
        case 11: return onchip_launch<T, 11>(a, s0 + 3, st);
        case 12: return onchip_launch<T, 12>(a, s0 + 4, st);
        case 13: return onchip_launch<T, 13>(a, s0 + 5, st);
        case 14: if constexpr (sizeof(T) == 4) return onchip_launch<T, 14>(a, s0 + 6, st); else return cudaErrorInvalidValue;
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace agn

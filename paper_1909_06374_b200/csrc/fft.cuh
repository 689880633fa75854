// fft.cuh -- hand-written power-of-two complex FFT for sm_100a: shared-memory Stockham radix-8/4/2
// stages with register butterflies, composed into 1..3 passes over HBM.
//
// Decomposition (no transposes, no bit-reversal pass): L = R_0 * R_1 * ... * R_{P-1}.
//   forward pass i (decimation in frequency) works inside contiguous blocks of L_i = L / (R_0..R_{i-1})
//   viewed as [R_i][S_i], S_i = L_i / R_i:  for every column m:  V = FFT_{R_i}(v[.][m]);
//   V[k] *= w_{L_i}^{m k};  written back to [k][m].  The last pass has S = 1 (contiguous rows).
//   After all passes the element at mixed-radix position (k_0, k_1, .., k_{P-1}) (k_{P-1} fastest) holds
//   the DFT bin k = k_0 + R_0 k_1 + R_0 R_1 k_2 + ...  ("position order").
//   The inverse runs the mirror image (decimation in time): passes P-1..0, twiddle conj(w) applied on
//   load, and returns natural order.  Everything between a forward and an inverse transform
//   (amplitude replace, real-FFT untangle) is done in position order, so no reordering pass exists.
// DFT definition: Eq. A1 with the usual sign (forward e^{-2 pi i jk/N}), O5.
#pragma once
#include "common.cuh"

namespace agn {

constexpr int kLogTw = 14;        // fine table: exp(-2 pi i m / 2^14)
constexpr int kLogLo = 16;        // per-level low table: room for exp(-2 pi i l / D), l < 2^16; a level uses its first 2^lo_bits(logD) entries
__host__ __device__ __forceinline__ int lo_bits(int logD) { return logD - kLogTw > 13 ? logD - kLogTw : 13; }   // levels up to D = 2^30
constexpr int kMaxPass = 3;
constexpr int kFftThreads = 512;

constexpr int kMaxDigits = 6;
struct Digits {           // pass / stage radices (log2), forward order
    int n;
    int lg[kMaxDigits];
    int logL;
};

__host__ __device__ __forceinline__ uint32_t pos2k(const Digits& d, uint32_t pos) {
    int shift = d.logL;
    uint32_t k = 0;
    int ks = 0;
    for (int i = 0; i < d.n; ++i) {
        shift -= d.lg[i];
        uint32_t dig = (pos >> shift) & ((1u << d.lg[i]) - 1u);
        k |= dig << ks;
        ks += d.lg[i];
    }
    return k;
}
__host__ __device__ __forceinline__ uint32_t k2pos(const Digits& d, uint32_t k) {
    int shift = d.logL;
    uint32_t pos = 0;
    for (int i = 0; i < d.n; ++i) {
        shift -= d.lg[i];
        uint32_t dig = k & ((1u << d.lg[i]) - 1u);
        k >>= d.lg[i];
        pos |= dig << shift;
    }
    return pos;
}

// Twiddle level: w_D^idx = exp(-2 pi i idx / D), D = 2^logD <= 2^30, any idx < D.
template <typename T> struct TwLevel {
    const typename Cx<T>::type* tw14;   // exp(-2 pi i m / 2^14)
    const typename Cx<T>::type* lo;     // exp(-2 pi i l / D), l < 2^lo_bits(logD) (only if logD > kLogTw)
    int logD;
};

template <typename T>
__device__ __forceinline__ typename Cx<T>::type tw_lookup(const TwLevel<T>& lv, uint32_t idx) {
    if (lv.logD <= kLogTw) return lv.tw14[idx << (kLogTw - lv.logD)];
    const int lb = lo_bits(lv.logD);            // 13 up to D = 2^27 (64 KB of low table), logD - 14 above
    uint32_t h = idx >> lb, l = idx & ((1u << lb) - 1u);
    // exp(-2 pi i h 2^lb / D) = tw14[h * 2^kLogTw * 2^lb / D]
    return cmul(lv.tw14[h << (kLogTw + lb - lv.logD)], lv.lo[l]);
}

// table init: out[m] = exp(-2 pi i m / 2^logD), m < n
template <typename T>
__global__ void tw_init_kernel(typename Cx<T>::type* out, int n, int logD) {
    int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    double s, c;
    sincos_2pi_frac((uint64_t)m, logD, &s, &c);
    out[m] = mk<T>((T)c, (T)(-s));
}

// ------------------------------------------------------------------------------------------------
// register butterflies (forward sign).  Inverse transforms use swap(FFT(swap(x))).
// ------------------------------------------------------------------------------------------------
template <typename C> __device__ __forceinline__ void bfly2(C& a, C& b) {
    C t = csub(a, b); a = cadd(a, b); b = t;
}
// in: v0..v3 natural; out: X0..X3 natural
template <typename C> __device__ __forceinline__ void fft4(C& v0, C& v1, C& v2, C& v3) {
    C c0 = cadd(v0, v2), d0 = csub(v0, v2);
    C c1 = cadd(v1, v3), d1 = cmul_mi(csub(v1, v3));
    v0 = cadd(c0, c1); v2 = csub(c0, c1);
    v1 = cadd(d0, d1); v3 = csub(d0, d1);
}
template <typename T, typename C> __device__ __forceinline__ void fft8(C* v) {
    const T h = (T)0.70710678118654752440084436210485;
    C a0 = cadd(v[0], v[4]), b0 = csub(v[0], v[4]);
    C a1 = cadd(v[1], v[5]), b1 = csub(v[1], v[5]);
    C a2 = cadd(v[2], v[6]), b2 = csub(v[2], v[6]);
    C a3 = cadd(v[3], v[7]), b3 = csub(v[3], v[7]);
    // b_t *= w8^t
    C t1; t1.x = h * (b1.x + b1.y); t1.y = h * (b1.y - b1.x); b1 = t1;
    b2 = cmul_mi(b2);
    C t3; t3.x = h * (b3.y - b3.x); t3.y = -h * (b3.x + b3.y); b3 = t3;
    fft4(a0, a1, a2, a3);   // X0 X2 X4 X6
    fft4(b0, b1, b2, b3);   // X1 X3 X5 X7
    v[0] = a0; v[2] = a1; v[4] = a2; v[6] = a3;
    v[1] = b0; v[3] = b1; v[5] = b2; v[7] = b3;
}

// ------------------------------------------------------------------------------------------------
// One Stockham stage of radix RAD on a tile of C columns x R points held in shared memory.
// LAYOUT_A: element (n, c) at n*C + c        (lanes along c; used by strided passes, C >= 16)
// LAYOUT_B: element (n, c) at c*Rp + n + (n>>4), Rp = R + R/16   (lanes along n; contiguous rows)
// EPT = elements per thread (tile = THREADS*EPT elements).
// ------------------------------------------------------------------------------------------------
template <bool LAYB> __device__ __forceinline__ int phys_idx(int n, int c, int logC, int Rp) {
    if (LAYB) return c * Rp + n + (n >> 4);
    return (n << logC) + c;
}

template <typename T, int RAD, int THREADS, int EPT, bool LAYB>
__device__ __forceinline__ void fft_stage(typename Cx<T>::type* s, int logR, int logNs, int logC, int Rp,
                                          const typename Cx<T>::type* __restrict__ tw14) {
    typedef typename Cx<T>::type C;
    constexpr int NIT = EPT / RAD;
    constexpr int LOGRAD = (RAD == 8) ? 3 : (RAD == 4 ? 2 : 1);
    const int logRr = logR - LOGRAD;           // items per column
    const int Rr = 1 << logRr;
    const int Ns = 1 << logNs;
    C v[NIT][RAD];
    int jj[NIT], cc[NIT];
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
        int w = threadIdx.x + it * THREADS;
        int j, c;
        if (LAYB) { j = w & (Rr - 1); c = w >> logRr; }
        else { c = w & ((1 << logC) - 1); j = w >> logC; }
        jj[it] = j; cc[it] = c;
#pragma unroll
        for (int t = 0; t < RAD; ++t) v[it][t] = s[phys_idx<LAYB>(j + t * Rr, c, logC, Rp)];
        if (logNs > 0) {
            int k = j & (Ns - 1);
            // w_{Ns*RAD}^{k t} = tw14[k t 2^14/(Ns RAD)]
            int sh = kLogTw - logNs - LOGRAD;
            C w1 = tw14[k << sh];
            if (RAD == 2) {
                v[it][1] = cmul(v[it][1], w1);
            } else if (RAD == 4) {
                C w2 = tw14[(2 * k) << sh];
                C w3 = cmul(w1, w2);
                v[it][1] = cmul(v[it][1], w1); v[it][2] = cmul(v[it][2], w2); v[it][3] = cmul(v[it][3], w3);
            } else {
                C w2 = tw14[(2 * k) << sh];
                C w4 = tw14[(4 * k) << sh];
                C w3 = cmul(w1, w2), w5 = cmul(w1, w4), w6 = cmul(w2, w4);
                C w7 = cmul(w3, w4);
                v[it][1] = cmul(v[it][1], w1); v[it][2] = cmul(v[it][2], w2); v[it][3] = cmul(v[it][3], w3);
                v[it][4] = cmul(v[it][4], w4); v[it][5] = cmul(v[it][5], w5); v[it][6] = cmul(v[it][6], w6);
                v[it][7] = cmul(v[it][7], w7);
            }
        }
        if (RAD == 8) fft8<T, C>(v[it]);
        else if (RAD == 4) fft4(v[it][0], v[it][1], v[it][2], v[it][3]);
        else bfly2(v[it][0], v[it][1]);
    }
    __syncthreads();
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
        int j = jj[it], c = cc[it];
        int k = j & (Ns - 1);
        int base = ((j - k) << LOGRAD) + k;
#pragma unroll
        for (int t = 0; t < RAD; ++t) s[phys_idx<LAYB>(base + t * Ns, c, logC, Rp)] = v[it][t];
    }
    __syncthreads();
}

// full length-R FFT of every column of the tile (forward sign, natural in -> natural out)
template <typename T, int THREADS, int EPT, bool LAYB>
__device__ __forceinline__ void cta_fft(typename Cx<T>::type* s, int logR, int logC, int Rp,
                                        const typename Cx<T>::type* __restrict__ tw14) {
    int logNs = 0;
    while (logR - logNs >= 3) {
        fft_stage<T, 8, THREADS, EPT, LAYB>(s, logR, logNs, logC, Rp, tw14);
        logNs += 3;
    }
    if (logR - logNs == 2) fft_stage<T, 4, THREADS, EPT, LAYB>(s, logR, logNs, logC, Rp, tw14);
    else if (logR - logNs == 1) fft_stage<T, 2, THREADS, EPT, LAYB>(s, logR, logNs, logC, Rp, tw14);
}

// ------------------------------------------------------------------------------------------------
// pass kernel
// ------------------------------------------------------------------------------------------------
template <typename T> struct PassArgs {
    const typename Cx<T>::type* in;
    typename Cx<T>::type* out;
    long long bstride_in, bstride_out;   // per-transform stride (complex elements)
    int logL;        // transform length
    int nbatch;      // number of transforms addressed through grid y/z
    long long total; // contiguous pass: number of valid elements addressed by this grid row
    int logLi;       // block length of this pass
    int logR;        // radix of this pass
    int logC;        // columns (strided) or rows (contiguous) per CTA tile
    int inverse;     // 0: forward (twiddle on store), 1: inverse (conj twiddle on load, swap trick)
    T scale;         // applied on store
    TwLevel<T> lv;   // twiddle level for w_{L_i}
};

template <typename T, int THREADS, int EPT>
__global__ void __launch_bounds__(THREADS) fft_pass_kernel(PassArgs<T> a) {
    typedef typename Cx<T>::type C;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* s = reinterpret_cast<C*>(smem_raw);
    const int logS = a.logLi - a.logR;
    const int R = 1 << a.logR;
    const int logC = a.logC;
    const long long bb = bidx();
    if (bb >= a.nbatch) return;
    const C* __restrict__ in = a.in + bb * a.bstride_in;
    C* __restrict__ out = a.out + bb * a.bstride_out;
    const long long Ltot = a.total;
    if (logS == 0) {
        // contiguous rows: tile = 2^logC rows of R points; global element index = tile*E + e
        const int Rp = R + (R >> 4);
        const long long base = (long long)blockIdx.x * (THREADS * EPT);
#pragma unroll
        for (int i = 0; i < EPT; ++i) {
            int e = threadIdx.x + i * THREADS;
            int n = e & (R - 1), c = e >> a.logR;
            long long g = base + e;
            C v = mk<T>((T)0, (T)0);
            if (g < Ltot) v = in[g];
            if (a.inverse) v = cswap(v);
            s[phys_idx<true>(n, c, logC, Rp)] = v;
        }
        __syncthreads();
        cta_fft<T, THREADS, EPT, true>(s, a.logR, logC, Rp, a.lv.tw14);
#pragma unroll
        for (int i = 0; i < EPT; ++i) {
            int e = threadIdx.x + i * THREADS;
            int n = e & (R - 1), c = e >> a.logR;
            long long g = base + e;
            C v = s[phys_idx<true>(n, c, logC, Rp)];
            if (a.inverse) v = cswap(v);
            v.x *= a.scale; v.y *= a.scale;
            if (g < Ltot) out[g] = v;
        }
    } else {
        // strided: block o of length L_i viewed as [R][S]; tile = columns m0 .. m0 + C - 1
        const int Cn = 1 << logC;
        const int tiles_per_block = 1 << (logS - logC);
        const long long o = blockIdx.x >> (logS - logC);
        const int m0 = (int)(blockIdx.x & (tiles_per_block - 1)) << logC;
        const long long base = (o << a.logLi) + m0;
#pragma unroll
        for (int i = 0; i < EPT; ++i) {
            int e = threadIdx.x + i * THREADS;
            int c = e & (Cn - 1), n = e >> logC;
            C v = in[base + ((long long)n << logS) + c];
            if (a.inverse) {
                C w = tw_lookup<T>(a.lv, (uint32_t)(m0 + c) * (uint32_t)n);
                v = cswap(cmulc(v, w));
            }
            s[(n << logC) + c] = v;
        }
        __syncthreads();
        cta_fft<T, THREADS, EPT, false>(s, a.logR, logC, 0, a.lv.tw14);
#pragma unroll
        for (int i = 0; i < EPT; ++i) {
            int e = threadIdx.x + i * THREADS;
            int c = e & (Cn - 1), n = e >> logC;
            C v = s[(n << logC) + c];
            if (a.inverse) v = cswap(v);
            else v = cmul(v, tw_lookup<T>(a.lv, (uint32_t)(m0 + c) * (uint32_t)n));
            v.x *= a.scale; v.y *= a.scale;
            out[base + ((long long)n << logS) + c] = v;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// host-side plan
// ------------------------------------------------------------------------------------------------
template <typename T> struct FftCfg {
    static constexpr int EPT = (sizeof(T) == 4) ? 16 : 8;            // tile = 8192 (fp32) / 4096 (fp64) points = 64 KB
    static constexpr int logE = (sizeof(T) == 4) ? 13 : 12;
    static constexpr int maxStrided = logE - 4;                       // keep >= 16 columns per tile
};

template <typename T> struct FftPlan {
    typedef typename Cx<T>::type C;
    Digits dg;
    const C* tw14;
    const C* lo[kMaxPass];    // low tables of the pass levels that need one
    // untangle level (real FFT of length 2L)
    const C* lo_real;
    static size_t table_elems() { return ((size_t)1 << kLogTw) + (size_t)(kMaxPass + 1) * ((size_t)1 << kLogLo); }
};

template <typename T> inline Digits make_digits(int logL) {
    Digits d;
    d.logL = logL;
    const int logE = FftCfg<T>::logE, ms = FftCfg<T>::maxStrided;
    if (logL <= logE) { d.n = 1; d.lg[0] = logL; d.lg[1] = d.lg[2] = 0; }
    else if (logL <= logE - 1 + ms) {
        int last = logE - 1;                       // 2 rows per tile in the contiguous pass
        int r0 = logL - last;
        if (r0 < 3) { r0 = 3; last = logL - r0; }
        d.n = 2; d.lg[0] = r0; d.lg[1] = last; d.lg[2] = 0;
    } else {
        int last = logE - 2;
        int rest = logL - last;
        d.n = 3; d.lg[0] = (rest + 1) / 2; d.lg[1] = rest / 2; d.lg[2] = last;
    }
    return d;
}

// Build tables into `tables` (FftPlan<T>::table_elems() complex elements) and return the plan.
template <typename T>
inline FftPlan<T> fft_plan_init(int logL, typename Cx<T>::type* tables, cudaStream_t st) {
    typedef typename Cx<T>::type C;
    FftPlan<T> p;
    p.dg = make_digits<T>(logL);
    C* t = tables;
    AGN_LAUNCH(K_TABLES, st, (tw_init_kernel<T><<<(1 << kLogTw) / 256, 256, 0, st>>>(t, 1 << kLogTw, kLogTw)));
    p.tw14 = t; t += (size_t)1 << kLogTw;
    int logLi = logL;
    for (int i = 0; i < kMaxPass; ++i) {
        p.lo[i] = nullptr;
        if (i < p.dg.n) {
            if (logLi > kLogTw && i < p.dg.n - 1) {
                AGN_LAUNCH(K_TABLES, st, (tw_init_kernel<T><<<(1 << kLogLo) / 256, 256, 0, st>>>(t, 1 << kLogLo, logLi)));
                p.lo[i] = t;
            }
            logLi -= p.dg.lg[i];
        }
        t += (size_t)1 << kLogLo;
    }
    p.lo_real = nullptr;
    if (logL + 1 > kLogTw) {
        AGN_LAUNCH(K_TABLES, st, (tw_init_kernel<T><<<(1 << kLogLo) / 256, 256, 0, st>>>(t, 1 << kLogLo, logL + 1)));
        p.lo_real = t;
    }
    return p;
}

template <typename T> inline TwLevel<T> real_level(const FftPlan<T>& p) {
    TwLevel<T> lv; lv.tw14 = p.tw14; lv.lo = p.lo_real; lv.logD = p.dg.logL + 1; return lv;
}

template <typename T> inline size_t fft_smem_bytes(bool contiguous) {
    size_t e = (size_t)1 << FftCfg<T>::logE;
    if (contiguous) e += e >> 4;
    return e * sizeof(typename Cx<T>::type);
}

template <typename T> inline cudaError_t fft_set_attrs() {
    cudaFuncSetAttribute(fft_pass_kernel<T, kFftThreads, FftCfg<T>::EPT>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    return cudaFuncSetAttribute(fft_pass_kernel<T, kFftThreads, FftCfg<T>::EPT>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem_bytes<T>(true));
}

// One pass.  i = pass index in forward numbering.
template <typename T>
inline void fft_launch_pass(const FftPlan<T>& p, int i, bool inverse, const typename Cx<T>::type* in,
                            typename Cx<T>::type* out, long long bstride_in, long long bstride_out, int batch,
                            T scale, cudaStream_t st) {
    PassArgs<T> a;
    int logLi = p.dg.logL;
    for (int q = 0; q < i; ++q) logLi -= p.dg.lg[q];
    a.in = in; a.out = out; a.bstride_in = bstride_in; a.bstride_out = bstride_out;
    a.logL = p.dg.logL; a.logLi = logLi; a.logR = p.dg.lg[i];
    a.logC = FftCfg<T>::logE - a.logR;
    a.inverse = inverse ? 1 : 0;
    a.scale = scale;
    a.lv.tw14 = p.tw14; a.lv.lo = p.lo[i]; a.lv.logD = logLi;
    bool contiguous = (i == p.dg.n - 1);
    const long long Lc = 1ll << p.dg.logL;
    a.total = Lc;
    int gy = batch;
    if (contiguous && bstride_in == Lc && bstride_out == Lc) { a.total = Lc * batch; gy = 1; }   // dense batch: one row space
    long long tiles = (a.total + (1ll << FftCfg<T>::logE) - 1) >> FftCfg<T>::logE;
    a.nbatch = gy;
    dim3 grid = bgrid((unsigned)tiles, gy);
    AGN_LAUNCH((contiguous ? K_FFT_CONTIG : K_FFT_STRIDED), st, (fft_pass_kernel<T, kFftThreads, FftCfg<T>::EPT>
        <<<grid, kFftThreads, fft_smem_bytes<T>(contiguous), st>>>(a)));
}

// forward complex FFT: in (natural) -> out (position order).  in may equal out.
template <typename T>
inline void fft_forward(const FftPlan<T>& p, const typename Cx<T>::type* in, typename Cx<T>::type* out,
                        long long bstride_in, long long bstride_out, int batch, cudaStream_t st) {
    for (int i = 0; i < p.dg.n; ++i) {
        fft_launch_pass<T>(p, i, false, i == 0 ? in : out, out, i == 0 ? bstride_in : bstride_out, bstride_out,
                           batch, (T)1, st);
    }
}
// inverse complex FFT: in (position order) -> out (natural), scaled by `scale` (1/L for a true inverse)
template <typename T>
inline void fft_inverse(const FftPlan<T>& p, const typename Cx<T>::type* in, typename Cx<T>::type* out,
                        long long bstride_in, long long bstride_out, int batch, T scale, cudaStream_t st) {
    for (int i = p.dg.n - 1; i >= 0; --i) {
        bool first = (i == p.dg.n - 1), last = (i == 0);
        fft_launch_pass<T>(p, i, true, first ? in : out, out, first ? bstride_in : bstride_out, bstride_out,
                           batch, last ? scale : (T)1, st);
    }
}

}  // namespace agn

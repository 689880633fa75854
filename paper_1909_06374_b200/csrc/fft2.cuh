// fft2.cuh -- the E13 loop's FFT for long fp32 curves (L = N/2 >= 2^14 complex points per curve):
//   L = R0 * R1,  R1 = 2^13 contiguous "rows", R0 = L / R1 split into 1..3 column sub-passes of radix <= 64.
//
//   fft_col_kernel   one persistent launch runs ALL column sub-passes of one direction.  A thread owns one
//                    column and does a radix-2^k butterfly entirely in registers (fft_reg.cuh): no shared
//                    memory, every global access is a full coalesced row segment.  Sub-pass e+1 of a column
//                    group starts when sub-pass e of that group is complete (per-group counters, tickets
//                    handed out in dependency order), so the intermediate is re-read from L2 (a group is a
//                    few MB), and the whole column transform costs one HBM read + one HBM write.
//   fft_mid_kernel   one CTA per row pair (k0, R0-k0): forward row FFT in shared memory, real-FFT untangle
//                    + amplitude replace (L2 of the paper's path, O6 step 2) on the pairs (K, L-K), which
//                    live in the two rows, inverse row FFT.  Read Z once, write Z' once.
// Bin K = k0 + R0 k sits at row rowpos(k0), position p with k = digit-reversal of p ("position order");
// nothing is ever un-permuted: A_norm is permuted once (perm_anorm_kernel) and the inverse mirrors the forward.
// HBM bytes per real sample and iteration: 8 (columns fwd) + 10 (mid) + 8 (columns inv) = 26.
#pragma once
#include "common.cuh"
#include "fft.cuh"
#include "fft_reg.cuh"
#include "kernels.cuh"

namespace agn {

constexpr int kLogR1 = 13;              // row length of the mid kernel
constexpr int kColThreads = 128;        // columns per column tile
constexpr int kMaxColPhases = 3;
constexpr int kColMaxLog = 6;            // largest column radix (log2): radix 64 in registers, 2 sub-passes for N = 2^26 (radix 16 with 3 sub-passes and 3.5x the warps measured 12 % slower)

// ------------------------------------------------------------------------------------------------
// column sub-passes
// ------------------------------------------------------------------------------------------------
template <typename T> struct ColArgs {
    typedef typename Cx<T>::type C;
    const C* in;                  // read by stage 0 only (may differ from out)
    C* out;                       // stages >= 1 work in place on out
    long long bstride_in, bstride_out;
    int B, logS, G, nph, D;       // curves; log2 row length; column groups per curve; stages; pipeline distance
    int logRad[kMaxColPhases];    // by stage, in execution order
    int logStr[kMaxColPhases];    // log2 of the butterfly stride (elements)
    int tiles[kMaxColPhases];     // tiles per (group, stage) = R0 / radix
    int prefix[kMaxColPhases + 1];
    TwLevel<T> lv[kMaxColPhases]; // twiddle level w_{radix * stride}
    int inverse;
    T scale;                      // applied by the last stage
    unsigned int* ticket;         // zero on entry
    unsigned int* done;           // [B*G][nph], zero on entry
    unsigned int total;           // number of tickets
};

template <typename T, int LOGRAD, int THREADS>
__device__ __forceinline__ void col_tile(const ColArgs<T>& a, int e, int b, int g, int q) {
    typedef typename Cx<T>::type C;
    constexpr int RAD = 1 << LOGRAD;
    const int logStr = a.logStr[e];
    const int lo = q & ((1 << (logStr - a.logS)) - 1), hi = q >> (logStr - a.logS);
    const uint32_t col = ((uint32_t)lo << a.logS) + (uint32_t)(g * THREADS + threadIdx.x);
    const long long base = ((long long)hi << (LOGRAD + logStr)) + col;
    const C* __restrict__ src = (e == 0 ? a.in + (long long)b * a.bstride_in : a.out + (long long)b * a.bstride_out) + base;
    C* __restrict__ dst = a.out + (long long)b * a.bstride_out + base;
    const bool last = (e == a.nph - 1);
    C v[RAD];
    if (e == 0) {
#pragma unroll
        for (int i = 0; i < RAD; ++i) v[i] = __ldcs(src + ((long long)i << logStr));
    } else {
#pragma unroll
        for (int i = 0; i < RAD; ++i) v[i] = __ldcg(src + ((long long)i << logStr));   // written by other SMs: L2
    }
    // twiddle powers of w = w_{RAD*stride}^{col}: w^k = W8[k >> 3] * W1[k & 7]
    C W1[8], W8[8];
    pow8<T, C>(tw_lookup<T>(a.lv[e], col), W1);
    if (RAD > 8) pow8<T, C>(tw_lookup<T>(a.lv[e], col << 3), W8);
    if (!a.inverse) {
        fft_reg_dif<T, RAD, C>(v);
#pragma unroll
        for (int k = 0; k < RAD; ++k) {
            C x = v[bitrev<RAD>(k)];
            if (k > 0) {
                if (k < 8) x = cmul(x, W1[k]);
                else if ((k & 7) == 0) x = cmul(x, W8[k >> 3]);
                else x = cmul(x, cmul(W8[k >> 3], W1[k & 7]));
            }
            if (last) { x.x *= a.scale; x.y *= a.scale; }
            if (last) __stcs(dst + ((long long)k << logStr), x);
            else dst[(long long)k << logStr] = x;
        }
    } else {
#pragma unroll
        for (int k = 0; k < RAD; ++k) {
            C x = v[k];
            if (k > 0) {
                if (k < 8) x = cmulc(x, W1[k]);
                else if ((k & 7) == 0) x = cmulc(x, W8[k >> 3]);
                else x = cmulc(x, cmul(W8[k >> 3], W1[k & 7]));
            }
            v[k] = cswap(x);
        }
        fft_reg_dif<T, RAD, C>(v);
#pragma unroll
        for (int n = 0; n < RAD; ++n) {
            C x = cswap(v[bitrev<RAD>(n)]);
            if (last) { x.x *= a.scale; x.y *= a.scale; }
            if (last) __stcs(dst + ((long long)n << logStr), x);
            else dst[(long long)n << logStr] = x;
        }
    }
}

// MAXLOG: largest radix (log2) this instantiation can run; the register budget follows it (radix 64: 164 registers,
// 3 CTAs per SM -- measured 0.71 ms per direction against 0.78 with 255 registers / 2 CTAs and 0.84 with 128 / 4 and spills)
template <typename T, int THREADS, int MAXLOG>
__global__ void __launch_bounds__(THREADS, (MAXLOG >= 6 ? 3 : (MAXLOG == 5 ? 4 : 5))) fft_col_kernel(ColArgs<T> a) {
    __shared__ unsigned int s_ticket;
    const int slots = a.prefix[a.nph];
    const int nsg = a.B * a.G;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_ticket = atomicAdd(a.ticket, 1u);
        __syncthreads();
        const unsigned int t = s_ticket;
        if (t >= a.total) break;
        const int s = (int)(t / (unsigned)slots), r = (int)(t % (unsigned)slots);
        int e = 0;
        while (e + 1 < a.nph && r >= a.prefix[e + 1]) ++e;
        const int q = r - a.prefix[e];
        const int sg = s - e * a.D;
        if (sg < 0 || sg >= nsg) continue;
        const int b = sg / a.G, g = sg - b * a.G;
        if (e > 0) {
            if (threadIdx.x == 0) {
                volatile unsigned int* d = a.done + (size_t)sg * a.nph + (e - 1);
                const unsigned int need = (unsigned)a.tiles[e - 1];
                while (*d < need) __nanosleep(64);
                __threadfence();
            }
            __syncthreads();
        }
        switch (a.logRad[e]) {
            case 6: if constexpr (MAXLOG >= 6) col_tile<T, 6, THREADS>(a, e, b, g, q); break;
            case 5: if constexpr (MAXLOG >= 5) col_tile<T, 5, THREADS>(a, e, b, g, q); break;
            case 4: col_tile<T, 4, THREADS>(a, e, b, g, q); break;
            case 3: col_tile<T, 3, THREADS>(a, e, b, g, q); break;
            case 2: col_tile<T, 2, THREADS>(a, e, b, g, q); break;
            default: col_tile<T, 1, THREADS>(a, e, b, g, q); break;
        }
        if (e + 1 < a.nph) {
            __threadfence();
            __syncthreads();
            if (threadIdx.x == 0) atomicAdd(a.done + (size_t)sg * a.nph + e, 1u);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// mid kernel: rows of R1 = 2^13 = 16 * 16 * 32, two rows per CTA, 512 threads
// Rows (64 KB, contiguous in HBM) and their target amplitudes (32 KB) arrive by BULK ASYNCHRONOUS COPIES
// (cp.async.bulk global -> shared, completion on an mbarrier): one elected thread issues one copy per row, no LSU
// instruction and no register is spent on the transfer, and the copy of the next work item's rows overlaps the
// last butterflies and the stores of the current one.  A bulk copy lands linearly, so the rows are not padded:
// bank conflicts are avoided by an XOR swizzle of the low five index bits with the next five (mid_swz), which
// forward stage 1 applies on its write (it reads the linear landing layout, conflict-free as it is; a warp only ever
// touches its own sixteen 32-element groups in that stage, so the linear -> swizzled rewrite is safe in place).
// ------------------------------------------------------------------------------------------------
constexpr int kMidThreads = 512;
constexpr int kMidL1 = 4, kMidL2 = 4, kMidL3 = 5;        // log2 of the stage radices
__host__ __device__ constexpr int mid_swz(int a) { return a ^ ((a >> 5) & 31); }
constexpr int kMidRowElems = 1 << kLogR1;
constexpr size_t kMidSmemBytes = 2 * (size_t)kMidRowElems * sizeof(float2) + 2 * ((size_t)1 << kLogR1) * sizeof(float);   // rows + their A_norm

template <typename T> struct MidArgs {
    typedef typename Cx<T>::type C;
    C* Z;                         // [B][L] in place
    long long bstride;            // L
    int B, logR0;
    Digits dcol;                  // digits of the row index (column sub-pass radices), logL = logR0
    const T* Ap;                  // [B][L+1] target amplitudes in position order (entry L = Nyquist bin)
    const C* twpos;               // [R1] w_{2 R1}^{k(p)} in position order
    const unsigned short* sp;     // [R1] position of bin (R1 - k(p)) mod R1
    const C* tw14;
    TwLevel<T> rlv;               // w_N (N = 2L) for the row factor w_N^{k0}
};

// mbarrier + bulk-copy primitives (sm_90+ PTX; SASS: SYNCS.* and UBLKCP)
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(a), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"((unsigned)__cvta_generic_to_shared(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(bar))
                 : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }

template <typename T>
__global__ void __launch_bounds__(kMidThreads, 1) fft_mid_kernel(MidArgs<T> a) {
    typedef typename Cx<T>::type C;
    static_assert(sizeof(T) == 4, "fp32 rows");
    constexpr int R1 = 1 << kLogR1;
    constexpr int RAD1 = 1 << kMidL1, RAD2 = 1 << kMidL2, RAD3 = 1 << kMidL3;
    constexpr int J1 = R1 / RAD1;                 // 512 butterflies per row in stages 1 and 2
    constexpr int LOG23 = kMidL2 + kMidL3;
    constexpr unsigned kRowBytes = R1 * sizeof(C), kAmpBytes = R1 * sizeof(T);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C* s = reinterpret_cast<C*>(smem_raw);
    __shared__ C s_wrow[2];
    __shared__ __align__(8) unsigned long long s_bar[3];      // row 0, row 1, amplitudes
    const int t = threadIdx.x;
    const int R0 = 1 << a.logR0;
    const int nrows = (R0 == 1) ? 1 : 2;
    const int gx = (R0 == 1) ? 1 : (R0 >> 1);
    const long long total = (long long)a.B * gx;
    T* sA = reinterpret_cast<T*>(smem_raw + 2 * (size_t)kMidRowElems * sizeof(C));
    // Persistent CTA (one per SM: 192 KB of shared memory): work item = (curve b, row pair pid).
    auto row_pos = [&](int pid, int r) -> int {
        const int k = (r == 0) ? pid : ((pid == 0) ? (R0 >> 1) : (R0 - pid));
        return (R0 == 1) ? 0 : (int)k2pos(a.dcol, (uint32_t)k);
    };
    // issued by thread 0 only, after a CTA barrier that follows the last generic-proxy access to the destination
    auto fetch_row = [&](long long bb, int rp_, int r) {
        fence_proxy_async();
        mbar_expect_tx(&s_bar[r], kRowBytes);
        bulk_g2s(s + r * kMidRowElems, a.Z + bb * a.bstride + ((long long)rp_ << kLogR1), kRowBytes, &s_bar[r]);
    };
    auto fetch_amps = [&](long long bb, int pid_) {
        fence_proxy_async();
        mbar_expect_tx(&s_bar[2], kAmpBytes * (unsigned)nrows);
        for (int r = 0; r < nrows; ++r)
            bulk_g2s(sA + r * R1, a.Ap + bb * (a.bstride + kApPad) + ((long long)row_pos(pid_, r) << kLogR1), kAmpBytes, &s_bar[2]);
    };
    long long work = blockIdx.x;
    if (work >= total) return;
    if (t == 0) {
        mbar_init(&s_bar[0], 1); mbar_init(&s_bar[1], 1); mbar_init(&s_bar[2], 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();
    if (t == 0) {
        const long long b0 = work / gx;
        const int pid0 = (int)(work - b0 * gx);
        for (int r = 0; r < nrows; ++r) fetch_row(b0, row_pos(pid0, r), r);
        fetch_amps(b0, pid0);
    }
    unsigned phase = 0;
    for (; work < total; work += gridDim.x, phase ^= 1u) {
    const long long b = work / gx;
    const int pid = (int)(work - b * gx);         // 0: rows 0 and R0/2 (self-paired); else rows pid, R0 - pid
    const long long work_n = work + gridDim.x;
    const bool has_next = work_n < total;
    const long long b_n = has_next ? work_n / gx : 0;
    const int pid_n = has_next ? (int)(work_n - b_n * gx) : 0;
    int k0[2], rp[2];
    k0[0] = pid; k0[1] = (pid == 0) ? (R0 >> 1) : (R0 - pid);
    rp[0] = (int)k2pos(a.dcol, (uint32_t)k0[0]);
    rp[1] = (R0 == 1) ? 0 : (int)k2pos(a.dcol, (uint32_t)k0[1]);
    C* zrow[2];
    zrow[0] = a.Z + b * a.bstride + ((long long)rp[0] << kLogR1);
    zrow[1] = a.Z + b * a.bstride + ((long long)rp[1] << kLogR1);
    if (t < 2) s_wrow[t] = tw_lookup<T>(a.rlv, (uint32_t)(t == 0 ? k0[0] : k0[1]));      // no dynamic index: k0 stays in registers
    C pw[16];

    // ---- forward stage 1: thread j = t owns (d2, d3) = j, butterfly over d1 (stride J1).  Reads the LINEAR landing
    //      layout, writes the swizzled working layout (same 32-element groups: private to this warp).
    pow16<T, C>(a.tw14[t << (kLogTw - kLogR1)], pw);
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        if (r < nrows) {
            mbar_wait(&s_bar[r], phase);          // this item's row r has landed
            C v[RAD1];
#pragma unroll
            for (int i = 0; i < RAD1; ++i) v[i] = s[r * kMidRowElems + i * J1 + t];
            __syncwarp();
            fft_reg_dif<T, RAD1, C>(v);
#pragma unroll
            for (int k = 0; k < RAD1; ++k) {
                C x = v[bitrev<RAD1>(k)];
                if (k > 0) x = cmul(x, pw[k]);
                s[r * kMidRowElems + mid_swz(k * J1 + t)] = x;
            }
        }
    }
    __syncthreads();
    // ---- forward stage 2: thread (k1, d3), butterfly over d2 (stride RAD3), in place
    const int k1 = t >> kMidL3, d3 = t & (RAD3 - 1);
    pow16<T, C>(a.tw14[d3 << (kLogTw - LOG23)], pw);
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        if (r < nrows) {
            C v[RAD2];
            C* sr = s + r * kMidRowElems;
#pragma unroll
            for (int i = 0; i < RAD2; ++i) v[i] = sr[mid_swz((k1 << LOG23) + (i << kMidL3) + d3)];
            fft_reg_dif<T, RAD2, C>(v);
#pragma unroll
            for (int k = 0; k < RAD2; ++k) {
                C x = v[bitrev<RAD2>(k)];
                if (k > 0) x = cmul(x, pw[k]);
                sr[mid_swz((k1 << LOG23) + (k << kMidL3) + d3)] = x;
            }
        }
    }
    __syncthreads();
    // ---- forward stage 3: thread (row, u = (k1, k2)), butterfly over d3 (stride 1), in place
    const int r3 = t >> (kLogR1 - kMidL3), u = t & ((R1 >> kMidL3) - 1);
    if (r3 < nrows) {
        C v[RAD3];
        C* sr = s + r3 * kMidRowElems + u * RAD3;              // group u: element i sits at i ^ (u & 31)
        const int x5 = u & (RAD3 - 1);
#pragma unroll
        for (int i = 0; i < RAD3; ++i) v[i] = sr[i ^ x5];
        fft_reg_dif<T, RAD3, C>(v);
#pragma unroll
        for (int k = 0; k < RAD3; ++k) sr[k ^ x5] = v[bitrev<RAD3>(k)];
    }
    __syncthreads();
    // ---- L2: untangle + amplitude replace on the pairs (K, L - K)
    mbar_wait(&s_bar[2], phase);                  // the amplitudes of this item have landed
    {
        const T* Ab = a.Ap + b * (a.bstride + kApPad);
        if (pid != 0) {
            // bin k of row A pairs with bin R1-1-k of row B: position p <-> R1-1-p
            const C wrow = s_wrow[0];
            const T* A1p = sA;
            const T* A2p = sA + R1;
#pragma unroll 4
            for (int p = t; p < R1; p += kMidThreads) {
                const int p2 = R1 - 1 - p;
                C z1 = s[mid_swz(p)], z2 = s[kMidRowElems + mid_swz(p2)];
                replace_pair<T>(z1, z2, cmul(wrow, a.twpos[p]), A1p[p], A2p[p2]);
                s[mid_swz(p)] = z1;
                s[kMidRowElems + mid_swz(p2)] = z2;
            }
        } else {
            // row 0: bin k pairs with (R1 - k) mod R1 (table sp); k = 0 holds DC and Nyquist
            const T* A1p = sA;
            for (int p = t; p < R1; p += kMidThreads) {
                const int p2 = a.sp[p];
                if (p2 < p) continue;
                if (p == 0) {
                    C z0 = s[0];
                    T x0 = z0.x + z0.y, xl = z0.x - z0.y;
                    T a0 = A1p[0], al = Ab[a.bstride];
                    T y0 = (x0 != (T)0) ? (x0 > (T)0 ? a0 : -a0) : a0;
                    T yl = (xl != (T)0) ? (xl > (T)0 ? al : -al) : al;
                    s[0] = mk<T>((T)0.5 * (y0 + yl), (T)0.5 * (y0 - yl));
                } else {
                    C z1 = s[mid_swz(p)], z2 = s[mid_swz(p2)];
                    replace_pair<T>(z1, z2, a.twpos[p], A1p[p], A1p[p2]);       // w_N^{0} = 1
                    s[mid_swz(p)] = z1;
                    s[mid_swz(p2)] = z2;
                }
            }
            if (nrows == 2) {
                // row R0/2 pairs with itself: position p <-> R1-1-p
                const C wrow = s_wrow[1];
                const T* A2p = sA + R1;
                C* sr = s + kMidRowElems;
                for (int p = t; p < R1 / 2; p += kMidThreads) {
                    const int p2 = R1 - 1 - p;
                    C z1 = sr[mid_swz(p)], z2 = sr[mid_swz(p2)];
                    replace_pair<T>(z1, z2, cmul(wrow, a.twpos[p]), A2p[p], A2p[p2]);
                    sr[mid_swz(p)] = z1;
                    sr[mid_swz(p2)] = z2;
                }
            }
        }
    }
    __syncthreads();
    if (has_next && t == 0) fetch_amps(b_n, pid_n);        // sA is free now
    // ---- inverse stage 3
    if (r3 < nrows) {
        C v[RAD3];
        C* sr = s + r3 * kMidRowElems + u * RAD3;
        const int x5 = u & (RAD3 - 1);
#pragma unroll
        for (int i = 0; i < RAD3; ++i) v[i] = cswap(sr[i ^ x5]);
        fft_reg_dif<T, RAD3, C>(v);
#pragma unroll
        for (int n = 0; n < RAD3; ++n) sr[n ^ x5] = cswap(v[bitrev<RAD3>(n)]);
    }
    __syncthreads();
    // ---- inverse stage 2 (pw still holds w_{512}^{k d3})
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        if (r < nrows) {
            C v[RAD2];
            C* sr = s + r * kMidRowElems;
#pragma unroll
            for (int k = 0; k < RAD2; ++k) {
                C x = sr[mid_swz((k1 << LOG23) + (k << kMidL3) + d3)];
                if (k > 0) x = cmulc(x, pw[k]);
                v[k] = cswap(x);
            }
            fft_reg_dif<T, RAD2, C>(v);
#pragma unroll
            for (int n = 0; n < RAD2; ++n) sr[mid_swz((k1 << LOG23) + (n << kMidL3) + d3)] = cswap(v[bitrev<RAD2>(n)]);
        }
    }
    __syncthreads();
    // ---- inverse stage 1: results go straight from registers to HBM; as soon as every thread has read its inputs of
    //      row r, the bulk copy of the next item's row r is started (it overlaps the butterflies and stores that follow)
    pow16<T, C>(a.tw14[t << (kLogTw - kLogR1)], pw);
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        if (r < nrows) {
            C v[RAD1];
#pragma unroll
            for (int k = 0; k < RAD1; ++k) {
                C x = s[r * kMidRowElems + mid_swz(k * J1 + t)];
                if (k > 0) x = cmulc(x, pw[k]);
                v[k] = cswap(x);
            }
            __syncthreads();
            if (has_next && t == 0) fetch_row(b_n, row_pos(pid_n, r), r);
            fft_reg_dif<T, RAD1, C>(v);
#pragma unroll
            for (int n = 0; n < RAD1; ++n) zrow[r][n * J1 + t] = cswap(v[bitrev<RAD1>(n)]);
        }
    }
    }   // work loop
}

// ------------------------------------------------------------------------------------------------
// tables of the mid kernel: twpos[p] = w_{2 R1}^{k(p)}, sp[p] = position of bin (R1 - k(p)) mod R1
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void mid_tables_kernel(typename Cx<T>::type* __restrict__ twpos, unsigned short* __restrict__ sp, Digits d3) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= (1 << kLogR1)) return;
    const uint32_t k = pos2k(d3, (uint32_t)p);
    double sn, cs;
    sincos_2pi_frac((uint64_t)k, kLogR1 + 1, &sn, &cs);
    twpos[p] = mk<T>((T)cs, (T)(-sn));
    sp[p] = (unsigned short)k2pos(d3, ((1u << kLogR1) - k) & ((1u << kLogR1) - 1u));
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
template <typename T> struct Fft2Plan {
    typedef typename Cx<T>::type C;
    int logL, logR0, nph;
    int logRad[kMaxColPhases];          // forward order (phase 0 has the largest stride)
    Digits dfull;                       // position -> bin digits of the whole length-L transform
    Digits dcol;                        // row index digits
    const C* tw14;
    const C* lo[kMaxColPhases];         // low tables of the column levels with D > 2^14
    const C* lo_real;
    const C* twpos;
    const unsigned short* sp;
    unsigned int* counters;             // [1 + B*G*nph] ticket + done
    static size_t table_elems() {
        return ((size_t)1 << kLogTw) + (size_t)(kMaxColPhases + 1) * ((size_t)1 << kLogLo) + ((size_t)1 << kLogR1) +
               ((size_t)1 << (kLogR1 - 2));
    }
    static size_t counter_words(long long B) {
        return 1 + (size_t)B * ((size_t)1 << kLogR1) / kColThreads * kMaxColPhases;
    }
};

inline bool fft2_applicable(size_t elem_size, int logL) { return elem_size == 4 && logL >= kLogR1 + 1 && logL <= kLogR1 + 16; }   // N = 2^15 .. 2^30 (three column phases of radix <= 64 reach R0 = 2^18)

template <typename T>
inline Fft2Plan<T> fft2_plan_init(int logL, typename Cx<T>::type* tables, unsigned int* counters, cudaStream_t st) {
    typedef typename Cx<T>::type C;
    Fft2Plan<T> p;
    p.logL = logL;
    p.logR0 = logL - kLogR1;
    p.nph = (p.logR0 + kColMaxLog - 1) / kColMaxLog;
    if (p.nph > kMaxColPhases) p.nph = kMaxColPhases;
    {
        int base = p.logR0 / p.nph, extra = p.logR0 % p.nph;
        for (int i = 0; i < kMaxColPhases; ++i) p.logRad[i] = (i < p.nph) ? base + (i < extra ? 1 : 0) : 0;
    }
    p.dcol.n = p.nph; p.dcol.logL = p.logR0;
    p.dfull.n = p.nph + 3; p.dfull.logL = logL;
    for (int i = 0; i < kMaxDigits; ++i) { p.dcol.lg[i] = 0; p.dfull.lg[i] = 0; }
    for (int i = 0; i < p.nph; ++i) { p.dcol.lg[i] = p.logRad[i]; p.dfull.lg[i] = p.logRad[i]; }
    p.dfull.lg[p.nph] = kMidL1; p.dfull.lg[p.nph + 1] = kMidL2; p.dfull.lg[p.nph + 2] = kMidL3;
    C* t = tables;
    AGN_LAUNCH(K_TABLES, st, (tw_init_kernel<T><<<(1 << kLogTw) / 256, 256, 0, st>>>(t, 1 << kLogTw, kLogTw)));
    p.tw14 = t; t += (size_t)1 << kLogTw;
    int logStr = logL;
    for (int i = 0; i < kMaxColPhases; ++i) {
        p.lo[i] = nullptr;
        if (i < p.nph) {
            const int logD = logStr;                 // block length of phase i = radix * stride
            if (logD > kLogTw) {
                AGN_LAUNCH(K_TABLES, st, (tw_init_kernel<T><<<(1 << kLogLo) / 256, 256, 0, st>>>(t, 1 << kLogLo, logD)));
                p.lo[i] = t;
            }
            logStr -= p.logRad[i];
        }
        t += (size_t)1 << kLogLo;
    }
    AGN_LAUNCH(K_TABLES, st, (tw_init_kernel<T><<<(1 << kLogLo) / 256, 256, 0, st>>>(t, 1 << kLogLo, logL + 1)));
    p.lo_real = t; t += (size_t)1 << kLogLo;
    Digits d3; d3.n = 3; d3.logL = kLogR1;
    for (int i = 0; i < kMaxDigits; ++i) d3.lg[i] = 0;
    d3.lg[0] = kMidL1; d3.lg[1] = kMidL2; d3.lg[2] = kMidL3;
    C* twpos = t; t += (size_t)1 << kLogR1;
    unsigned short* sp = (unsigned short*)t;
    AGN_LAUNCH(K_TABLES, st, (mid_tables_kernel<T><<<(1 << kLogR1) / 256, 256, 0, st>>>(twpos, sp, d3)));
    p.twpos = twpos; p.sp = sp;
    p.counters = counters;
    return p;
}

template <typename T> inline cudaError_t fft2_set_attrs() {
    cudaFuncSetAttribute(fft_mid_kernel<T>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    return cudaFuncSetAttribute(fft_mid_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMidSmemBytes);
}

inline int fft2_col_grid(const void* func, int threads, int slot) {
    int& cached = dev_cache().grid[slot];
    if (cached) return cached;
    int per = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per, func, threads, 0);
    if (per < 1) per = 1;
    cached = dev_cache().sms * per;
    return cached;
}

// all column sub-passes of one direction, one persistent launch.  forward: in (natural) -> out; inverse: in place on out.
template <typename T>
inline cudaError_t fft2_columns(const Fft2Plan<T>& p, bool inverse, const typename Cx<T>::type* in,
                                typename Cx<T>::type* out, int B, T scale, cudaStream_t st) {
    ColArgs<T> a;
    const long long L = 1ll << p.logL;
    a.in = in; a.out = out; a.bstride_in = L; a.bstride_out = L;
    a.B = B; a.logS = kLogR1; a.G = (1 << kLogR1) / kColThreads; a.nph = p.nph; a.D = 2;
    a.inverse = inverse ? 1 : 0; a.scale = scale;
    int logStrF[kMaxColPhases], logStr = p.logL;
    for (int i = 0; i < p.nph; ++i) { logStr -= p.logRad[i]; logStrF[i] = logStr; }
    a.prefix[0] = 0;
    for (int e = 0; e < kMaxColPhases; ++e) {
        if (e < p.nph) {
            const int i = inverse ? p.nph - 1 - e : e;
            a.logRad[e] = p.logRad[i]; a.logStr[e] = logStrF[i];
            a.tiles[e] = 1 << (p.logR0 - p.logRad[i]);
            a.lv[e].tw14 = p.tw14; a.lv[e].lo = p.lo[i]; a.lv[e].logD = p.logRad[i] + logStrF[i];
            a.prefix[e + 1] = a.prefix[e] + a.tiles[e];
        } else {
            a.logRad[e] = 0; a.logStr[e] = 0; a.tiles[e] = 0; a.lv[e] = a.lv[0]; a.prefix[e + 1] = a.prefix[e];
        }
    }
    const size_t words = 1 + (size_t)B * a.G * p.nph;
    cudaError_t e = cudaMemsetAsync(p.counters, 0, words * sizeof(unsigned int), st);
    if (e != cudaSuccess) return e;
    a.ticket = p.counters; a.done = p.counters + 1;
    a.total = (unsigned)((B * a.G + (p.nph - 1) * a.D) * a.prefix[p.nph]);
    int maxlog = 0;
    for (int i = 0; i < p.nph; ++i) maxlog = std::max(maxlog, p.logRad[i]);
    if (maxlog <= 4) {
        const int grid = fft2_col_grid((const void*)fft_col_kernel<T, kColThreads, 4>, kColThreads, 0);
        AGN_LAUNCH(K_FFT_COL, st, (fft_col_kernel<T, kColThreads, 4><<<grid, kColThreads, 0, st>>>(a)));
    } else if (maxlog == 5) {
        const int grid = fft2_col_grid((const void*)fft_col_kernel<T, kColThreads, 5>, kColThreads, 1);
        AGN_LAUNCH(K_FFT_COL, st, (fft_col_kernel<T, kColThreads, 5><<<grid, kColThreads, 0, st>>>(a)));
    } else {
        const int grid = fft2_col_grid((const void*)fft_col_kernel<T, kColThreads, 6>, kColThreads, 2);
        AGN_LAUNCH(K_FFT_COL, st, (fft_col_kernel<T, kColThreads, 6><<<grid, kColThreads, 0, st>>>(a)));
    }
    return cudaGetLastError();
}

template <typename T>
inline cudaError_t fft2_mid(const Fft2Plan<T>& p, typename Cx<T>::type* Z, const T* Ap, int B, cudaStream_t st) {
    MidArgs<T> m;
    m.Z = Z; m.bstride = 1ll << p.logL; m.B = B; m.logR0 = p.logR0; m.dcol = p.dcol; m.Ap = Ap;
    m.twpos = p.twpos; m.sp = p.sp; m.tw14 = p.tw14;
    m.rlv.tw14 = p.tw14; m.rlv.lo = p.lo_real; m.rlv.logD = p.logL + 1;
    const unsigned gx = p.logR0 == 0 ? 1u : (1u << (p.logR0 - 1));
    const int sms = dev_cache().sms;
    const unsigned grid = (unsigned)std::min<long long>((long long)gx * B, sms);
    AGN_LAUNCH(K_FFT_MID, st, (fft_mid_kernel<T><<<grid, kMidThreads, kMidSmemBytes, st>>>(m)));
    return cudaGetLastError();
}

}  // namespace agn

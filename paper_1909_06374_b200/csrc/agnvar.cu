// agnvar.cu -- C ABI (include/agnvar.h) of the B200-native E13 light-curve generator.
// Host side: argument validation, workspace carving, kernel sequencing on the caller's stream.
// Every step of the path runs in the kernels of fft.cuh / sort.cuh / kernels.cuh; there is no CPU
// fallback and no vendor FFT / sort library call.
#include "../../include/agnvar.h"
#include "common.cuh"
#include "fft.cuh"
#include "sort.cuh"
#include "kernels.cuh"
#include "fft2.cuh"
#include "sort32.cuh"
#include "sf.cuh"
#include "onchip.cuh"
#include "slice.cuh"

#include <cmath>
#include <cstring>
#include <mutex>
#include <vector>

using namespace agn;

namespace {

struct Carver {
    unsigned char* base;
    size_t off;
    explicit Carver(void* p) : base((unsigned char*)p), off(0) {}
    template <typename U> U* take(size_t count) {
        U* r = base ? (U*)(base + off) : nullptr;
        off += align_up(count * sizeof(U), 256);
        return r;
    }
};

inline bool is_pow2(int64_t n) { return n > 0 && (n & (n - 1)) == 0; }
inline bool valid_BN(int64_t B, int64_t N) {
    return B >= 1 && B <= (int64_t)1 << 30 && is_pow2(N) && N >= 4 && N <= ((int64_t)1 << 30);
}
inline bool valid_dtype(int d) { return d == AGNVAR_F32 || d == AGNVAR_F64; }
// the generic FFT plan has three passes: 2^29 complex points in fp32 (8192-point tiles), 2^26 in fp64 (4096-point tiles);
// sizes above that are refused (AGNVAR_EUNSUPPORTED), never silently wrong
inline bool size_supported(int dtype, int64_t len) { return len <= (dtype == AGNVAR_F64 ? ((int64_t)1 << 27) : ((int64_t)1 << 30)); }
inline bool aligned(const void* p, size_t a) { return ((uintptr_t)p % a) == 0; }
inline bool valid_oversample(int o) { return o == 1 || o == 2 || o == 4 || o == 8 || o == 10 || o == 16 || o == 20; }

template <typename T> cudaError_t ensure_attrs() {
    bool& done = dev_cache().attrs[sizeof(T) == 8 ? 1 : 0];
    if (done) return cudaSuccess;
    cudaError_t e = fft_set_attrs<T>();
    if (e != cudaSuccess) return e;
    e = sort_set_attrs<T>();
    if (e != cudaSuccess) return e;
    if (sizeof(T) == 4) {
        e = fft2_set_attrs<float>();
        if (e != cudaSuccess) return e;
        e = sort32_set_attrs();
        if (e != cudaSuccess) return e;
    }
    done = true;
    return cudaSuccess;
}

inline unsigned cdiv(long long a, long long b) { return (unsigned)((a + b - 1) / b); }

// ---- workspace sizes -----------------------------------------------------------------------------
template <typename T> size_t sort_ws_any(int64_t B, int64_t N) {
    size_t s = sort_ws_bytes<T>(B, N);
    if (sort32_applicable(sizeof(T), N)) s = std::max(s, sort32_ws_bytes(B, N));
    return s;
}
inline int delta_chunks(int64_t N) { return (int)((N + kDeltaChunk - 1) / kDeltaChunk); }
template <typename T> size_t ws_e13(int64_t B, int64_t N, bool delta) {
    typedef typename Cx<T>::type C;
    Carver c(nullptr);
    c.take<C>(std::max(FftPlan<T>::table_elems(), Fft2Plan<T>::table_elems()));
    c.take<unsigned int>(Fft2Plan<T>::counter_words(B));
    c.take<T>((size_t)B * N);                 // Z / x_adj
    c.take<T>((size_t)B * (N / 2 + kApPad));  // A_norm in position order
    c.take<uint32_t>((size_t)B * N);          // permutation ping-pong
    c.take<unsigned long long>((size_t)B);    // changed counters
    c.take<int>((size_t)B + 1);               // first_stop [B], n_stopped
    c.take<uint32_t>((size_t)B * kRadix);     // bin cursors of the two-level scatter
    if (delta) {
        c.take<T>((size_t)B * N);             // x_sim ping
        c.take<T>((size_t)B * N);             // x_sim pong
        c.take<uint32_t>((size_t)B * N);      // second working permutation (d_perm is output only)
        c.take<double>((size_t)B * delta_chunks(N));
    }
    if (bucket1_wb_applicable(sizeof(T), N)) c.take<unsigned char>(bucket1_wb_bytes(B, N));   // write-back records of the sort
    return c.off + sort_ws_any<T>(B, N);
}
template <typename T> size_t ws_tk(int64_t B, int64_t N, int os) {
    typedef typename Cx<T>::type C;
    Carver c(nullptr);
    const int64_t M = N * os;
    c.take<C>(FftPlan<T>::table_elems());     // tables, length-M transform
    c.take<C>(FftPlan<T>::table_elems());     // tables, length-N transform
    c.take<PsdDev>((size_t)B);
    c.take<double>((size_t)B * 1024);         // partial sums
    if (os % 5 == 0) c.take<C>((size_t)B * 3 * (M / 5));
    else c.take<T>((size_t)B * M);
    c.take<T>((size_t)B * N);                 // x_norm
    c.take<T>((size_t)B * N);                 // spectrum of x_norm
    return c.off;
}
template <typename T> size_t ws_erdf(int64_t B, int64_t N, int64_t G) {
    Carver c(nullptr);
    c.take<ErdfDev>((size_t)B);
    c.take<double>((size_t)B * G);
    c.take<T>((size_t)B * N);                 // the draw in draw order
    return c.off + sort_ws_any<T>(B, N);
}
template <typename T> size_t ws_pgram(int64_t B, int64_t N, int64_t nbins) {
    typedef typename Cx<T>::type C;
    Carver c(nullptr);
    c.take<C>(FftPlan<T>::table_elems());
    c.take<T>((size_t)B * N);
    c.take<double>((size_t)B);
    c.take<double>((size_t)B * (N / 2));
    c.take<long long>((size_t)nbins + 1);
    return c.off;
}

inline int cuda_status(cudaError_t e) { return e == cudaSuccess ? AGNVAR_OK : AGNVAR_ECUDA; }
// CUDA runtime call inside an int-returning implementation: a failure is AGNVAR_ECUDA
#define CK(call) do { if ((call) != cudaSuccess) return AGNVAR_ECUDA; } while (0)

// real forward FFT of B series of length N held in `Z` (in place, viewed as [B][N/2] complex);
// result in position order.
template <typename T> void rfft_inplace(const FftPlan<T>& p, T* Z, int64_t B, cudaStream_t st) {
    typedef typename Cx<T>::type C;
    const long long L = 1ll << p.dg.logL;
    fft_forward<T>(p, (const C*)Z, (C*)Z, L, L, (int)B, st);
}

// ---- E13 -------------------------------------------------------------------------------------------
struct E13Opts {
    double delta_threshold = 0.0;
    double* d_delta_hist = nullptr;
    int32_t* d_sort_fallbacks = nullptr;
    int check_every = 0;
    bool delta() const { return delta_threshold > 0.0 || d_delta_hist != nullptr; }
};

template <typename T>
int e13_impl(int64_t B, int64_t N, const void* d_anorm, const void* d_sorted, uint32_t* d_perm, void* d_x,
             int max_iter, int32_t* d_iters_used, int64_t* d_changed_hist, void* d_xadj_dbg, const E13Opts& opt,
             void* d_ws, size_t ws_bytes, cudaStream_t st) {
    typedef typename Cx<T>::type C;
    const bool dmode = opt.delta();
    if (ws_bytes < ws_e13<T>(B, N, dmode) || !d_ws || !aligned(d_ws, 256)) return AGNVAR_EWORKSPACE;
    if (ensure_attrs<T>() != cudaSuccess) return AGNVAR_ECUDA;
    const int logL = ilog2_u64((uint64_t)N) - 1;
    const long long L = N / 2;
    Carver c(d_ws);
    C* tables = c.take<C>(std::max(FftPlan<T>::table_elems(), Fft2Plan<T>::table_elems()));
    unsigned int* counters = c.take<unsigned int>(Fft2Plan<T>::counter_words(B));
    T* Z = c.take<T>((size_t)B * N);
    T* Ap = c.take<T>((size_t)B * (N / 2 + kApPad));
    uint32_t* P1 = c.take<uint32_t>((size_t)B * N);
    unsigned long long* changed = c.take<unsigned long long>((size_t)B);
    int* first_stop = c.take<int>((size_t)B + 1);
    unsigned int* n_stopped = (unsigned int*)(first_stop + B);
    uint32_t* cursor = c.take<uint32_t>((size_t)B * kRadix);
    T *XA = nullptr, *XB = nullptr;
    uint32_t* P0 = nullptr;
    double* dpartial = nullptr;
    const int nch = delta_chunks(N);
    if (dmode) {
        XA = c.take<T>((size_t)B * N);
        XB = c.take<T>((size_t)B * N);
        P0 = c.take<uint32_t>((size_t)B * N);
        dpartial = c.take<double>((size_t)B * nch);
    }
    // long fp32 curves: the sort also carries the values home (L4 + L5 in three kernels, bucket1.cuh write-back mode)
    const bool wb_mode = bucket1_wb_applicable(sizeof(T), N);
    B1Wb wb;
    memset(&wb, 0, sizeof(wb));
    if (wb_mode) bucket1_wb_carve(c.take<unsigned char>(bucket1_wb_bytes(B, N)), B, N, &wb);
    void* sort_ws = (unsigned char*)d_ws + c.off;
    const bool two_level = N >= (1ll << kTwoLevelScatterLog);
    // the binned (value, dst) pairs live in the sort's ping-pong buffers, which are idle after the sort
    T* pv = (T*)sort_ws;
    uint32_t* pd = (uint32_t*)((unsigned char*)sort_ws + 2 * align_up((size_t)B * N * sizeof(T), 256));
    const T* sorted = (const T*)d_sorted;

    // short curves (fp32 to 2^14, fp64 to 2^13): the whole loop inside one CTA per curve (onchip.cuh); per-curve early exit
    // at changed = 0.
    // The delta_i rule (Eq. 4) runs there too: x_sim,k is parked in d_x during an iteration (onchip.cuh).
    if (onchip_applicable(sizeof(T), N)) {
        AGN_LAUNCH(K_TABLES, st, (tw_init_kernel<T><<<(1 << kLogTw) / 256, 256, 0, st>>>(tables, 1 << kLogTw, kLogTw)));
        CK(cudaMemsetAsync(counters, 0, sizeof(unsigned int), st));
        if (d_changed_hist) CK(cudaMemsetAsync(d_changed_hist, 0, (size_t)B * max_iter * sizeof(int64_t), st));
        if (opt.d_sort_fallbacks) CK(cudaMemsetAsync(opt.d_sort_fallbacks, 0, (size_t)B * sizeof(int32_t), st));
        if (opt.d_delta_hist) CK(cudaMemsetAsync(opt.d_delta_hist, 0, (size_t)B * max_iter * sizeof(double), st));
        OnchipArgs<T> oa;
        oa.anorm = (const T*)d_anorm; oa.sorted = (const T*)d_sorted; oa.perm = d_perm; oa.x = (T*)d_x;
        oa.xadj_dbg = (T*)d_xadj_dbg; oa.iters_used = d_iters_used; oa.hist = (long long*)d_changed_hist;
        oa.tw14 = (const C*)tables; oa.ticket = counters; oa.max_iter = max_iter; oa.B = B;
        oa.delta_threshold = opt.delta_threshold; oa.delta_hist = opt.d_delta_hist;
        if (onchip_run<T>(ilog2_u64((uint64_t)N), oa, st) != cudaSuccess) return AGNVAR_ECUDA;
        return cuda_status(cudaGetLastError());
    }
    // long fp32 curves: column sub-passes in registers + fused mid kernel (fft2.cuh); otherwise the generic passes
    const bool use2 = fft2_applicable(sizeof(T), logL);
    FftPlan<T> plan;
    Fft2Plan<T> plan2;
    TwLevel<T> rlv;
    if (use2) {
        if constexpr (sizeof(T) == 4) {
            plan2 = fft2_plan_init<T>(logL, tables, counters, st);
            plan.dg = plan2.dfull;
        }
    } else {
        plan = fft_plan_init<T>(logL, tables, st);
        rlv = real_level<T>(plan);
    }
    CK(cudaMemsetAsync(changed, 0, (size_t)B * sizeof(unsigned long long), st));
    CK(cudaMemsetAsync(first_stop, 0, ((size_t)B + 1) * sizeof(int), st));
    CK(cudaMemsetAsync(cursor, 0, (size_t)B * kRadix * sizeof(uint32_t), st));
    if (opt.d_sort_fallbacks) CK(cudaMemsetAsync(opt.d_sort_fallbacks, 0, (size_t)B * sizeof(int32_t), st));
    if (opt.d_delta_hist) CK(cudaMemsetAsync(opt.d_delta_hist, 0, (size_t)B * max_iter * sizeof(double), st));
    // entries of iterations that never run (early return with check_every > 0) read 0, as on the on-chip path
    if (d_changed_hist) CK(cudaMemsetAsync(d_changed_hist, 0, (size_t)B * max_iter * sizeof(int64_t), st));
    AGN_LAUNCH(K_PERM_ANORM, st, (perm_anorm_kernel<T><<<bgrid(cdiv(L + 1, 256), B), 256, 0, st>>>((const T*)d_anorm, Ap, plan.dg, (int)B)));
    const unsigned sg = (unsigned)std::min<long long>((N + 1023) / 1024, 148 * 16);
    // working buffers: x_sim in the caller's d_x and the permutations in (d_perm, P1) -- or, when delta_k is wanted,
    // everything in the workspace (x_sim,k and x_sim,k+1 must both exist, and a stopped curve's state is copied out
    // while the batch goes on)
    uint32_t* cur = d_perm;
    uint32_t* nxt = P1;
    T* x = (T*)d_x;
    T* xn = (T*)d_x;
    if (dmode) {
        CK(cudaMemcpyAsync(P0, d_perm, (size_t)B * N * 4, cudaMemcpyDeviceToDevice, st));
        cur = P0; x = XA; xn = XB;
    }
    // gate != null: only the curves with gate[b] != 0 (those the write-back sort gave up on)
    auto rank_scatter = [&](const uint32_t* inew, const uint32_t* iold, T* xout, void* spare, bool count,
                            const uint32_t* gate) -> int {
        if constexpr (sizeof(T) == 4) {
            if (two_level && sort32_applicable(sizeof(T), N)) {
                if (rank_scatter_two_level32(inew, iold, sorted, xout, B, N, (uint2*)spare, cursor, changed, st, gate) != cudaSuccess)
                    return AGNVAR_ECUDA;
                return AGNVAR_OK;
            }
        }
        if (two_level) {
            if (rank_scatter_two_level<T>(inew, iold, sorted, xout, B, N, pv, pd, cursor, changed, st) != cudaSuccess)
                return AGNVAR_ECUDA;
        } else if (count) {
            AGN_LAUNCH(gate ? K_SORT_FALLBACK : K_SCATTER, st, (scatter_count_kernel<T, true><<<bgrid(sg, B), 256, 0, st>>>(inew, iold, sorted, xout, N, changed, (int)B, gate)));
        } else {
            AGN_LAUNCH(K_SCATTER, st, (scatter_count_kernel<T, false><<<bgrid(sg, B), 256, 0, st>>>(inew, nullptr, sorted, xout, N, nullptr, (int)B)));
        }
        return AGNVAR_OK;
    };
    // first x_sim: the draw in draw order (Q15); idx_old = idx_new, so the change count stays 0
    if (int rc = rank_scatter(cur, cur, x, sort_ws, false, nullptr)) return rc;
    int k_done = 0;
    for (int k = 1; k <= max_iter; ++k) {
        if constexpr (sizeof(T) == 4) if (use2) {
            // L1 column sub-passes (x_sim -> Z), then rows: forward FFT + L2 amplitude replace + inverse FFT
            // in one kernel, then L3 inverse column sub-passes (Z -> x_adj, natural order, 1/L)
            if (fft2_columns<T>(plan2, false, (const C*)x, (C*)Z, (int)B, (T)1, st) != cudaSuccess) return AGNVAR_ECUDA;
            if (fft2_mid<T>(plan2, (C*)Z, Ap, (int)B, st) != cudaSuccess) return AGNVAR_ECUDA;
            if (fft2_columns<T>(plan2, true, (const C*)Z, (C*)Z, (int)B, (T)(1.0 / (double)L), st) != cudaSuccess)
                return AGNVAR_ECUDA;
        }
        if (!use2) {
            // L1 forward FFT (x_sim -> Z, position order)
            fft_forward<T>(plan, (const C*)x, (C*)Z, L, L, (int)B, st);
            // L2 amplitude replace
            AGN_LAUNCH(K_REPLACE, st, (replace_kernel<T><<<bgrid(cdiv(L, 256), B), 256, 0, st>>>((C*)Z, Ap, plan.dg, rlv, (int)B)));
            // L3 inverse FFT (Z -> x_adj, natural order, 1/L)
            fft_inverse<T>(plan, (const C*)Z, (C*)Z, L, L, (int)B, (T)(1.0 / (double)L), st);
        }
        // L4 segmented stable argsort
        void* spare = sort_ws;
        const uint32_t* sort_gate = nullptr;       // per-curve "took the LSD fallback" flags of this iteration
        bool sorted_here = false;
        if constexpr (sizeof(T) == 4) {
            if (sort32_applicable(sizeof(T), N)) {
                uint2* sp = nullptr;
                if (wb_mode) { wb.sorted = (const float*)sorted; wb.idx_old = cur; wb.changed = changed; wb.x_out = (float*)xn; }
                if (seg_argsort32((const float*)Z, nxt, nullptr, B, N, sort_ws, &sp, st, &sort_gate, wb_mode ? &wb : nullptr) != cudaSuccess)
                    return AGNVAR_ECUDA;
                spare = sp;
                sorted_here = true;
            }
        }
        if (!sorted_here && seg_argsort<T>(Z, nxt, nullptr, B, N, sort_ws, st) != cudaSuccess) return AGNVAR_ECUDA;
        // L5 rank scatter + change count (write-back mode: already done by the sort, except for curves on the fallback)
        if (int rc = rank_scatter(nxt, cur, xn, spare, true, wb_mode ? sort_gate : nullptr)) return rc;
        // delta_k (Eq. 4) between x_sim,k (x) and x_sim,k+1 (xn)
        if (dmode)
            AGN_LAUNCH(K_DELTA, st, (delta_partial_kernel<T><<<bgrid((unsigned)nch, B), 256, 0, st>>>(x, xn, N, dpartial, nch, (int)B)));
        // L6 bookkeeping
        PostArgs pa;
        pa.changed = changed; pa.first_stop = first_stop; pa.hist = (long long*)d_changed_hist;
        pa.partial = dpartial; pa.delta_hist = opt.d_delta_hist; pa.threshold = opt.delta_threshold;
        pa.N = N; pa.nchunks = nch; pa.k = k; pa.max_iter = max_iter; pa.n_stopped = n_stopped;
        pa.overflow = sort_gate; pa.fallbacks = opt.d_sort_fallbacks;
        AGN_LAUNCH(K_ITER_POST, st, (post_iter_kernel<<<(unsigned)B, 256, 0, st>>>(pa)));
        if (dmode) {
            // curves that stopped in this iteration: their state goes out now (the batch keeps iterating them)
            AGN_LAUNCH(K_COPY, st, (snapshot_kernel<T><<<bgrid(cdiv(N, 4096), B), 256, 0, st>>>(first_stop, k, xn, nxt, (T*)d_x, d_perm, N, (int)B)));
            std::swap(x, xn);
        }
        std::swap(cur, nxt);
        k_done = k;
        if (opt.check_every > 0 && k % opt.check_every == 0 && k < max_iter) {
            unsigned int h_stopped = 0;
            if (cudaStreamSynchronize(st) != cudaSuccess) return AGNVAR_ECUDA;
            if (cudaMemcpy(&h_stopped, n_stopped, sizeof(unsigned int), cudaMemcpyDeviceToHost) != cudaSuccess) return AGNVAR_ECUDA;
            if ((int64_t)h_stopped >= B) break;
        }
    }
    if (dmode) {
        AGN_LAUNCH(K_COPY, st, (snapshot_kernel<T><<<bgrid(cdiv(N, 4096), B), 256, 0, st>>>(first_stop, 0, x, cur, (T*)d_x, d_perm, N, (int)B)));
    } else if (cur != d_perm) {
        CK(cudaMemcpyAsync(d_perm, cur, (size_t)B * N * 4, cudaMemcpyDeviceToDevice, st));
    }
    if (d_xadj_dbg)
        AGN_LAUNCH(K_COPY, st, (copy_canon_kernel<T><<<cdiv(B * N, 256), 256, 0, st>>>(Z, (T*)d_xadj_dbg, (long long)B * N)));
    if (d_iters_used) AGN_LAUNCH(K_ITER_POST, st, (finalize_iters_kernel<<<cdiv(B, 256), 256, 0, st>>>(first_stop, d_iters_used, k_done, (int)B)));
    return cuda_status(cudaGetLastError());
}

// ---- TK ----------------------------------------------------------------------------------------------
template <typename T>
int tk_impl(const agnvar_psd* h_psd, int64_t n_psd, int64_t B, int64_t N, double dt, int os, uint64_t seed,
            uint32_t curve0, void* d_xnorm, void* d_anorm, void* d_ws, size_t ws_bytes, cudaStream_t st) {
    typedef typename Cx<T>::type C;
    if (ws_bytes < ws_tk<T>(B, N, os) || !d_ws || !aligned(d_ws, 256)) return AGNVAR_EWORKSPACE;
    if (ensure_attrs<T>() != cudaSuccess) return AGNVAR_ECUDA;
    const int64_t M = N * os;
    const bool five = (os % 5 == 0);
    Carver c(d_ws);
    C* tabM = c.take<C>(FftPlan<T>::table_elems());
    C* tabN = c.take<C>(FftPlan<T>::table_elems());
    PsdDev* psd = c.take<PsdDev>((size_t)B);
    double* partial = c.take<double>((size_t)B * 1024);
    T* ZM = five ? (T*)c.take<C>((size_t)B * 3 * (M / 5)) : c.take<T>((size_t)B * M);
    T* xn = c.take<T>((size_t)B * N);
    T* ZN = c.take<T>((size_t)B * N);

    std::vector<PsdDev> hp((size_t)B);
    bool need_norm = false;
    for (int64_t b = 0; b < B; ++b) {
        const agnvar_psd& p = h_psd[n_psd == 1 ? 0 : b];
        hp[(size_t)b] = PsdDev{p.A, p.f_b, p.alpha_low, p.alpha_high};
        if (!(p.A > 0.0)) need_norm = true;
    }
    // pageable host -> device: the copy is staged before the call returns
    if (cudaMemcpyAsync(psd, hp.data(), (size_t)B * sizeof(PsdDev), cudaMemcpyHostToDevice, st) != cudaSuccess)
        return AGNVAR_ECUDA;
    if (need_norm) {
        long long half = M / 2;
        int nchunks = (int)std::min<long long>(1024, (half + 4095) / 4096);
        int chunk = (int)((half + nchunks - 1) / nchunks);
        AGN_LAUNCH(K_PSD, st, (psd_norm_partial_kernel<<<bgrid(nchunks, B), 256, 0, st>>>(psd, M, dt, chunk, partial, nchunks, (int)B)));
        AGN_LAUNCH(K_PSD, st, (psd_norm_final_kernel<<<(unsigned)B, 256, 0, st>>>(psd, partial, nchunks, M)));
    }
    T* xsrc;   // where x_norm ends up
    if (five) {
        const int64_t Mp = M / 5;
        const int logMp = ilog2_u64((uint64_t)Mp);
        FftPlan<T> pm = fft_plan_init<T>(logMp, tabM, st);
        AGN_LAUNCH(K_TK_FILL, st, (tk_fill5_kernel<T><<<bgrid(cdiv(Mp, 256), 3 * B), 256, 0, st>>>((C*)ZM, psd, pm.dg, dt, seed, curve0, (int)B)));
        fft_inverse<T>(pm, (const C*)ZM, (C*)ZM, Mp, Mp, (int)(3 * B), (T)1, st);
        AGN_LAUNCH(K_TK_COMBINE, st, (tk_combine5_kernel<T><<<bgrid(cdiv(N, 256), B), 256, 0, st>>>((const C*)ZM, xn, Mp, N, (M - N) / 2, (int)B)));
        xsrc = xn;
    } else {
        const int logLM = ilog2_u64((uint64_t)M) - 1;
        const long long LM = M / 2;
        FftPlan<T> pm = fft_plan_init<T>(logLM, tabM, st);
        AGN_LAUNCH(K_TK_FILL, st, (tk_fill_kernel<T><<<bgrid(cdiv(LM / 2 + 1, 256), B), 256, 0, st>>>((C*)ZM, psd, pm.dg, dt, seed, curve0, (int)B)));
        fft_inverse<T>(pm, (const C*)ZM, (C*)ZM, LM, LM, (int)B, (T)(1.0 / (double)LM), st);
        if (os == 1) xsrc = ZM;
        else {
            AGN_LAUNCH(K_TK_COMBINE, st, (crop_kernel<T><<<bgrid(cdiv(N, 256), B), 256, 0, st>>>(ZM, M, (M - N) / 2, xn, N, (int)B)));
            xsrc = xn;
        }
    }
    if (d_xnorm) CK(cudaMemcpyAsync(d_xnorm, xsrc, (size_t)B * N * sizeof(T), cudaMemcpyDeviceToDevice, st));
    if (d_anorm) {
        const int logL = ilog2_u64((uint64_t)N) - 1;
        const long long L = N / 2;
        FftPlan<T> pn = fft_plan_init<T>(logL, tabN, st);
        fft_forward<T>(pn, (const C*)xsrc, (C*)ZN, L, L, (int)B, st);
        AGN_LAUNCH(K_UNTANGLE_OUT, st, (untangle_out_kernel<T, 0><<<bgrid(cdiv(L, 256), B), 256, 0, st>>>((const C*)ZN, pn.dg, real_level<T>(pn),
                                                                          (T*)d_anorm, nullptr, nullptr, (int)B)));
    }
    return cuda_status(cudaGetLastError());
}

// ---- ERDF ----------------------------------------------------------------------------------------------
template <typename T>
int erdf_impl(const agnvar_erdf* h_erdf, int64_t n_erdf, int64_t B, int64_t N, uint64_t seed, uint32_t curve0,
              int G, void* d_sorted, uint32_t* d_perm0, void* d_draw, void* d_ws, size_t ws_bytes, cudaStream_t st,
              const agnvar_slice_opts* slice = nullptr) {
    if (ws_bytes < ws_erdf<T>(B, N, G) || !d_ws || !aligned(d_ws, 256)) return AGNVAR_EWORKSPACE;
    if (ensure_attrs<T>() != cudaSuccess) return AGNVAR_ECUDA;
    Carver c(d_ws);
    ErdfDev* erdf = c.take<ErdfDev>((size_t)B);
    double* Ctab = c.take<double>((size_t)B * G);
    T* draw = c.take<T>((size_t)B * N);
    void* sort_ws = (unsigned char*)d_ws + c.off;
    if (d_draw) draw = (T*)d_draw;
    std::vector<ErdfDev> he((size_t)n_erdf);
    for (int64_t i = 0; i < n_erdf; ++i) {
        const agnvar_erdf& e = h_erdf[i];
        he[(size_t)i] = ErdfDev{e.kind, 0, e.lam_star, e.delta1, e.delta2, e.mu_log10, e.sigma_log10,
                                std::log10(e.lam_min), std::log10(e.lam_max)};
    }
    if (cudaMemcpyAsync(erdf, he.data(), (size_t)n_erdf * sizeof(ErdfDev), cudaMemcpyHostToDevice, st) != cudaSuccess)
        return AGNVAR_ECUDA;
    if (slice) {
        // NEXT-3: the paper's sampler (slice.cuh), one thread per chain
        SliceArgs sa;
        sa.erdf = erdf; sa.per_curve = n_erdf == 1 ? 0 : 1; sa.gtab = slice->d_density; sa.G = slice->density_points;
        sa.N = N; sa.chains = slice->chains; sa.burn_in = slice->burn_in; sa.thin = slice->thin; sa.m = slice->max_steps;
        sa.w = slice->width; sa.seed = seed; sa.curve0 = curve0; sa.B = (int)B;
        AGN_LAUNCH(K_SLICE_SAMPLE, st, (slice_sample_kernel<T><<<bgrid(cdiv(slice->chains, 128), B), 128, 0, st>>>(sa, draw, slice->d_u_dbg)));
    } else {
        AGN_LAUNCH(K_ERDF_TABLE, st, (erdf_table_kernel<<<(unsigned)n_erdf, 256, 0, st>>>(erdf, G, Ctab)));
        AGN_LAUNCH(K_ERDF_SAMPLE, st, (erdf_sample_kernel<T><<<bgrid(cdiv(N / 2, 256), B), 256, 0, st>>>(erdf, n_erdf == 1 ? 0 : 1, Ctab, G, N, seed,
                                                                          curve0, draw, (int)B)));
    }
    // stable ascending sort carrying the draw index; perm0 is needed internally even if the caller
    // does not want it -> use the tail of the sort workspace? no: sort straight into d_perm0 or a scratch
    uint32_t* perm = d_perm0;
    if (!perm) return AGNVAR_EINVAL;   // guarded by the caller (scratch provided there)
    if constexpr (sizeof(T) == 4) {
        if (sort32_applicable(sizeof(T), N)) {
            if (seg_argsort32(draw, perm, (T*)d_sorted, B, N, sort_ws, nullptr, st) != cudaSuccess) return AGNVAR_ECUDA;
            return cuda_status(cudaGetLastError());
        }
    }
    cudaError_t e = seg_argsort<T>(draw, perm, (T*)d_sorted, B, N, sort_ws, st);
    if (e != cudaSuccess) return AGNVAR_ECUDA;
    return cuda_status(cudaGetLastError());
}

// ---- periodogram -----------------------------------------------------------------------------------------
template <typename T>
int pgram_impl(int64_t B, int64_t N, const void* d_x, double dt, int norm, int nbins, const int64_t* h_edges,
               double* d_out, int64_t* d_counts, void* d_ws, size_t ws_bytes, cudaStream_t st) {
    typedef typename Cx<T>::type C;
    if (ws_bytes < ws_pgram<T>(B, N, nbins) || !d_ws || !aligned(d_ws, 256)) return AGNVAR_EWORKSPACE;
    if (ensure_attrs<T>() != cudaSuccess) return AGNVAR_ECUDA;
    Carver c(d_ws);
    C* tables = c.take<C>(FftPlan<T>::table_elems());
    T* Z = c.take<T>((size_t)B * N);
    double* scale = c.take<double>((size_t)B);
    double* P = c.take<double>((size_t)B * (N / 2));
    long long* edges = c.take<long long>((size_t)nbins + 1);
    const int logL = ilog2_u64((uint64_t)N) - 1;
    const long long L = N / 2;
    FftPlan<T> plan = fft_plan_init<T>(logL, tables, st);
    AGN_LAUNCH(K_PGRAM, st, (pgram_scale_kernel<T><<<(unsigned)B, 256, 0, st>>>((const T*)d_x, N, dt, norm, scale)));
    fft_forward<T>(plan, (const C*)d_x, (C*)Z, L, L, (int)B, st);
    double* Pout = nbins > 0 ? P : d_out;
    AGN_LAUNCH(K_UNTANGLE_OUT, st, (untangle_out_kernel<T, 1><<<bgrid(cdiv(L, 256), B), 256, 0, st>>>((const C*)Z, plan.dg, real_level<T>(plan), nullptr,
                                                                      Pout, scale, (int)B)));
    if (nbins > 0) {
        if (cudaMemcpyAsync(edges, h_edges, (size_t)(nbins + 1) * sizeof(int64_t), cudaMemcpyHostToDevice, st) != cudaSuccess)
            return AGNVAR_ECUDA;
        AGN_LAUNCH(K_PGRAM, st, (pgram_bin_kernel<<<bgrid((unsigned)nbins, B), 256, 0, st>>>(P, L, edges, nbins, d_out, (long long*)d_counts, (int)B)));
    }
    return cuda_status(cudaGetLastError());
}

// ---- NEXT-2: structure function, Delta-m probabilities --------------------------------------------------------
inline int sf_chunks(int64_t N) { return (int)((N + kSfChunk - 1) / kSfChunk); }
inline size_t ws_sf(int64_t B, int64_t N, int64_t nlags, bool counts) {
    Carver c(nullptr);
    c.take<long long>((size_t)nlags);
    c.take<double>((size_t)B * N);                                  // magnitudes
    c.take<unsigned char>((size_t)B * N);                           // detection flags
    if (counts) {
        c.take<unsigned long long>((size_t)B * nlags * kSfMaxRef);
        c.take<unsigned long long>((size_t)B * nlags);
    } else {
        c.take<double>((size_t)B * nlags * sf_chunks(N));
    }
    return c.off;
}

template <typename T>
int sf_impl(int64_t B, int64_t N, const void* d_x, const int64_t* h_lags, int nlags, int mag, double* d_sf2,
            int64_t* d_pairs, double* d_mean, double* d_se, void* d_ws, size_t ws_bytes, cudaStream_t st) {
    if (ws_bytes < ws_sf(B, N, nlags, false) || !d_ws || !aligned(d_ws, 256)) return AGNVAR_EWORKSPACE;
    Carver c(d_ws);
    long long* lags = c.take<long long>((size_t)nlags);
    double* mags = c.take<double>((size_t)B * N);
    c.take<unsigned char>((size_t)B * N);
    const int nch = sf_chunks(N);
    double* partial = c.take<double>((size_t)B * nlags * nch);
    CK(cudaMemcpyAsync(lags, h_lags, (size_t)nlags * sizeof(int64_t), cudaMemcpyHostToDevice, st));
    const dim3 grid((unsigned)nch, sf_lag_groups(nlags), (unsigned)B);
    if (mag) {
        AGN_LAUNCH(K_SF, st, (sf_mag_kernel<T><<<cdiv(B * N, 256), 256, 0, st>>>((const T*)d_x, (long long)B * N, 0.0, 0, 0.0, mags, nullptr)));
        AGN_LAUNCH(K_SF, st, (sf_partial_kernel<double><<<grid, 256, 0, st>>>(mags, N, lags, nlags, partial, nch, (int)B)));
    } else {
        AGN_LAUNCH(K_SF, st, (sf_partial_kernel<T><<<grid, 256, 0, st>>>((const T*)d_x, N, lags, nlags, partial, nch, (int)B)));
    }
    AGN_LAUNCH(K_SF, st, (sf_final_kernel<<<dim3((unsigned)nlags, (unsigned)B), 256, 0, st>>>(partial, nch, N, lags, nlags, d_sf2, (long long*)d_pairs)));
    if (d_mean || d_se) AGN_LAUNCH(K_SF, st, (sf_rep_kernel<<<(unsigned)nlags, 256, 0, st>>>(d_sf2, (int)B, nlags, d_mean, d_se)));
    return cuda_status(cudaGetLastError());
}

template <typename T>
int dm_impl(int64_t B, int64_t N, const void* d_x, const int64_t* h_lags, int nlags, const double* h_ref, int nref,
            double m_zero, int use_cut, double m_cut, double* d_prob, int64_t* d_considered, void* d_ws, size_t ws_bytes,
            cudaStream_t st) {
    if (ws_bytes < ws_sf(B, N, nlags, true) || !d_ws || !aligned(d_ws, 256)) return AGNVAR_EWORKSPACE;
    Carver c(d_ws);
    long long* lags = c.take<long long>((size_t)nlags);
    double* mags = c.take<double>((size_t)B * N);
    unsigned char* det = c.take<unsigned char>((size_t)B * N);
    unsigned long long* counts = c.take<unsigned long long>((size_t)B * nlags * kSfMaxRef);
    unsigned long long* cons = c.take<unsigned long long>((size_t)B * nlags);
    CK(cudaMemcpyAsync(lags, h_lags, (size_t)nlags * sizeof(int64_t), cudaMemcpyHostToDevice, st));
    CK(cudaMemsetAsync(counts, 0, (size_t)B * nlags * kSfMaxRef * sizeof(unsigned long long), st));
    CK(cudaMemsetAsync(cons, 0, (size_t)B * nlags * sizeof(unsigned long long), st));
    DmRefs refs;
    for (int r = 0; r < kSfMaxRef; ++r) refs.ref[r] = r < nref ? h_ref[r] : 0.0;
    AGN_LAUNCH(K_SF, st, (sf_mag_kernel<T><<<cdiv(B * N, 256), 256, 0, st>>>((const T*)d_x, (long long)B * N, m_zero, use_cut, m_cut, mags, det)));
    const dim3 grid((unsigned)sf_chunks(N), (unsigned)nlags, (unsigned)B);
    AGN_LAUNCH(K_SF, st, (dm_count_kernel<<<grid, 256, 0, st>>>(mags, det, N, lags, nlags, refs, nref, counts, cons, (int)B)));
    AGN_LAUNCH(K_SF, st, (dm_final_kernel<<<cdiv(B * nlags * nref, 256), 256, 0, st>>>(counts, cons, (long long)B * nlags, nref, d_prob, (long long*)d_considered)));
    return cuda_status(cudaGetLastError());
}

// ---- NEXT-4: ensemble SF of masked sub-segments ---------------------------------------------------------------
inline size_t ws_ens(int64_t B, int64_t n_sub, int64_t nlags) {
    Carver c(nullptr);
    c.take<long long>((size_t)nlags);
    c.take<double>((size_t)B * n_sub);
    c.take<unsigned char>((size_t)B * n_sub);
    c.take<unsigned long long>((size_t)nlags);
    c.take<double>((size_t)B * nlags * sf_chunks(n_sub));
    return c.off;
}
template <typename T>
int ens_impl(int64_t B, int64_t N, const void* d_x, int64_t n_sub, double keep, uint64_t seed, uint32_t curve0,
             const int64_t* h_lags, int nlags, int mag, double* d_sf2, int64_t* d_pairs, int64_t* d_offsets, void* d_ws,
             size_t ws_bytes, cudaStream_t st) {
    if (ws_bytes < ws_ens(B, n_sub, nlags) || !d_ws || !aligned(d_ws, 256)) return AGNVAR_EWORKSPACE;
    Carver c(d_ws);
    long long* lags = c.take<long long>((size_t)nlags);
    double* v = c.take<double>((size_t)B * n_sub);
    unsigned char* kept = c.take<unsigned char>((size_t)B * n_sub);
    unsigned long long* count = c.take<unsigned long long>((size_t)nlags);
    const int nch = sf_chunks(n_sub);
    double* partial = c.take<double>((size_t)B * nlags * nch);
    CK(cudaMemcpyAsync(lags, h_lags, (size_t)nlags * sizeof(int64_t), cudaMemcpyHostToDevice, st));
    CK(cudaMemsetAsync(count, 0, (size_t)nlags * sizeof(unsigned long long), st));
    AGN_LAUNCH(K_SF, st, (ens_prepare_kernel<T><<<bgrid(cdiv(n_sub, 256), B), 256, 0, st>>>((const T*)d_x, N, n_sub, keep, seed, curve0, mag, v, kept,
                                                                                        (long long*)d_offsets, (int)B)));
    AGN_LAUNCH(K_SF, st, (ens_partial_kernel<<<dim3((unsigned)nch, (unsigned)nlags, (unsigned)B), 256, 0, st>>>(v, kept, n_sub, lags, nlags, partial, count, nch, (int)B)));
    AGN_LAUNCH(K_SF, st, (ens_final_kernel<<<(unsigned)nlags, 256, 0, st>>>(partial, count, nch, nlags, (int)B, d_sf2, (long long*)d_pairs)));
    return cuda_status(cudaGetLastError());
}

}  // namespace

// =====================================================================================================
// C ABI
// =====================================================================================================
extern "C" {

const char* agnvar_strerror(int status) {
    switch (status) {
        case AGNVAR_OK: return "ok";
        case AGNVAR_EINVAL: return "invalid argument";
        case AGNVAR_EWORKSPACE: return "workspace too small, NULL or misaligned";
        case AGNVAR_ECUDA: return "CUDA launch or API failure";
        case AGNVAR_EUNSUPPORTED: return "unsupported configuration";
        case AGNVAR_ESTATIC_LIMIT: return "request does not fit the library's built-in scratch array (agnvar_static_scratch_bytes)";
        default: return "unknown status";
    }
}

#ifndef AGNVAR_SRC_HASH
#define AGNVAR_SRC_HASH "unknown"
#endif
const char* agnvar_version(void) { return "agnvar 0.2 (sm_100a) src:" AGNVAR_SRC_HASH; }

uint64_t agnvar_launch_count(void) { return trace_state().launches; }

int agnvar_trace_begin(void) {
    TraceState& t = trace_state();
    t.n = 0;
    t.pool_used = 0;
    t.on = true;
    return AGNVAR_OK;
}

int agnvar_trace_end(int64_t cap, int32_t* h_ids, float* h_ms, int64_t* h_n) {
    TraceState& t = trace_state();
    if (!t.on) return AGNVAR_EINVAL;
    t.on = false;
    if (h_n) *h_n = (int64_t)t.n;
    int rc = AGNVAR_OK;
    for (size_t i = 0; i < t.n; ++i) {
        if (cudaEventSynchronize(t.recs[i].e1) != cudaSuccess) { rc = AGNVAR_ECUDA; break; }
        if ((int64_t)i < cap && h_ids && h_ms) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, t.recs[i].e0, t.recs[i].e1) != cudaSuccess) { rc = AGNVAR_ECUDA; break; }
            h_ids[i] = t.recs[i].id;
            h_ms[i] = ms;
        }
    }
    t.n = 0;
    t.pool_used = 0;
    return rc;
}

const char* agnvar_kernel_name(int id) { return (id >= 0 && id < K_NIDS) ? kKernelNames[id] : nullptr; }

size_t agnvar_workspace_bytes(int op, int64_t B, int64_t N, int dtype, int oversample, int64_t aux) {
    if (op == AGNVAR_OP_ENSEMBLE_SF) {   // N is n_sub here: any length agnvar_ensemble_sf accepts, not only powers of two
        if (B < 1 || B > 65535 || N < 2 || N > ((int64_t)1 << 30) || !valid_dtype(dtype) || aux < 1 || aux > 4096) return 0;
        return ws_ens(B, N, aux);
    }
    if (!valid_BN(B, N) || !valid_dtype(dtype) || !size_supported(dtype, N)) return 0;
    const bool f32 = dtype == AGNVAR_F32;
    switch (op) {
        case AGNVAR_OP_E13_ITERATE: return f32 ? ws_e13<float>(B, N, aux != 0) : ws_e13<double>(B, N, aux != 0);
        case AGNVAR_OP_TK_GENERATE:
            if (!valid_oversample(oversample) || !size_supported(dtype, N * (int64_t)oversample)) return 0;
            return f32 ? ws_tk<float>(B, N, oversample) : ws_tk<double>(B, N, oversample);
        case AGNVAR_OP_ERDF_SAMPLE_SORTED:
            if (aux < 2 || aux > 65536) return 0;
            // + a scratch permutation for callers that pass d_perm0 = NULL
            return (f32 ? ws_erdf<float>(B, N, aux) : ws_erdf<double>(B, N, aux)) + align_up((size_t)B * N * 4, 256);
        case AGNVAR_OP_SLICE_SAMPLE_SORTED:
            return (f32 ? ws_erdf<float>(B, N, 2) : ws_erdf<double>(B, N, 2)) + align_up((size_t)B * N * 4, 256);
        case AGNVAR_OP_PERIODOGRAM:
            if (aux < 0 || aux > 4096) return 0;
            return f32 ? ws_pgram<float>(B, N, aux) : ws_pgram<double>(B, N, aux);
        case AGNVAR_OP_STRUCTURE_FUNCTION:
            if (aux < 1 || aux > 4096 || B > 65535) return 0;
            return ws_sf(B, N, aux, false);
        case AGNVAR_OP_DELTA_M_PROB:
            if (aux < 1 || aux > 4096 || B > 65535) return 0;
            return ws_sf(B, N, aux, true);
        default: return 0;
    }
}

int agnvar_philox_u32(uint64_t seed, uint64_t i0, int64_t n, uint32_t curve, uint32_t tag, uint32_t* d_out,
                      void* stream) {
    if (n < 0) return AGNVAR_EINVAL;
    if (n == 0) return AGNVAR_OK;
    if (!d_out) return AGNVAR_EINVAL;
    AGN_LAUNCH(K_PHILOX, (cudaStream_t)stream, (philox_words_kernel<<<cdiv(n, 256), 256, 0, (cudaStream_t)stream>>>(seed, i0, n, curve, tag, (uint4*)d_out)));
    return cuda_status(cudaGetLastError());
}

int agnvar_psd_bpl(const double* d_f, int64_t n, const agnvar_psd* h_p, double* d_out, void* stream) {
    if (n < 0 || !h_p) return AGNVAR_EINVAL;
    if (!std::isfinite(h_p->A) || !std::isfinite(h_p->f_b) || !std::isfinite(h_p->alpha_low) ||
        !std::isfinite(h_p->alpha_high) || !(h_p->f_b > 0.0))
        return AGNVAR_EINVAL;
    if (n == 0) return AGNVAR_OK;
    if (!d_f || !d_out) return AGNVAR_EINVAL;
    PsdDev p{h_p->A, h_p->f_b, h_p->alpha_low, h_p->alpha_high};
    AGN_LAUNCH(K_PSD, (cudaStream_t)stream, (psd_bpl_kernel<<<cdiv(n, 256), 256, 0, (cudaStream_t)stream>>>(d_f, n, p, d_out)));
    return cuda_status(cudaGetLastError());
}

static bool valid_erdf(const agnvar_erdf* h_erdf, int64_t n_erdf, bool allow_table = false) {
    for (int64_t i = 0; i < n_erdf; ++i) {
        const agnvar_erdf& e = h_erdf[i];
        if (e.kind != AGNVAR_ERDF_BPL && e.kind != AGNVAR_ERDF_LOGNORMAL && !(allow_table && e.kind == AGNVAR_ERDF_TABLE))
            return false;
        if (!std::isfinite(e.lam_min) || !std::isfinite(e.lam_max) || !(e.lam_min > 0.0) || !(e.lam_min < e.lam_max))
            return false;
        if (e.kind == AGNVAR_ERDF_TABLE) continue;
        if (e.kind == AGNVAR_ERDF_BPL) {
            if (!std::isfinite(e.lam_star) || !(e.lam_star > 0.0) || !std::isfinite(e.delta1) || !std::isfinite(e.delta2))
                return false;
        } else {
            if (!std::isfinite(e.mu_log10) || !std::isfinite(e.sigma_log10) || !(e.sigma_log10 > 0.0)) return false;
        }
    }
    return true;
}

int agnvar_erdf_table(const agnvar_erdf* h_erdf, int64_t n_erdf, int grid_points, double* d_out, void* stream) {
    if (!h_erdf || n_erdf < 1 || n_erdf > ((int64_t)1 << 30) || grid_points < 2 || grid_points > 65536 || !d_out)
        return AGNVAR_EINVAL;
    if (!valid_erdf(h_erdf, n_erdf)) return AGNVAR_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    // the parameter structs travel as kernel arguments, kErdfArgBatch tables per launch: no device scratch is needed
    for (int64_t i0 = 0; i0 < n_erdf; i0 += kErdfArgBatch) {
        ErdfBatch eb;
        const int n = (int)std::min<int64_t>(kErdfArgBatch, n_erdf - i0);
        for (int i = 0; i < n; ++i) {
            const agnvar_erdf& e = h_erdf[i0 + i];
            eb.e[i] = ErdfDev{e.kind, 0, e.lam_star, e.delta1, e.delta2, e.mu_log10, e.sigma_log10,
                              std::log10(e.lam_min), std::log10(e.lam_max)};
        }
        AGN_LAUNCH(K_ERDF_TABLE, st, (erdf_table_args_kernel<<<(unsigned)n, 256, 0, st>>>(eb, grid_points, d_out + (size_t)i0 * grid_points)));
    }
    return cuda_status(cudaGetLastError());
}

int agnvar_erdf_sample_sorted(const agnvar_erdf* h_erdf, int64_t n_erdf, int64_t B, int64_t N, int dtype,
                              uint64_t seed, uint32_t curve0, int grid_points, void* d_sorted, uint32_t* d_perm0,
                              void* d_draw, void* d_ws, size_t ws_bytes, void* stream) {
    if (!valid_BN(B, N) || !valid_dtype(dtype) || !h_erdf || !d_sorted) return AGNVAR_EINVAL;
    if (!size_supported(dtype, N)) return AGNVAR_EUNSUPPORTED;
    if (!(n_erdf == 1 || n_erdf == B) || grid_points < 2 || grid_points > 65536) return AGNVAR_EINVAL;
    if (!valid_erdf(h_erdf, n_erdf)) return AGNVAR_EINVAL;
    size_t need = agnvar_workspace_bytes(AGNVAR_OP_ERDF_SAMPLE_SORTED, B, N, dtype, 1, grid_points);
    if (!d_ws || ws_bytes < need || !aligned(d_ws, 256)) return AGNVAR_EWORKSPACE;
    const size_t tail = align_up((size_t)B * N * 4, 256);
    uint32_t* perm = d_perm0 ? d_perm0 : (uint32_t*)((unsigned char*)d_ws + (need - tail));
    if (dtype == AGNVAR_F32)
        return erdf_impl<float>(h_erdf, n_erdf, B, N, seed, curve0, grid_points, d_sorted, perm, d_draw, d_ws,
                                need - tail, (cudaStream_t)stream);
    return erdf_impl<double>(h_erdf, n_erdf, B, N, seed, curve0, grid_points, d_sorted, perm, d_draw, d_ws, need - tail,
                             (cudaStream_t)stream);
}

int agnvar_slice_sample_sorted(const agnvar_erdf* h_erdf, int64_t n_erdf, int64_t B, int64_t N, int dtype,
                               uint64_t seed, uint32_t curve0, const agnvar_slice_opts* h_opts, void* d_sorted,
                               uint32_t* d_perm0, void* d_draw, void* d_ws, size_t ws_bytes, void* stream) {
    if (!valid_BN(B, N) || !valid_dtype(dtype) || !h_erdf || !d_sorted || !h_opts) return AGNVAR_EINVAL;
    if (!size_supported(dtype, N)) return AGNVAR_EUNSUPPORTED;
    if (!(n_erdf == 1 || n_erdf == B) || !valid_erdf(h_erdf, n_erdf, true)) return AGNVAR_EINVAL;
    const agnvar_slice_opts& o = *h_opts;
    if (o.chains < 1 || o.chains > ((int64_t)1 << 32) || N % o.chains != 0 || o.burn_in < 0 || o.thin < 1 || o.max_steps < 1 ||
        !(o.width > 0.0) || !std::isfinite(o.width))
        return AGNVAR_EINVAL;
    for (int64_t i = 0; i < n_erdf; ++i)
        if (h_erdf[i].kind == AGNVAR_ERDF_TABLE && (!o.d_density || o.density_points < 2)) return AGNVAR_EINVAL;
    size_t need = agnvar_workspace_bytes(AGNVAR_OP_SLICE_SAMPLE_SORTED, B, N, dtype, 1, 0);
    if (!d_ws || ws_bytes < need || !aligned(d_ws, 256)) return AGNVAR_EWORKSPACE;
    const size_t tail = align_up((size_t)B * N * 4, 256);
    uint32_t* perm = d_perm0 ? d_perm0 : (uint32_t*)((unsigned char*)d_ws + (need - tail));
    if (dtype == AGNVAR_F32)
        return erdf_impl<float>(h_erdf, n_erdf, B, N, seed, curve0, 2, d_sorted, perm, d_draw, d_ws, need - tail,
                                (cudaStream_t)stream, h_opts);
    return erdf_impl<double>(h_erdf, n_erdf, B, N, seed, curve0, 2, d_sorted, perm, d_draw, d_ws, need - tail,
                             (cudaStream_t)stream, h_opts);
}

int agnvar_tk_generate(const agnvar_psd* h_psd, int64_t n_psd, int64_t B, int64_t N, double dt, int oversample,
                       int dtype, uint64_t seed, uint32_t curve0, void* d_xnorm, void* d_anorm, void* d_ws,
                       size_t ws_bytes, void* stream) {
    if (!valid_BN(B, N) || !valid_dtype(dtype) || !h_psd || !valid_oversample(oversample)) return AGNVAR_EINVAL;
    if (!(n_psd == 1 || n_psd == B) || !(dt > 0.0) || !std::isfinite(dt)) return AGNVAR_EINVAL;
    if (!d_xnorm && !d_anorm) return AGNVAR_EINVAL;
    for (int64_t i = 0; i < n_psd; ++i) {
        const agnvar_psd& p = h_psd[i];
        if (!std::isfinite(p.A) || !std::isfinite(p.f_b) || !(p.f_b > 0.0) || !std::isfinite(p.alpha_low) ||
            !std::isfinite(p.alpha_high))
            return AGNVAR_EINVAL;
    }
    if (!size_supported(dtype, N * (int64_t)oversample)) return AGNVAR_EUNSUPPORTED;
    if (dtype == AGNVAR_F32)
        return tk_impl<float>(h_psd, n_psd, B, N, dt, oversample, seed, curve0, d_xnorm, d_anorm, d_ws, ws_bytes,
                              (cudaStream_t)stream);
    return tk_impl<double>(h_psd, n_psd, B, N, dt, oversample, seed, curve0, d_xnorm, d_anorm, d_ws, ws_bytes,
                           (cudaStream_t)stream);
}

int agnvar_e13_iterate(int64_t B, int64_t N, int dtype, const void* d_anorm, const void* d_sorted, uint32_t* d_perm,
                       void* d_x, int max_iter, int32_t* d_iters_used, int64_t* d_changed_hist, void* d_xadj_dbg,
                       const agnvar_e13_opts* h_opts, void* d_ws, size_t ws_bytes, void* stream) {
    if (!valid_BN(B, N) || !valid_dtype(dtype) || max_iter < 1) return AGNVAR_EINVAL;
    if (!size_supported(dtype, N)) return AGNVAR_EUNSUPPORTED;
    if (!d_anorm || !d_sorted || !d_perm || !d_x) return AGNVAR_EINVAL;
    if (!aligned(d_perm, 16) || !aligned(d_x, 16) || !aligned(d_sorted, 16)) return AGNVAR_EINVAL;
    E13Opts opt;
    if (h_opts) {
        if (!std::isfinite(h_opts->delta_threshold) || h_opts->check_every < 0) return AGNVAR_EINVAL;
        opt.delta_threshold = h_opts->delta_threshold > 0.0 ? h_opts->delta_threshold : 0.0;
        opt.d_delta_hist = h_opts->d_delta_hist;
        opt.d_sort_fallbacks = h_opts->d_sort_fallbacks;
        opt.check_every = h_opts->check_every;
    }
    if (dtype == AGNVAR_F32)
        return e13_impl<float>(B, N, d_anorm, d_sorted, d_perm, d_x, max_iter, d_iters_used, d_changed_hist,
                               d_xadj_dbg, opt, d_ws, ws_bytes, (cudaStream_t)stream);
    return e13_impl<double>(B, N, d_anorm, d_sorted, d_perm, d_x, max_iter, d_iters_used, d_changed_hist, d_xadj_dbg,
                            opt, d_ws, ws_bytes, (cudaStream_t)stream);
}

static bool valid_lags(const int64_t* h_lags, int nlags) {
    if (!h_lags || nlags < 1 || nlags > 4096) return false;
    for (int q = 0; q < nlags; ++q)
        if (h_lags[q] < 1) return false;
    return true;
}

int agnvar_structure_function(int64_t B, int64_t N, int dtype, const void* d_x, const int64_t* h_lags, int nlags, int mag,
                              double* d_sf2, int64_t* d_pairs, double* d_rep_mean, double* d_rep_stderr, void* d_ws,
                              size_t ws_bytes, void* stream) {
    if (!valid_BN(B, N) || B > 65535 || !valid_dtype(dtype) || !d_x || !d_sf2 || !valid_lags(h_lags, nlags)) return AGNVAR_EINVAL;
    if (dtype == AGNVAR_F32)
        return sf_impl<float>(B, N, d_x, h_lags, nlags, mag, d_sf2, d_pairs, d_rep_mean, d_rep_stderr, d_ws, ws_bytes,
                              (cudaStream_t)stream);
    return sf_impl<double>(B, N, d_x, h_lags, nlags, mag, d_sf2, d_pairs, d_rep_mean, d_rep_stderr, d_ws, ws_bytes,
                           (cudaStream_t)stream);
}

int agnvar_delta_m_prob(int64_t B, int64_t N, int dtype, const void* d_x, const int64_t* h_lags, int nlags,
                        const double* h_dm_ref, int nref, double m_zero, int use_cut, double m_cut, double* d_prob,
                        int64_t* d_considered, void* d_ws, size_t ws_bytes, void* stream) {
    if (!valid_BN(B, N) || B > 65535 || !valid_dtype(dtype) || !d_x || !d_prob || !valid_lags(h_lags, nlags)) return AGNVAR_EINVAL;
    if (!h_dm_ref || nref < 1 || nref > kSfMaxRef || !std::isfinite(m_zero) || (use_cut && !std::isfinite(m_cut))) return AGNVAR_EINVAL;
    for (int r = 0; r < nref; ++r)
        if (!std::isfinite(h_dm_ref[r])) return AGNVAR_EINVAL;
    if (dtype == AGNVAR_F32)
        return dm_impl<float>(B, N, d_x, h_lags, nlags, h_dm_ref, nref, m_zero, use_cut, m_cut, d_prob, d_considered, d_ws,
                              ws_bytes, (cudaStream_t)stream);
    return dm_impl<double>(B, N, d_x, h_lags, nlags, h_dm_ref, nref, m_zero, use_cut, m_cut, d_prob, d_considered, d_ws,
                           ws_bytes, (cudaStream_t)stream);
}

int agnvar_ensemble_sf(int64_t B, int64_t N, int dtype, const void* d_x, int64_t n_sub, double keep, uint64_t seed,
                       uint32_t curve0, const int64_t* h_lags, int nlags, int mag, double* d_sf2, int64_t* d_pairs,
                       int64_t* d_offsets, void* d_ws, size_t ws_bytes, void* stream) {
    if (!valid_BN(B, N) || B > 65535 || !valid_dtype(dtype) || !d_x || !d_sf2 || !valid_lags(h_lags, nlags)) return AGNVAR_EINVAL;
    if (n_sub < 2 || n_sub > N || !(keep > 0.0) || !(keep <= 1.0)) return AGNVAR_EINVAL;
    if (dtype == AGNVAR_F32)
        return ens_impl<float>(B, N, d_x, n_sub, keep, seed, curve0, h_lags, nlags, mag, d_sf2, d_pairs, d_offsets, d_ws,
                               ws_bytes, (cudaStream_t)stream);
    return ens_impl<double>(B, N, d_x, n_sub, keep, seed, curve0, h_lags, nlags, mag, d_sf2, d_pairs, d_offsets, d_ws,
                            ws_bytes, (cudaStream_t)stream);
}

int agnvar_moments(int64_t B, int64_t N, int dtype, const void* d_x, double* d_out, void* stream) {
    if (!valid_BN(B, N) || B > 0x7fffffffll || !valid_dtype(dtype) || !d_x || !d_out) return AGNVAR_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == AGNVAR_F32) AGN_LAUNCH(K_SF, st, (moments_kernel<float><<<(unsigned)B, 256, 0, st>>>((const float*)d_x, N, d_out)));
    else AGN_LAUNCH(K_SF, st, (moments_kernel<double><<<(unsigned)B, 256, 0, st>>>((const double*)d_x, N, d_out)));
    return cuda_status(cudaGetLastError());
}

int agnvar_periodogram(int64_t B, int64_t N, int dtype, const void* d_x, double dt, int norm, int nbins,
                       const int64_t* h_bin_edges_j, double* d_out, int64_t* d_counts, void* d_ws, size_t ws_bytes,
                       void* stream) {
    if (!valid_BN(B, N) || !valid_dtype(dtype) || !d_x || !d_out) return AGNVAR_EINVAL;
    if (!(norm == 0 || norm == 1) || !(dt > 0.0) || !std::isfinite(dt) || nbins < 0 || nbins > 4096) return AGNVAR_EINVAL;
    if (!aligned(d_x, 16)) return AGNVAR_EINVAL;
    if (!size_supported(dtype, N)) return AGNVAR_EUNSUPPORTED;
    if (nbins > 0) {
        if (!h_bin_edges_j) return AGNVAR_EINVAL;
        if (h_bin_edges_j[0] < 1 || h_bin_edges_j[nbins] > N / 2 + 1) return AGNVAR_EINVAL;
        for (int e = 0; e < nbins; ++e)
            if (!(h_bin_edges_j[e] < h_bin_edges_j[e + 1])) return AGNVAR_EINVAL;
    }
    if (dtype == AGNVAR_F32)
        return pgram_impl<float>(B, N, d_x, dt, norm, nbins, h_bin_edges_j, d_out, d_counts, d_ws, ws_bytes,
                                 (cudaStream_t)stream);
    return pgram_impl<double>(B, N, d_x, dt, norm, nbins, h_bin_edges_j, d_out, d_counts, d_ws, ws_bytes,
                              (cudaStream_t)stream);
}

}  // extern "C"

// =====================================================================================================
// agnvar_structure_function_static -- the structure function for callers that have no scratch to give
// =====================================================================================================
// Every other call of this library works in a scratch buffer the caller allocates (d_ws).  Some callers cannot
// produce one: a plug-in that is handed the light curves and an output slot but no allocator; a serving process whose
// device memory was given, whole, to another component's pool at start-up, so that a cudaMalloc made now fails or eats
// into somebody else's budget; a latency-bound loop that must not pay the device-wide wait an allocation can imply.
// For them the partial sums, the lags and (mag = 1) the magnitudes live in the array below.  It is part of the
// library's image: every GPU that loads libagnvar.so gives up AGNVAR_STATIC_SCRATCH_BYTES of memory for it when the
// module is loaded there and keeps it until the process exits, which is why it is small.
//
// The name `g_sf_static_scratch` means two different things.  In device code it is the array.  In host code it is only
// a handle by which the runtime finds the array: it is NOT an address a kernel can use (passing it would make the
// kernel fault or, on a system where the GPU can read host memory, quietly work in the wrong place).  The host asks for
// the real address with cudaGetSymbolAddress, once per device, with that device current (sf_static_base below), and
// hands that pointer to the kernels -- the same sf_partial / sf_final / sf_rep kernels the workspace path launches.
static __device__ __align__(256) unsigned char g_sf_static_scratch[AGNVAR_STATIC_SCRATCH_BYTES];

namespace {

struct StaticLags { long long l[AGNVAR_STATIC_MAX_LAGS]; };

// the lags arrive as a kernel argument (2 KB) and are written to the head of the scratch, where the pair kernels read
// them: no host-to-device copy, hence no staging buffer of any kind
__global__ void __launch_bounds__(AGNVAR_STATIC_MAX_LAGS) sf_static_lags_kernel(StaticLags h, int nlags, long long* __restrict__ lags) {
    if ((int)threadIdx.x < nlags) lags[threadIdx.x] = h.l[threadIdx.x];
}

// bytes of the array a request uses: lags | magnitudes (mag only) | per-chunk partial sums
inline size_t sf_static_need(int64_t B, int64_t N, int nlags, int mag) {
    Carver c(nullptr);
    c.take<long long>((size_t)nlags);
    if (mag) c.take<double>((size_t)B * N);
    c.take<double>((size_t)B * nlags * sf_chunks(N));
    return c.off;
}

// Device address of g_sf_static_scratch on the CURRENT device; looked up on the first call per device and remembered
// (ordinals >= 64 are looked up every time).  Returns NULL when the runtime refuses.
void* sf_static_base() {
    static std::mutex mu;
    static void* known[64] = {nullptr};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0) return nullptr;
    std::lock_guard<std::mutex> lock(mu);
    if (dev < 64 && known[dev]) return known[dev];
    void* ptr = nullptr;
    if (cudaGetSymbolAddress((void**)&ptr, g_sf_static_scratch) != cudaSuccess || !ptr) return nullptr;
    if (dev < 64) known[dev] = ptr;
    return ptr;
}

template <typename T>
int sf_static_impl(int64_t B, int64_t N, const void* d_x, const int64_t* h_lags, int nlags, int mag, double* d_sf2,
                   int64_t* d_pairs, double* d_mean, double* d_se, cudaStream_t st) {
    void* base = sf_static_base();
    if (!base) return AGNVAR_ECUDA;
    Carver c(base);
    long long* lags = c.take<long long>((size_t)nlags);
    double* mags = mag ? c.take<double>((size_t)B * N) : nullptr;
    const int nch = sf_chunks(N);
    double* partial = c.take<double>((size_t)B * nlags * nch);
    // Nothing in the array has to start at zero: the lags, every magnitude and every (curve, lag, chunk) partial sum
    // are written by this call before anything reads them, so what an earlier call left behind is never seen.
    StaticLags hl;
    for (int q = 0; q < AGNVAR_STATIC_MAX_LAGS; ++q) hl.l[q] = q < nlags ? (long long)h_lags[q] : 0;
    AGN_LAUNCH(K_SF, st, (sf_static_lags_kernel<<<1, AGNVAR_STATIC_MAX_LAGS, 0, st>>>(hl, nlags, lags)));
    const dim3 grid((unsigned)nch, sf_lag_groups(nlags), (unsigned)B);
    if (mag) {
        AGN_LAUNCH(K_SF, st, (sf_mag_kernel<T><<<cdiv(B * N, 256), 256, 0, st>>>((const T*)d_x, (long long)B * N, 0.0, 0, 0.0, mags, nullptr)));
        AGN_LAUNCH(K_SF, st, (sf_partial_kernel<double><<<grid, 256, 0, st>>>(mags, N, lags, nlags, partial, nch, (int)B)));
    } else {
        AGN_LAUNCH(K_SF, st, (sf_partial_kernel<T><<<grid, 256, 0, st>>>((const T*)d_x, N, lags, nlags, partial, nch, (int)B)));
    }
    AGN_LAUNCH(K_SF, st, (sf_final_kernel<<<dim3((unsigned)nlags, (unsigned)B), 256, 0, st>>>(partial, nch, N, lags, nlags, d_sf2, (long long*)d_pairs)));
    if (d_mean || d_se) AGN_LAUNCH(K_SF, st, (sf_rep_kernel<<<(unsigned)nlags, 256, 0, st>>>(d_sf2, (int)B, nlags, d_mean, d_se)));
    return cuda_status(cudaGetLastError());
}

}  // namespace

extern "C" {

size_t agnvar_static_scratch_bytes(void) { return (size_t)AGNVAR_STATIC_SCRATCH_BYTES; }

size_t agnvar_structure_function_static_bytes(int64_t B, int64_t N, int nlags, int mag) {
    if (!valid_BN(B, N) || B > 65535 || nlags < 1 || nlags > AGNVAR_STATIC_MAX_LAGS) return 0;
    return sf_static_need(B, N, nlags, mag);
}

int agnvar_structure_function_static(int64_t B, int64_t N, int dtype, const void* d_x, const int64_t* h_lags, int nlags,
                                     int mag, double* d_sf2, int64_t* d_pairs, double* d_rep_mean, double* d_rep_stderr,
                                     void* stream) {
    if (!valid_BN(B, N) || B > 65535 || !valid_dtype(dtype) || !d_x || !d_sf2 || !valid_lags(h_lags, nlags)) return AGNVAR_EINVAL;
    if (nlags > AGNVAR_STATIC_MAX_LAGS) return AGNVAR_ESTATIC_LIMIT;
    if (sf_static_need(B, N, nlags, mag) > (size_t)AGNVAR_STATIC_SCRATCH_BYTES) return AGNVAR_ESTATIC_LIMIT;
    if (dtype == AGNVAR_F32)
        return sf_static_impl<float>(B, N, d_x, h_lags, nlags, mag, d_sf2, d_pairs, d_rep_mean, d_rep_stderr, (cudaStream_t)stream);
    return sf_static_impl<double>(B, N, d_x, h_lags, nlags, mag, d_sf2, d_pairs, d_rep_mean, d_rep_stderr, (cudaStream_t)stream);
}

}  // extern "C"

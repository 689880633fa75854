// fft_reg.cuh -- register-resident radix-2^k butterflies (k <= 6) with compile-time twiddles.
// A thread holds N complex values in registers; fft_reg_dif<N> is an in-place decimation-in-frequency
// FFT of them (forward sign, Eq. A1 of the paper with the usual sign, O5).  All indices are
// compile-time after unrolling, twiddles are immediates (twc64.cuh), trivial twiddles (1, -i, the two
// sqrt(1/2) ones) are special-cased.  Output: X[k] is left in v[bitrev<N>(k)].
// Inverse transforms use swap(FFT(swap(x))) -- the swaps are register renames.
#pragma once
#include "common.cuh"
#include "twc64.cuh"

namespace agn {

template <int N> __host__ __device__ constexpr int bitrev(int k) {
    int r = 0;
    for (int n = N >> 1; n > 0; n >>= 1) { r = (r << 1) | (k & 1); k >>= 1; }
    return r;
}

// Packed fp32 pair arithmetic of sm_100 (FADD2 / FMUL2 / FFMA2: one issue slot for both halves of a complex number).
__device__ __forceinline__ unsigned long long pk(float2 a) {
    unsigned long long u;
    asm("mov.b64 %0, {%1, %2};" : "=l"(u) : "f"(a.x), "f"(a.y));
    return u;
}
__device__ __forceinline__ float2 unpk(unsigned long long u) {
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(u));
    return r;
}
__device__ __forceinline__ float2 pk_add(float2 a, float2 b) {
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a)), "l"(pk(b)));
    return unpk(r);
}
__device__ __forceinline__ float2 pk_sub(float2 a, float2 b) {
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a)), "l"(pk(b)));
    return unpk(r);
}
__device__ __forceinline__ float2 pk_mul(float2 a, float2 b) {
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk(a)), "l"(pk(b)));
    return unpk(r);
}
__device__ __forceinline__ float2 pk_fma(float2 a, float2 b, float2 c) {
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(pk(a)), "l"(pk(b)), "l"(pk(c)));
    return unpk(r);
}
// d * (c - i s) for a compile-time twiddle: (d.x c + d.y s, d.y c - d.x s) = d * (c, c) + (d.y, d.x) * (s, -s)
__device__ __forceinline__ float2 pk_twiddle(float2 d, float c, float s) {
    return pk_fma(make_float2(d.y, d.x), make_float2(s, -s), pk_mul(d, make_float2(c, c)));
}

template <typename T, int N, int LEN, typename C> struct RegDifLevel {
    static __device__ __forceinline__ void run(C (&v)[N]) {
        constexpr int HALF = LEN / 2;
        constexpr int STEP = 64 / LEN;           // w_LEN^j = w_64^{j * STEP}
#pragma unroll
        for (int blk = 0; blk < N; blk += LEN) {
#pragma unroll
            for (int j = 0; j < HALF; ++j) {
                const C a = v[blk + j], b = v[blk + j + HALF];
                const int tw = j * STEP;
                if constexpr (sizeof(T) == 4) {
                    v[blk + j] = pk_add(a, b);
                    const C d = pk_sub(a, b);
                    if (tw == 0) v[blk + j + HALF] = d;
                    else if (tw == 16) v[blk + j + HALF] = cmul_mi(d);
                    else v[blk + j + HALF] = pk_twiddle(d, (float)cos64(tw), (float)sin64(tw));
                    continue;
                }
                v[blk + j] = cadd(a, b);
                const C d = csub(a, b);
                C r;
                if (tw == 0) r = d;
                else if (tw == 16) r = cmul_mi(d);
                else if (tw == 8) {
                    const T h = (T)0.70710678118654752440084436210485;
                    r.x = h * (d.x + d.y); r.y = h * (d.y - d.x);
                } else if (tw == 24) {
                    const T h = (T)0.70710678118654752440084436210485;
                    r.x = h * (d.y - d.x); r.y = -h * (d.x + d.y);
                } else {
                    const T c = (T)cos64(tw), s = (T)sin64(tw);     // w = c - i s
                    r.x = d.x * c + d.y * s; r.y = d.y * c - d.x * s;
                }
                v[blk + j + HALF] = r;
            }
        }
        RegDifLevel<T, N, LEN / 2, C>::run(v);
    }
};
template <typename T, int N, typename C> struct RegDifLevel<T, N, 1, C> {
    static __device__ __forceinline__ void run(C (&)[N]) {}
};

template <typename T, int N, typename C> __device__ __forceinline__ void fft_reg_dif(C (&v)[N]) {
    static_assert(N >= 1 && N <= 64 && (N & (N - 1)) == 0, "register FFT length");
    RegDifLevel<T, N, N, C>::run(v);
}

// squares and products used to build twiddle powers with short dependency chains
template <typename C> __device__ __forceinline__ C csq(C a) {
    C r; r.x = a.x * a.x - a.y * a.y; r.y = (a.x + a.x) * a.y; return r;
}
// pw[k] = w^k, k = 0..7 (pw[0] = 1), each a product of at most 3 factors deep
template <typename T, typename C> __device__ __forceinline__ void pow8(C w, C (&pw)[8]) {
    pw[0] = mk<T>((T)1, (T)0);
    pw[1] = w;
    pw[2] = csq(w);
    pw[3] = cmul(pw[2], w);
    pw[4] = csq(pw[2]);
    pw[5] = cmul(pw[4], w);
    pw[6] = cmul(pw[4], pw[2]);
    pw[7] = cmul(pw[4], pw[3]);
}
// pw[k] = w^k, k = 0..15
template <typename T, typename C> __device__ __forceinline__ void pow16(C w, C (&pw)[16]) {
    C lo[8];
    pow8<T, C>(w, lo);
#pragma unroll
    for (int k = 0; k < 8; ++k) pw[k] = lo[k];
    pw[8] = csq(lo[4]);
#pragma unroll
    for (int k = 1; k < 8; ++k) pw[8 + k] = cmul(pw[8], lo[k]);
}

}  // namespace agn

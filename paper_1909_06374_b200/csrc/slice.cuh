// slice.cuh -- NEXT-3: the paper's sampler for the random draw, slice sampling (Neal 2003, Ann. Statist. 31, 705;
// PAPER.md:124 "for the random draw step we apply slice sampling (Neal 2003) from a normalised ERDF ... additional
// functional forms can be added if needed": the step that limits the paper's running time).
//
// One thread = one Markov chain in u = log10(lambda); density g(u) ~ xi(10^u) on [u_lo, u_hi], 0 outside (Q10), or a
// caller-supplied table on a uniform grid, linearly interpolated (kind 2).  Update = Neal's Fig. 3 (stepping out,
// width w, at most m intervals) + Fig. 5 (shrinkage); reading Q24 of DESIGN.md fixes what the paper leaves open:
// chain c of curve b draws its uniforms in order from Philox counter (call, c, b, tag 5), starts at
// u_lo + U (u_hi - u_lo), keeps every thin-th state after burn_in updates; kept state j is sample n = j * chains + c
// (so a warp's stores are coalesced).  All arithmetic fp64 with one rounding per written operation (__dmul_rn /
// __dadd_rn: never contracted into FMAs), so that a chain follows the plain CPU statement bit by bit as long as no
// accept / step decision sits within a rounding error of the libm-vs-CUDA difference in pow / exp.
#pragma once
#include "common.cuh"
#include "kernels.cuh"

namespace agn {

constexpr int kSliceMaxShrink = 1000;
constexpr uint32_t kSliceTag = 5u;

struct SliceArgs {
    const ErdfDev* erdf;        // [n_erdf] (kind 0 / 1 / 2)
    int per_curve;              // 1: erdf[b], table row b; 0: erdf[0], row 0
    const double* gtab;         // kind 2: [n_erdf][G] un-normalised density on the uniform grid over [u_lo, u_hi]
    long long G;
    long long N, chains;
    int burn_in, thin, m;
    double w;
    uint64_t seed;
    uint32_t curve0;
    int B;
};

struct SliceUniforms {
    uint64_t seed, q;
    uint32_t chain, curve;
    uint4 wd;
    __device__ __forceinline__ double next() {
        if ((q & 1ull) == 0ull) wd = philox_stream(seed, ((uint64_t)chain << 32) | (q >> 1), curve, kSliceTag);
        const double U = (q & 1ull) ? u53(wd.z, wd.w) : u53(wd.x, wd.y);
        ++q;
        return U;
    }
};

__device__ __forceinline__ double slice_density(const ErdfDev& e, double u, const double* __restrict__ gt, long long G,
                                                double D) {
    if (u < e.u_lo || u > e.u_hi) return 0.0;
    if (e.kind == 2) {
        const double t = __ddiv_rn(__dsub_rn(u, e.u_lo), D);
        long long k = (long long)t;
        if (k > G - 2) k = G - 2;
        const double f = __dsub_rn(t, (double)k);
        const double g0 = gt[k], g1 = gt[k + 1];
        return __dadd_rn(g0, __dmul_rn(f, __dsub_rn(g1, g0)));
    }
    return erdf_xi(e, u);
}

template <typename T>
__global__ void __launch_bounds__(128) slice_sample_kernel(SliceArgs a, T* __restrict__ out, double* __restrict__ u_out) {
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int b = (int)bidx();
    if (c >= a.chains || b >= a.B) return;
    const int row = a.per_curve ? b : 0;
    const ErdfDev e = a.erdf[row];
    const double* gt = a.gtab ? a.gtab + (long long)row * a.G : nullptr;
    const double D = (e.kind == 2) ? __ddiv_rn(__dsub_rn(e.u_hi, e.u_lo), (double)(a.G - 1)) : 0.0;
    SliceUniforms rng;
    rng.seed = a.seed; rng.q = 0; rng.chain = (uint32_t)c; rng.curve = a.curve0 + (uint32_t)b;
    const double w = a.w;
    double x = __dadd_rn(e.u_lo, __dmul_rn(rng.next(), __dsub_rn(e.u_hi, e.u_lo)));
    const long long n_keep = a.N / a.chains;
    const long long total = (long long)a.burn_in + n_keep * (long long)a.thin;
    int until_keep = a.burn_in + a.thin;              // updates until the next kept state
    long long j = 0;
    for (long long t = 1; t <= total; ++t) {
        const double y = __dmul_rn(slice_density(e, x, gt, a.G, D), rng.next());
        double L = __dsub_rn(x, __dmul_rn(w, rng.next()));
        double R = __dadd_rn(L, w);
        int J = (int)floor(__dmul_rn((double)a.m, rng.next()));
        int K = (a.m - 1) - J;
        while (J > 0 && y < slice_density(e, L, gt, a.G, D)) { L = __dsub_rn(L, w); --J; }
        while (K > 0 && y < slice_density(e, R, gt, a.G, D)) { R = __dadd_rn(R, w); --K; }
        for (int it = 0; it < kSliceMaxShrink; ++it) {
            const double x1 = __dadd_rn(L, __dmul_rn(rng.next(), __dsub_rn(R, L)));
            if (y < slice_density(e, x1, gt, a.G, D)) { x = x1; break; }
            if (x1 < x) L = x1; else R = x1;
        }
        if (--until_keep == 0) {
            until_keep = a.thin;
            const long long n = j * a.chains + c;
            out[(long long)b * a.N + n] = (T)exp10(x);
            if (u_out) u_out[(long long)b * a.N + n] = x;
            ++j;
        }
    }
}

}  // namespace agn

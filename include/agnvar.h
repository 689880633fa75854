/*
 * agnvar.h -- C ABI of the B200-native light-curve generator (hot path of Sartori et al. 2019,
 * arXiv:1909.06374): batched light curves with a prescribed PSD (bending power law, Eq. 3) and a
 * prescribed value distribution (the ERDF, Eq. 1-2), by Timmer & Koenig + Emmanoulopoulos-style
 * iterative amplitude adjustment (sec. 2.1, sec. 3.2.2).
 *
 * Citations "PAPER.md:<line>" are to the paper text; "Qn"/"On" are the readings listed in DESIGN.md.
 *
 * Conventions (all calls)
 *   - d_* are DEVICE pointers owned by the caller; h_* are HOST pointers, read before the call returns.
 *   - The library never allocates or frees device memory.  Scratch space is the caller's d_ws of
 *     ws_bytes >= agnvar_workspace_bytes(...), 256-byte aligned.
 *   - Every call only enqueues work on `stream` (a cudaStream_t passed as void*; NULL = default
 *     stream) and returns without synchronising.
 *   - Every call returns an agnvar_status; nothing throws or aborts.  AGNVAR_EINVAL is returned
 *     before any launch.  AGNVAR_ECUDA wraps a failed launch (sticky CUDA errors are not cleared).
 *   - Threads: the library keeps small per-device host tables (kernel attributes set, grid sizes, the launch trace)
 *     that are not locked.  Host threads that drive DIFFERENT devices may call concurrently; calls on the SAME device
 *     must be serialised by the caller (one thread inside the library per device at a time).
 *   - Arrays are row-major [B][N], one light curve contiguous.  N is a power of two,
 *     4 <= N <= 2^30 (the paper's own cap is 2^27, "set by memory limitations"; a 180 GB B200 holds
 *     the loop's working set, ~45 bytes per sample, well beyond it).  The fastest paths cover fp32 up to 2^26
 *     (one-level distribution sort) and 2^27 (register column FFT, two-level sort); longer series run through the
 *     generic three-pass FFT and the LSD sort.  fp64: N (and oversample * N) <= 2^27; beyond that AGNVAR_EUNSUPPORTED.
 *   - dtype selects the arithmetic AND storage type of series, spectra and sort keys (float or
 *     double).  PSD values, the ERDF table and the inverse-CDF arithmetic are always fp64.
 *   - Random numbers: Philox4x32-10, key = (seed lo, seed hi), counter = (i lo, i hi, curve b, tag);
 *     tag 0 = TK normals (i = frequency index j), tag 1 = ERDF uniforms (i = n >> 1), tag 3 / 4 = sub-sample offsets /
 *     masks (agnvar_ensemble_sf), tag 5 = slice-sampler uniforms (agnvar_slice_sample_sorted).  A curve's
 *     numbers depend on (seed, b0 + row) only, never on B or on the launch shape (b0 = `curve0`).
 */
#ifndef AGNVAR_H
#define AGNVAR_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    AGNVAR_OK = 0,
    AGNVAR_EINVAL = 1,       /* bad argument (see each call) */
    AGNVAR_EWORKSPACE = 2,   /* ws_bytes too small or d_ws NULL / misaligned */
    AGNVAR_ECUDA = 3,        /* a CUDA launch or API call failed */
    AGNVAR_EUNSUPPORTED = 4, /* valid request this build does not implement (oversample*N > 2^30; fp64 beyond 2^27) */
    AGNVAR_ESTATIC_LIMIT = 5 /* agnvar_structure_function_static only: the request needs more than the built-in array */
} agnvar_status;

typedef enum { AGNVAR_F32 = 0, AGNVAR_F64 = 1 } agnvar_dtype;
typedef enum { AGNVAR_ERDF_BPL = 0, AGNVAR_ERDF_LOGNORMAL = 1, AGNVAR_ERDF_TABLE = 2 /* agnvar_slice_sample_sorted only */ } agnvar_erdf_kind;
typedef enum {
    AGNVAR_OP_ERDF_SAMPLE_SORTED = 1,
    AGNVAR_OP_TK_GENERATE = 2,
    AGNVAR_OP_E13_ITERATE = 3,
    AGNVAR_OP_PERIODOGRAM = 4,
    AGNVAR_OP_STRUCTURE_FUNCTION = 5,
    AGNVAR_OP_DELTA_M_PROB = 6,
    AGNVAR_OP_ENSEMBLE_SF = 7,
    AGNVAR_OP_SLICE_SAMPLE_SORTED = 8
} agnvar_op;

/* Eq. 3: PSD(f) = A [ (f/f_b)^alpha_low + (f/f_b)^alpha_high ]^-1.
 * A <= 0 asks agnvar_tk_generate for the unit-variance normalisation (Q4):
 * A = M^2 / (2 sum_{1<=j<M/2} s_j + s_{M/2}), s_j the bracket at f_j = j/(M dt). */
typedef struct {
    double A, f_b, alpha_low, alpha_high;
} agnvar_psd;

/* Eq. 1, kind BPL:  xi(lambda) ~ [ (lambda/lam_star)^delta1 + (lambda/lam_star)^delta2 ]^-1
 * Eq. 2, kind LOGNORMAL: xi ~ exp(-(log10 lambda - mu_log10)^2 / (2 sigma_log10^2)).
 * xi is dN/dlog(lambda); the sampled density of u = log10(lambda) is proportional to xi(10^u) on
 * [log10 lam_min, log10 lam_max]  (Q10). */
typedef struct {
    int kind;
    int reserved;
    double lam_star, delta1, delta2;
    double mu_log10, sigma_log10;
    double lam_min, lam_max;
} agnvar_erdf;

/* Bytes of scratch the given op needs.  `oversample` matters for AGNVAR_OP_TK_GENERATE only
 * (pass 1 otherwise); `aux` = grid_points for ERDF_SAMPLE_SORTED, nbins for PERIODOGRAM, 1 for E13_ITERATE
 * with the delta_i rule / history (see agnvar_e13_opts), nlags for STRUCTURE_FUNCTION, DELTA_M_PROB and
 * ENSEMBLE_SF (pass n_sub as N for ENSEMBLE_SF: any 2 <= n_sub <= 2^30, not only powers of two), else 0
 * (SLICE_SAMPLE_SORTED: 0).  Returns 0 for invalid arguments. */
size_t agnvar_workspace_bytes(int op, int64_t B, int64_t N, int dtype, int oversample, int64_t aux);

/* S0 -- Eq. 3 at n given frequencies (fp64 in, fp64 out; d_out[i] = A * bracket(d_f[i])).
 * The unit of f is the unit of f_b (Q9).  A is used as given (must be finite).
 * EINVAL: n < 0, NULL pointer with n > 0, non-finite parameter, f_b <= 0. */
int agnvar_psd_bpl(const double* d_f, int64_t n, const agnvar_psd* h_p, double* d_out, void* stream);

/* S1 -- the random draw from the ERDF, sorted ("a random draw from the PDF";
 * PAPER.md:124).  Per curve b: table u_k = u_lo + k D (k < grid_points), p_k = xi(10^u_k),
 * C = normalised trapezoid cumulative; sample n: U from Philox (tag 1), k with C_k <= U < C_{k+1},
 * u = u_k + (U - C_k)/(C_{k+1} - C_k) D, lambda = 10^u rounded to dtype (O4).  Then a stable
 * ascending sort of the N draws carrying the draw index.
 *   h_erdf      n_erdf structs, n_erdf = 1 (shared) or B (one per curve)
 *   curve0      Philox curve number of row 0 (lets a caller shard a batch across GPUs)
 *   d_sorted    out [B][N] dtype: the draw in ascending order
 *   d_perm0     out [B][N] u32 or NULL: d_perm0[b][r] = draw (time) index of the r-th smallest (Q15:
 *               the first x_sim is the draw in draw order, x_sim[perm0[r]] = sorted[r])
 *   d_draw      out [B][N] dtype or NULL: the draw in draw order
 * EINVAL: bad B/N/dtype, n_erdf not 1 or B, grid_points < 2 or > 65536, NULL h_erdf/d_sorted,
 * non-finite parameter, lam_min <= 0, lam_min >= lam_max, sigma <= 0 (log-normal), lam_star <= 0 (BPL). */
int agnvar_erdf_sample_sorted(const agnvar_erdf* h_erdf, int64_t n_erdf, int64_t B, int64_t N, int dtype,
                              uint64_t seed, uint32_t curve0, int grid_points, void* d_sorted,
                              uint32_t* d_perm0, void* d_draw, void* d_ws, size_t ws_bytes, void* stream);

/* S1 by the paper's own sampler (NEXT-3) -- slice sampling (Neal 2003, Ann. Statist. 31, 705) from the ERDF or from
 * any un-normalised density ("for the random draw step we apply slice sampling (Neal 2003) from a
 * normalised ERDF ... additional functional forms can be added if needed"; the step that limits the
 * paper's running time), then the same stable sort as agnvar_erdf_sample_sorted, same outputs.  Same distribution as
 * the inverse-CDF sampler, different samples.  Reading Q24 for what the paper leaves open:
 *   state     u = log10(lambda); density g(u) ~ xi(10^u) on [log10 lam_min, log10 lam_max], 0 outside (Q10); kind
 *             AGNVAR_ERDF_TABLE: g = linear interpolation of d_density (density_points >= 2 values >= 0 on the
 *             uniform grid over that interval; one row per h_erdf entry; lam_star .. sigma_log10 ignored)
 *   chains    `chains` independent Markov chains per curve (N a multiple of chains); chain c starts at
 *             u_lo + U (u_hi - u_lo), makes burn_in + (N / chains) thin updates and keeps every thin-th state after
 *             the burn-in; kept state j of chain c is draw n = j * chains + c
 *   uniforms  Philox tag 5, counter (call, chain c, curve b, 5): uniform number q of a chain = words (0,1) of call
 *             q >> 1 if q is even, words (2,3) if odd
 *   update    y = g(x) U;  stepping out (Neal's Fig. 3): U: L = x - width U, R = L + width; V: J = floor(max_steps V),
 *             K = max_steps - 1 - J; while J > 0 and y < g(L): L -= width, J -= 1; while K > 0 and y < g(R):
 *             R += width, K -= 1;  shrinkage (Fig. 5): U: x1 = L + U (R - L); accept if y < g(x1), else L = x1 if
 *             x1 < x, else R = x1 (at most 1000 draws, then the chain stays: only where g = 0 around x)
 *   output    lambda = 10^x rounded to dtype; d_u_dbg (or NULL): [B][N] fp64, the states x in draw order
 * All arithmetic fp64, one rounding per written operation (no FMA contraction).
 * EINVAL: as agnvar_erdf_sample_sorted, plus NULL h_opts, chains < 1 or not a divisor of N or > 2^32, burn_in < 0,
 * thin < 1, max_steps < 1, width <= 0 or non-finite, kind TABLE without d_density or with density_points < 2. */
typedef struct {
    int64_t chains;
    int32_t burn_in, thin, max_steps, reserved;
    double width;                 /* w, in dex */
    const double* d_density;      /* kind TABLE: [n_erdf][density_points] fp64, else NULL */
    int64_t density_points;
    double* d_u_dbg;
} agnvar_slice_opts;
int agnvar_slice_sample_sorted(const agnvar_erdf* h_erdf, int64_t n_erdf, int64_t B, int64_t N, int dtype,
                               uint64_t seed, uint32_t curve0, const agnvar_slice_opts* h_opts, void* d_sorted,
                               uint32_t* d_perm0, void* d_draw, void* d_ws, size_t ws_bytes, void* stream);

/* S1 (table only) -- the normalised cumulative table C of agnvar_erdf_sample_sorted (O4), for checking the
 * sampler's premise against a reference: d_out [n_erdf][grid_points] fp64, C_0 = 0, C_{G-1} = 1.
 * Same validation as agnvar_erdf_sample_sorted; no workspace. */
int agnvar_erdf_table(const agnvar_erdf* h_erdf, int64_t n_erdf, int grid_points, double* d_out, void* stream);

/* S2 -- Timmer & Koenig series and its amplitudes.  M = oversample * N;
 * X_0 = 0; X_j = sqrt(S_j/2)(g_re + i g_im), 1 <= j < M/2; X_{M/2} = sqrt(S_{M/2}) g_re;
 * S_j = Eq. 3 at f_j = j/(M dt), fp64; g from Philox tag 0, Box-Muller (O1, O3);
 * x = inverse real DFT of length M with 1/M; x_norm = the central N samples
 * x[(M-N)/2 ... (M-N)/2+N-1] (oversampling, Q3); A_norm_j = |DFT_N(x_norm)_j|,
 * j = 0..N/2 (Q2: the amplitudes of the TK realisation are the target of the adjustment).
 *   h_psd       n_psd structs, n_psd = 1 or B
 *   oversample  one of 1, 2, 4, 8, 10, 16, 20
 *   d_xnorm     out [B][N] dtype or NULL
 *   d_anorm     out [B][N/2+1] dtype or NULL
 * EINVAL: bad B/N/dtype/oversample, n_psd not 1 or B, dt <= 0, f_b <= 0, non-finite parameter,
 * NULL h_psd, both outputs NULL.  EUNSUPPORTED: oversample * N > 2^30 (fp64: 2^27). */
int agnvar_tk_generate(const agnvar_psd* h_psd, int64_t n_psd, int64_t B, int64_t N, double dt, int oversample,
                       int dtype, uint64_t seed, uint32_t curve0, void* d_xnorm, void* d_anorm, void* d_ws,
                       size_t ws_bytes, void* stream);

/* Options of agnvar_e13_iterate (host struct, read before the call returns; NULL = all defaults).
 *   delta_threshold  > 0: the paper's own stopping rule (Eq. 4).  After iteration k,
 *                    delta_k = rms over the N samples of log10( x_sim,k+1[t] / x_sim,k[t] ) ("log" read as log10:
 *                    the paper speaks in dex, Q14); curve b stops at the first k with delta_k <= delta_threshold
 *                    (or changed = 0): iters_used[b] = k and d_x / d_perm receive the state after iteration k.
 *                    The batch keeps running until every curve has stopped or k = max_iter (see check_every);
 *                    <= 0: only the exact rank-change rule below.  Needs positive values in d_sorted.
 *                    Short curves (fp32 N <= 2^14, fp64 N <= 2^13) keep their one-CTA-per-curve loop under this rule
 *                    (delta_k is evaluated on chip; each curve leaves the loop at its own k); d_x serves as scratch
 *                    for x_sim,k while the call runs and holds the result when it has finished.
 *   d_delta_hist     out [B][max_iter] fp64 or NULL: delta_k of every executed iteration (later entries 0)
 *   d_sort_fallbacks out [B] i32 or NULL: number of iterations in which curve b's argsort left the distribution
 *                    sort for the LSD fallback (slab overflow: massive ties, adversarial keys); 0 in a normal run
 *   check_every      > 0: the call SYNCHRONISES the stream after every check_every iterations and returns early
 *                    once every curve has stopped (the only case in which a call of this library waits);
 *                    0: never waits, max_iter iterations are enqueued (stopped curves idle: their outputs are
 *                    already written)
 */
typedef struct {
    double delta_threshold;
    double* d_delta_hist;
    int32_t* d_sort_fallbacks;
    int32_t check_every;
    int32_t reserved;
} agnvar_e13_opts;

/* L1-L6 -- the iteration (steps O6).  Per curve, k = 1..max_iter:
 *   X = DFT_N(x_sim);  X'_j = A_norm_j X_j / |X_j|  (X'_j = A_norm_j if |X_j| = 0; DC and Nyquist
 *   real);  x_adj = IDFT_N(X') with 1/N, -0 -> +0;  idx_new = stable ascending argsort of x_adj
 *   (ties: lower time index first);  changed = #{r : idx_new[r] != idx_old[r]};
 *   x_sim[idx_new[r]] = sorted[r].
 * A curve is converged at the first k with changed = 0 (iters_used = k); a converged state is a fixed
 * point, so later iterations of a batch leave it unchanged (Q18).  Not converging within max_iter is
 * not an error: iters_used = max_iter.  h_opts adds the paper's delta_i rule (Eq. 4) and diagnostics.
 *   d_anorm        in  [B][N/2+1] dtype  target amplitudes (natural order, j = 0..N/2)
 *   d_sorted       in  [B][N] dtype      ascending values (the draw)
 *   d_perm         in/out [B][N] u32     in: idx_old of the first iteration (perm0); out: final permutation.
 *                                        Feeding the output back resumes the run.
 *   d_x            out [B][N] dtype      final x_sim  (x[perm[r]] = sorted[r])
 *   d_iters_used   out [B] i32 or NULL
 *   d_changed_hist out [B][max_iter] i64 or NULL: changed count of every executed iteration (entries of iterations that
 *                  did not run -- early return with check_every > 0, on-chip early exit -- are 0)
 *   d_xadj_dbg     out [B][N] dtype or NULL: x_adj of the last iteration (for lock-step checks: call
 *                  with max_iter = 1 to step the product kernels one iteration at a time)
 *   h_opts         NULL or options (above).  Workspace: query with aux = 1 when delta_threshold > 0 or
 *                  d_delta_hist is set (two more [B][N] value buffers and one more permutation buffer).
 * EINVAL: bad B/N/dtype, max_iter < 1, NULL d_anorm/d_sorted/d_perm/d_x, negative check_every,
 * non-finite delta_threshold. */
int agnvar_e13_iterate(int64_t B, int64_t N, int dtype, const void* d_anorm, const void* d_sorted,
                       uint32_t* d_perm, void* d_x, int max_iter, int32_t* d_iters_used,
                       int64_t* d_changed_hist, void* d_xadj_dbg, const agnvar_e13_opts* h_opts, void* d_ws,
                       size_t ws_bytes, void* stream);

/* P -- periodogram (Appendix A), bins j = 1..N/2 (DC excluded):
 *   norm 0 (Eq. A2):  P_j = (2/N^2) |DFT_j|^2
 *   norm 1 (Eq. A4):  P_j = (2 dt / (mu^2 N)) |DFT_j|^2,  mu = sample mean.
 * nbins = 0: d_out [B][N/2] fp64, d_out[b][j-1] = P_j.
 * nbins > 0 (Q19): h_bin_edges_j holds nbins+1 increasing integers j_0 >= 1 ... j_nb <= N/2+1; bin e is
 * the arithmetic mean of P_j over j_e <= j < j_{e+1}, the last bin closed at N/2; d_out [B][nbins] fp64;
 * d_counts [nbins] i64 or NULL receives the number of j per bin.  Sums are accumulated in fp64.
 * EINVAL: bad B/N/dtype/norm, dt <= 0, nbins < 0 or > 4096, edges not increasing or out of range, NULL d_x/d_out. */
int agnvar_periodogram(int64_t B, int64_t N, int dtype, const void* d_x, double dt, int norm, int nbins,
                       const int64_t* h_bin_edges_j, double* d_out, int64_t* d_counts, void* d_ws,
                       size_t ws_bytes, void* stream);

/* SF -- structure function of evenly sampled light curves (Eq. A6) at nlags integer lags l (tau = l dt):
 *   SF(tau)^2 = (1/P) sum over the P = N - l pairs (i, i + l) of [ v_i - v_{i+l} ]^2,
 * v = x (L/L_Edd units, mag = 0) or v = -2.5 log10 x (magnitudes, mag = 1; for a constant bolometric
 * correction m(t2) - m(t1) = -2.5 log10[L(t2)/L(t1)], the zero point cancels; needs x > 0).  Differences and sums in fp64.
 *   h_lags       nlags integers, 1 <= l; a lag l >= N has no pair: sf2 = 0, pairs = 0
 *   d_sf2        out [B][nlags] fp64
 *   d_pairs      out [nlags] i64 or NULL: P = N - l
 *   d_rep_mean, d_rep_stderr   out [nlags] fp64 or NULL: the representative SF over the B realisations (Eq. 6,
 *                PAPER.md:244-251): mean of SF_i(tau)^2 and its standard error (sample std / sqrt(B); 0 for B = 1)
 * EINVAL: bad B/N/dtype, nlags < 1 or > 4096, a lag < 1, NULL h_lags/d_x/d_sf2. */
int agnvar_structure_function(int64_t B, int64_t N, int dtype, const void* d_x, const int64_t* h_lags, int nlags, int mag,
                              double* d_sf2, int64_t* d_pairs, double* d_rep_mean, double* d_rep_stderr, void* d_ws,
                              size_t ws_bytes, void* stream);

/* SF without a workspace -- agnvar_structure_function for callers that cannot hand the library any scratch memory.
 *
 * Who this is for.  Every other call here works in a buffer the caller allocates.  That is no help to code that cannot
 * allocate on the device at all: a plug-in that is passed light curves and an output slot and nothing else; a process
 * whose device memory was handed over wholesale to another component's memory pool when it started, so that a fresh
 * cudaMalloc either fails or takes what someone else budgeted; a loop with a latency bound that cannot absorb the
 * device-wide stall an allocation may bring.  For those callers this one entry point keeps its scratch (the lags, the
 * per-chunk partial sums and, for mag = 1, the magnitudes) in an array that is compiled into the library.  It calls no
 * cudaMalloc, no cudaFree, no host-to-device copy and no routine that allocates; the caller passes the input and the
 * output arrays exactly as for agnvar_structure_function (same meaning, same results bit for bit: the same kernels run).
 *
 * The limit.  The array is AGNVAR_STATIC_SCRATCH_BYTES = 8 MiB, and every GPU on which the library's code is loaded
 * holds those 8 MiB until the process ends whether or not this call is ever used.  A request fits when
 *   agnvar_structure_function_static_bytes(B, N, nlags, mag) <= agnvar_static_scratch_bytes(),
 * i.e. 256-byte-rounded  8 nlags + (mag ? 8 B N : 0) + 8 B nlags ceil(N / 8192),  and nlags <= AGNVAR_STATIC_MAX_LAGS
 * (the lags travel as a kernel argument).  Examples that fit: mag = 0, B = 64 curves of 2^20 samples at 64 lags
 * (4 MiB); mag = 1, B N up to about 10^6 samples.  Anything larger returns AGNVAR_ESTATIC_LIMIT before any launch: use
 * agnvar_structure_function with a workspace instead.
 *
 * First call.  The first call on each device looks up the array's address on that device (the device that is current
 * when the call is made) and remembers it; that look-up may make the CUDA runtime load the library's code onto the
 * device.  Make this first call during start-up, outside any stream capture; later calls only enqueue kernels.
 *
 * Sharing.  There is one array per device and every call on that device uses it.  Two calls whose kernels can overlap
 * on the GPU (different streams, or different host threads without ordering between them) overwrite each other's
 * partial sums and return garbage: order such calls on one stream or with events.  Calls on one stream are safe back
 * to back.  Whatever a call leaves in the array is never read by the next one (each call writes all it reads), so
 * nothing needs clearing between calls.
 *
 * Returns: AGNVAR_EINVAL as agnvar_structure_function; AGNVAR_ESTATIC_LIMIT (nlags or the scratch need above the
 * limit); AGNVAR_ECUDA when the address look-up or a launch fails. */
#define AGNVAR_STATIC_SCRATCH_BYTES (8u << 20)
#define AGNVAR_STATIC_MAX_LAGS 256
size_t agnvar_static_scratch_bytes(void);
size_t agnvar_structure_function_static_bytes(int64_t B, int64_t N, int nlags, int mag);   /* 0 for invalid arguments */
int agnvar_structure_function_static(int64_t B, int64_t N, int dtype, const void* d_x, const int64_t* h_lags, int nlags,
                                     int mag, double* d_sf2, int64_t* d_pairs, double* d_rep_mean, double* d_rep_stderr,
                                     void* stream);

/* dM -- P(|dm| > dm_ref given tau) (Figs 16-17): per curve and lag, the number of pairs (i, i + l)
 * with |m_i - m_{i+l}| > dm_ref divided by the number of pairs considered, m = m_zero - 2.5 log10 x (fp64).
 * use_cut != 0: every point with m > m_cut is replaced by the upper limit m_cut and only pairs in which at least one
 * point is detected (m <= m_cut) are considered (Fig. 17); use_cut = 0: all N - l pairs.
 *   h_dm_ref      nref thresholds (1 <= nref <= 16)
 *   d_prob        out [B][nlags][nref] fp64 (0 where no pair is considered)
 *   d_considered  out [B][nlags] i64 or NULL
 * EINVAL: as above, nref out of range, non-finite m_zero / m_cut / dm_ref, NULL h_dm_ref/d_prob. */
int agnvar_delta_m_prob(int64_t B, int64_t N, int dtype, const void* d_x, const int64_t* h_lags, int nlags,
                        const double* h_dm_ref, int nref, double m_zero, int use_cut, double m_cut, double* d_prob,
                        int64_t* d_considered, void* d_ws, size_t ws_bytes, void* stream);

/* eSF -- ensemble structure function of sparsely sampled sub-segments (PAPER.md:253-259 sec. 3.2.5-3.2.6, :276, Fig. 7-8):
 * from every curve a CONSECUTIVE sub-sample of n_sub points at a random position, masked so that a random fraction
 * `keep` of its points survives; SF(tau)^2 at lag l = Eq. A6 over all pairs of kept points separated by l, pooled over
 * all B curves.  The paper does not say how positions and masks are drawn (Q23): Philox tag 3, call 0 of curve
 * curve0 + b: offset_b = floor(u (N - n_sub + 1)); tag 4: point j is kept iff u_j < keep, u_j from call j >> 1, words
 * (0, 1) if j is even, (2, 3) if odd.  mag as in agnvar_structure_function.
 *   d_sf2      out [nlags] fp64 (0 where no pair survives);  d_pairs  out [nlags] i64 or NULL (pooled pair counts)
 *   d_offsets  out [B] i64 or NULL
 * EINVAL: bad B/N/dtype, n_sub < 2 or > N, keep not in (0, 1], bad lags, NULL d_x/d_sf2. */
int agnvar_ensemble_sf(int64_t B, int64_t N, int dtype, const void* d_x, int64_t n_sub, double keep, uint64_t seed,
                       uint32_t curve0, const int64_t* h_lags, int nlags, int mag, double* d_sf2, int64_t* d_pairs,
                       int64_t* d_offsets, void* d_ws, size_t ws_bytes, void* stream);

/* Moments of each curve's value distribution (the TK95 output-PDF check of sec. 3.2.1 / Fig. 2):
 * d_out [B][4] fp64 = mean, variance (1/N), skewness m3 / m2^1.5, excess kurtosis m4 / m2^2 - 3.  No workspace.
 * EINVAL: bad B/N/dtype, B > 2^31 - 1, NULL pointer. */
int agnvar_moments(int64_t B, int64_t N, int dtype, const void* d_x, double* d_out, void* stream);

/* O1 -- the raw random words every other call consumes (for bit-exact checks of the generator):
 * d_out[4 i + w] = word w of Philox4x32-10 with counter (lo(i0+i), hi(i0+i), curve, tag) and key
 * (seed lo, seed hi), 0 <= i < n.  The paper only names cuRAND; the stream layout is
 * reading O1 of DESIGN.md.  EINVAL: n < 0, NULL d_out with n > 0. */
int agnvar_philox_u32(uint64_t seed, uint64_t i0, int64_t n, uint32_t curve, uint32_t tag, uint32_t* d_out,
                      void* stream);

/* Measurement aids (bench.py's roofline and gpu_launches figures).  Not thread-safe: one host thread
 * drives the library while a trace is open.
 *   agnvar_launch_count   kernels launched by the library in this process so far (memsets/copies excluded)
 *   agnvar_trace_begin    from now on every kernel launch is bracketed by two CUDA events on its stream
 *   agnvar_trace_end      stops tracing, waits for the recorded events and returns the launches in issue
 *                         order: h_ids[i] = kernel family (see agnvar_kernel_name), h_ms[i] = device time of
 *                         launch i in ms.  *h_n receives the number of launches recorded; at most `cap`
 *                         entries are written.  ECUDA if an event query fails; EINVAL if no trace is open.
 *   agnvar_kernel_name    name of kernel family `id`, NULL if id is out of range */
uint64_t agnvar_launch_count(void);
int agnvar_trace_begin(void);
int agnvar_trace_end(int64_t cap, int32_t* h_ids, float* h_ms, int64_t* h_n);
const char* agnvar_kernel_name(int id);

/* Static, never NULL. */
const char* agnvar_strerror(int status);

/* Library version string and the GPU architecture it was compiled for ("sm_100a"). */
const char* agnvar_version(void);

#ifdef __cplusplus
}
#endif
#endif /* AGNVAR_H */

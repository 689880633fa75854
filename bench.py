#!/usr/bin/env python
"""bench.py -- the headline benchmark: E13 light-curve samples x iterations per second on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl agnvar|reference] [--workload C4]

One "step" = one pass of the whole hot path (S1 ERDF draw + sort, S2 TK generate,
max_iter x [L1 FFT, L2 replace, L3 IFFT, L4 argsort, L5 scatter+count, L6 bookkeeping], P periodogram
where the configuration asks for it) over one batch of synthetic curves of BASELINE.json's configuration
(default C4: B=4, N=2^26, fp32, 50 iterations -- the configuration the metric is quoted on).
Prints ONE JSON line (rank 0).

N > 1: one rank per GPU, every rank runs its own batch of curves (curve numbers rank*B ...; no data-path
collective; weak scaling).  Under torchrun the ranks come from the environment; `python bench.py --gpus N`
without torchrun re-executes itself under `python -m torch.distributed.run` with N ranks on 127.0.0.1.

Timed regions: (1) `value`: K steps, device-resident, CUDA events, NO per-launch tracing; (2) `e2e`: K steps through
the public API with the result copied to pinned host memory inside the region; (3) one more step with per-launch
CUDA-event tracing switched on, which feeds `kernels`, `stages` and `roofline` (the traced step is not part of
`value`).

--impl reference times the CPU oracle (oracle/, fp64, plain) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import socket
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "E13 samples x iterations / s"
UNIT = "samples*iterations/s"

# Algorithmic (compulsory) bytes per light-curve sample and launch, fp32, by kernel family: every input
# read once, every output written once.  w = 4 bytes per value.
ALGO_BYTES_PER_SAMPLE = {
    "fft_pass_strided": 8.0,        # read + write one complex half-length array = 4 + 4 B per real sample
    "fft_pass_contiguous": 8.0,
    "fft_mid_fused": 10.0,          # read Z 4 + A_norm 2 + write Z' 4
    "fft_columns": 8.0,             # all column sub-passes of one direction: read 4 + write 4 (intermediates stay in L2)
    "amplitude_replace": 10.0,      # read Z 4 + A_norm 2 + write Z' 4
    "sort_digit_hist": 4.0,         # read keys
    "sort_onesweep": 16.0,          # read (key, idx) 8 + write (key, idx) 8 (first/last pass move less)
    "sort_cdf_tables": 0.5,         # one key in 64, a 32-byte sector each (+ small tables)
    "sort_part_level0": 12.0,       # key 4 -> (key, idx) pair 8
    "sort_part_level1": 16.0,       # pair 8 -> pair 8
    "sort_part_onelevel": 12.0,     # key 4 -> pair 8, straight into the fine buckets
    "sort_bucket_finish": 12.0,     # read (key, idx) 8 + write idx 4
    "sort_part_onelevel_rec": 18.0, # key 4 -> pair 8 + the write-back records (slab position 4, sample number 2)
    "sort_finish_writeback": 24.0,  # read pair 8 + sorted 4 + idx_old 4, write idx_new 4 + value at the slab position 4
    "scatter_gather_back": 14.0,    # read records 6 + slab value 4, write x 4
    "cta_argsort": 8.0,             # read key 4 + write idx 4
    "rank_scatter_count": 16.0,     # idx_new 4 + idx_old 4 + sorted 4 + write x 4
    "scatter_bin": 20.0,            # read 12 + write (val, dst) 8
    "scatter_place": 12.0,          # read 8 + write 4
    "e13_onchip_loop": 0.0,         # the whole loop on chip: per-iteration HBM traffic ~0 (see "hbm_equivalent")
    "sort_lsd_fallback_gated": 0.0, # the LSD passes behind the distribution sort: they exit at once unless a slab overflowed
}
# SURVEY.md 8(d) two-level model, bytes per sample per iteration, per stage (fp32)
STAGE_MODEL_BYTES = {"fft": 26.0, "argsort": 28.0, "scatter": 32.0}
# SURVEY.md 8(d) "floor": what the method must move with unlimited on-chip capacity (reported alongside)
STAGE_FLOOR_BYTES = {"fft": 10.0, "argsort": 8.0, "scatter": 16.0}
STAGE_OF = {
    "fft_pass_strided": "fft", "fft_pass_contiguous": "fft", "amplitude_replace": "fft", "fft_mid_fused": "fft", "fft_columns": "fft",
    "sort_digit_hist": "argsort", "sort_onesweep": "argsort", "cta_argsort": "argsort",
    "sort_part_level0": "argsort", "sort_part_level1": "argsort", "sort_part_onelevel": "argsort",
    "sort_bucket_finish": "argsort", "sort_cdf_tables": "argsort", "sort_lsd_fallback_gated": "argsort",
    "rank_scatter_count": "scatter", "scatter_bin": "scatter", "scatter_place": "scatter",
    "sort_part_onelevel_rec": "argsort", "sort_finish_writeback": "argsort", "scatter_gather_back": "scatter",
}


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def workload_label(cfg):
    s = (f"{cfg['name']}: B={cfg['B']} curves x N=2^{cfg['N'].bit_length() - 1} samples, {cfg['dtype']}, "
         f"max_iter={cfg['max_iter']}, oversample={cfg['oversample']}")
    if cfg.get("sampler") == "slice":
        s += f", S1 by slice sampling {cfg['slice']} (NOT the headline configuration)"
    if cfg.get("delta_threshold"):
        s += f", stopping rule delta_i <= {cfg['delta_threshold']:g} (Eq. 4; NOT the headline configuration)"
    return s


# ------------------------------------------------------------------------------------------------------
# the CPU oracle, timed as it stands on a bounded sample (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------------------
def oracle_sample_inputs(cfg, logn, curve=0):
    """The oracle's own S1 + S2 for one curve of the configuration's parameters at N = 2^logn."""
    import numpy as np
    import oracle
    N = 1 << logn
    e, p = cfg["erdf"][0], cfg["psd"][0]
    srt, perm0, _ = oracle.erdf_sample_sorted(e, cfg["grid_points"], N, cfg["seed"], curve, 0 if cfg["dtype"] == "f32" else 1)
    tk = oracle.tk_generate(0.0, p["f_b"], p["alpha_low"], p["alpha_high"], N, cfg["dt"], 1, cfg["seed"], curve)
    return np.ascontiguousarray(tk["A_norm"]), srt, perm0


def synthetic_loop_inputs(logn, seed=0):
    """Inputs of the right size and shape for TIMING the oracle's loop at sizes where its own S1/S2 would take minutes:
    a sorted log-normal draw, a random permutation and red-noise amplitudes, from numpy (no arithmetic of the method)."""
    import numpy as np
    N = 1 << logn
    rng = np.random.default_rng(seed)
    srt = np.sort(10.0 ** rng.normal(-2.0, 0.7, N))
    perm0 = rng.permutation(N).astype(np.uint32)
    j = np.arange(N // 2 + 1, dtype=np.float64)
    an = 1.0 / (1.0 + j)
    return an, srt, perm0


def oracle_time(logn, iters, inputs):
    import oracle
    an, srt, perm0 = inputs
    t0 = time.perf_counter()
    oracle.e13_iterate(an, srt, perm0, iters)
    dt = time.perf_counter() - t0
    return (1 << logn) * iters / dt, dt


def oracle_all_cores(cfg, logn, iters):
    """One curve per host thread (the oracle itself is single-threaded; ctypes releases the GIL during the call)."""
    from concurrent.futures import ThreadPoolExecutor
    cores = os.cpu_count() or 1
    inputs = synthetic_loop_inputs(logn)
    sets = [(inputs[0], inputs[1], inputs[2].copy()) for _ in range(cores)]
    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=cores) as ex:
        list(ex.map(lambda s: oracle_time(logn, iters, s), sets))
    dt = time.perf_counter() - t0
    return cores * (1 << logn) * iters / dt, dt, cores


REF_LOGN_CAP = 22      # the bounded CPU sample: one curve of the workload's parameters at N = 2^22 (1.5 s per iteration)


def reference_sample(cfg):
    """The ONE bounded sample both CPU legs time (--impl reference and the product line's cpu_baseline.value): one curve
    of the workload's PSD / ERDF parameters at N = min(2^22, the workload's N), inputs from the oracle's own S1 + S2, one
    E13 iteration (L1-L6) per repetition, fp64, one thread."""
    logn = min(REF_LOGN_CAP, cfg["N"].bit_length() - 1)
    sample = (f"1 curve of {cfg['name']}'s PSD/ERDF parameters at N=2^{logn}, 1 E13 iteration per step "
              f"(fp64 CPU oracle, 1 thread)")
    return logn, sample


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    logn, _ = reference_sample(cfg)
    iters = 1
    inputs = oracle_sample_inputs(cfg, logn)
    for _ in range(args.warmup):
        oracle_time(logn, iters, inputs)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_time(logn, iters, inputs)
    dt = time.perf_counter() - t0
    value = args.steps * (1 << logn) * iters / dt
    sample = reference_sample(cfg)[1]
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload_label(cfg), "sample": sample},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


# ------------------------------------------------------------------------------------------------------
# fp32 free-running context numbers (reported next to the lock-step gates, never gated)
# ------------------------------------------------------------------------------------------------------
def fp32_context(ag, cfg, dev):
    import numpy as np
    import oracle
    from paper_1909_06374_b200 import workloads
    logn, iters = 20, 10
    N = 1 << logn
    c = dict(cfg, B=1, N=N, max_iter=iters, nbins=0, oversample=1, psd=cfg["psd"][:1], erdf=cfg["erdf"][:1])
    srt, perm, _ = ag.agnvar_erdf_sample_sorted(c["erdf"], 1, N, "f32", c["seed"], 0, c["grid_points"], device=dev)
    _, an = ag.agnvar_tk_generate(c["psd"], 1, N, c["dt"], 1, "f32", c["seed"], 0, want_xnorm=False, device=dev)
    srt_h, an_h = srt.cpu().numpy()[0], an.cpu().numpy()[0]
    perm_h = perm.cpu().numpy().view(np.uint32)[0].copy()
    out = ag.agnvar_e13_iterate(an, srt, perm, iters, want_delta=True)
    xg = out["x"].cpu().numpy()[0].astype(np.float64)
    ref = oracle.e13_iterate_delta(an_h, srt_h, perm_h, iters, 0.0)      # same inputs (exact in fp64), fp64 arithmetic
    xo = ref["x"]
    edges = workloads.log_bin_edges(N, 64)
    pg, _ = oracle.periodogram_binned(xg, c["dt"], 0, edges)
    po, _ = oracle.periodogram_binned(xo, c["dt"], 0, edges)
    # the target: the amplitudes the loop is asked to reach, binned the same way (P_j = 2/N^2 A_j^2, Eq. A2)
    tgt = 2.0 / (N * float(N)) * an_h.astype(np.float64)[1:] ** 2
    pt = np.array([tgt[edges[e] - 1:edges[e + 1] - 1].mean() for e in range(len(edges) - 1)])
    return {"sample": f"1 curve of {cfg['name']}'s parameters, N=2^{logn}, {iters} iterations, fp32 product vs fp64 oracle, "
                      f"same inputs, free-running (reported, not gated: the map is chaotic w.r.t. rounding)",
            "value_equal_fraction": float(np.mean(xg == xo)),
            "dlog10_rms_dex": float(np.sqrt(np.mean(np.log10(xg / xo) ** 2))),
            "binned_periodogram_max_rel_diff": float(np.max(np.abs(pg / po - 1.0))),
            # shape consistency with the target amplitudes: scatter of log10(P / P_target) over the 64
            # bins about its mean (the level is fixed by the PDF, not by A_norm)
            "periodogram_vs_target_shape_rms_dex": {"gpu_fp32": float(np.std(np.log10(pg / pt))),
                                                    "oracle_fp64": float(np.std(np.log10(po / pt)))},
            "delta_last_iteration": {"gpu_fp32": float(out["delta_hist"][0, iters - 1]),
                                     "oracle_fp64": float(ref["delta_hist"][iters - 1])}}


# ------------------------------------------------------------------------------------------------------
# the other configurations (C1, C2, C3, C5), timed briefly after the headline's regions
# ------------------------------------------------------------------------------------------------------
def time_other_config(ag, torch, workloads, name, dev, peak, steps=3, warmup=2):
    """`steps` steps of the whole path (S1 + S2 + loop + P) of configuration `name`, CUDA events, untraced; then one traced
    step for the kernel time of the E13 call and, where the loop runs on chip, its rate on SURVEY 8(d)'s byte model."""
    cfg = workloads.config(name)
    B, N, iters = cfg["B"], cfg["N"], cfg["max_iter"]
    for _ in range(warmup):
        out = ag.generate_light_curves(cfg, device=dev)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        out = ag.generate_light_curves(cfg, device=dev)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    executed = int(out["iters_used"].sum().item())
    del out
    ag.trace_begin()
    marks = []
    out = ag.generate_light_curves(cfg, device=dev, phase_hook=lambda nm: marks.append((nm, ag.launch_count())))
    torch.cuda.synchronize()
    trace = ag.trace_end()
    del out
    lc0 = marks[0][1]
    idx = {nm: c - lc0 for nm, c in marks}
    order = [nm for nm, _ in marks]
    e13 = trace[idx["E13"]:idx[order[order.index("E13") + 1]]] if order.index("E13") + 1 < len(order) else trace[idx["E13"]:]
    e13_ms = sum(t for _, t in e13)
    onchip = any(nm == "e13_onchip_loop" for nm, _ in e13)
    model = sum(STAGE_MODEL_BYTES.values())
    res = {"workload": workload_label(cfg), "steps": steps, "warmup": warmup, "ms_per_step": ms,
           "value": N * executed / (ms * 1e-3), "unit": UNIT,
           "iterations_executed_per_curve_mean": executed / B,
           "nominal_value_at_max_iter": B * N * iters / (ms * 1e-3),
           "e13_call_kernel_ms_traced": e13_ms, "e13_launches": len(e13),
           "loop": "whole loop inside one CTA per curve (e13_onchip_loop)" if onchip else "multi-kernel loop",
           "loop_samples_x_iterations_per_s": N * executed / (e13_ms * 1e-3) if e13_ms > 0 else None,
           "l2": "inputs larger than L2" if B * N * (4 if cfg["dtype"] == "f32" else 8) > 2 ** 28 else
                 "arrays smaller than L2: not flushed between steps"}
    if e13_ms > 0:
        res["hbm_equivalent_frac_of_peak"] = model * (2 if cfg["dtype"] == "f64" else 1) * N * executed / (e13_ms * 1e-3) / 1e9 / peak
        res["hbm_equivalent_note"] = ("SURVEY 8(d)'s two-level model (86 B per sample per iteration in fp32, twice that in fp64) "
                                      "over the E13 call's kernel time; for the on-chip loop this is NOT its HBM traffic")
    return res


# ------------------------------------------------------------------------------------------------------
# NEXT-2: the structure function (Eq. A6) of the curves the path generates -- its own line, not the headline
# ------------------------------------------------------------------------------------------------------
def run_sf(args, cfg, ag, torch, dev, step):
    import numpy as np
    B, N = cfg["B"], cfg["N"]
    x = step()["x"]
    lags = sorted({int(round(v)) for v in np.logspace(0, np.log10(N // 2), 64)})
    for _ in range(max(args.warmup, 1)):
        ag.agnvar_structure_function(x, lags, want_rep=True)
    torch.cuda.synchronize()
    ag.trace_begin()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        ag.agnvar_structure_function(x, lags, want_rep=True)
    e1.record()
    torch.cuda.synchronize()
    trace = ag.trace_end()
    ms = e0.elapsed_time(e1) / args.steps
    pairs = B * sum(N - l for l in lags)                       # pair differences per call
    peak_hbm, peak_src = measured_peaks()
    w = 4 if cfg["dtype"] == "f32" else 8
    # What bounds it (profiles/r3_next_kernels_summary.md): not HBM -- the 60 lags of a curve run close together and find
    # it in L2, DRAM sees one pass over x -- but the float -> double conversions, which issue on the XU pipe at 16 lanes
    # per clock per SM (ncu: two conversions per pair at 1.77e12 pairs / s = 78 % of that pipe).  The kernel converts a
    # first member once per kSfLagGroup = 8 lags and the partner once per pair: 1.125 conversions per pair.
    conv = 1.125 * pairs if cfg["dtype"] == "f32" else 0.0
    try:
        sm_clock = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["sm_max_mhz"]) * 1e6
    except Exception:
        sm_clock = 1.965e9
    peak_conv = 16.0 * 148 * sm_clock
    top_ms = max(t for _, t in trace)
    print(json.dumps({"metric": "structure-function pair differences / s", "value": pairs / (ms * 1e-3),
                      "unit": "pairs/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
                      "higher_is_better": True, "dtype": cfg["dtype"], "data": "synthetic",
                      "config": {"workload": workload_label(cfg) + f"; agnvar_structure_function at {len(lags)} log-spaced lags, "
                                 "L/L_Edd units, with the representative SF (Eq. 6)", "lags": len(lags)},
                      "roofline": {"bound": "alu", "kernel": "sf_partial_kernel",
                                   "achieved": conv / (ms * 1e-3) / 1e9, "peak": peak_conv / 1e9, "unit": "G conversions/s",
                                   "frac": conv / (ms * 1e-3) / peak_conv if conv else None,
                                   "peak_source": "16 float->double conversions per clock per SM (XU pipe) x 148 SMs x the maximum SM "
                                                  "clock; fp32 input only (fp64 input needs no conversion: fp64-pipe / L2 bound)",
                                   "hbm_one_pass_bytes": float(w) * B * N,
                                   "hbm_frac_on_one_pass": float(w) * B * N / (ms * 1e-3) / 1e9 / peak_hbm,
                                   "hbm_peak": peak_hbm, "hbm_peak_source": peak_src,
                                   "longest_launch_ms": top_ms, "traffic": None},
                      "gpu_launches": len(trace)}), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------------
def respawn_under_torchrun(args):
    """`python bench.py --gpus N` without torchrun: run the same command line as N ranks on this node."""
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="agnvar", choices=["agnvar", "reference"])
    ap.add_argument("--workload", default="C4")
    ap.add_argument("--batch", type=int, default=None, help="override B (subset of the configuration)")
    ap.add_argument("--max-iter", type=int, default=None, help="override max_iter (NOT the headline configuration)")
    ap.add_argument("--sampler", default="inverse_cdf", choices=["inverse_cdf", "slice"],
                    help="S1 by the inverse-CDF table (north_star, the headline) or by the paper's slice sampler (NEXT-3)")
    ap.add_argument("--delta", type=float, default=0.0,
                    help="stop each curve by the paper's delta_i rule (Eq. 4) at this threshold (NOT the headline configuration)")
    ap.add_argument("--op", default="path", choices=["path", "sf"],
                    help="path: the hot path (the headline); sf: the structure function of the generated curves at 64 "
                         "log-spaced lags (NEXT-2, Eq. A6), one JSON line with its own metric and roofline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-context", action="store_true", help="skip the fp32 free-running context numbers")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the short timings of C1, C2, C3 and C5")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="process-group backend of the N > 1 plumbing (gloo: host-side tests of the spawn path)")
    ap.add_argument("--dry-ranks", action="store_true",
                    help="N > 1 plumbing only (rendezvous, curve partition, max-over-ranks, one JSON line), no GPU work")
    args = ap.parse_args()

    from paper_1909_06374_b200 import workloads
    cfg = workloads.config(args.workload, B=args.batch)
    if args.max_iter is not None:
        cfg["max_iter"] = args.max_iter
    if args.sampler == "slice":
        cfg["sampler"] = "slice"
        cfg["slice"] = dict(chains=min(cfg["N"], 65536), burn_in=50, thin=1, width=1.0, max_steps=8)
    if args.delta > 0.0:
        cfg["delta_threshold"] = args.delta
    if args.impl == "reference":
        run_reference(args, cfg)
        return 0
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return respawn_under_torchrun(args)

    import torch
    from paper_1909_06374_b200 import multirank

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    B, N, iters = cfg["B"], cfg["N"], cfg["max_iter"]
    curve0 = multirank.weak_curve0(B, rank)   # Philox curve numbers of this rank's rows: results do not depend on the partition
    units_per_step = B * N * iters

    if args.dry_ranks:
        import torch.distributed as dist
        dist.init_process_group(args.backend)
        ms = multirank.max_over_ranks(100.0 + rank, None, dist)
        if rank == 0:
            print(json.dumps({"metric": METRIC, "unit": UNIT, "n_gpus": world, "dry_ranks": True, "ms_max_over_ranks": ms,
                              "curve0_by_rank": [multirank.weak_curve0(B, r) for r in range(world)],
                              "config": {"workload": workload_label(cfg)}}), flush=True)
        dist.barrier()
        dist.destroy_process_group()
        return 0

    import paper_1909_06374_b200 as ag
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group(args.backend, device_id=dev if args.backend == "nccl" else None)
    ag.lib()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step(host_out=None, want_fallbacks=False, phase_hook=None):
        return ag.generate_light_curves(cfg, device=dev, host_out=host_out, curve0=curve0, want_fallbacks=want_fallbacks,
                                        phase_hook=phase_hook, delta_threshold=args.delta)

    if args.op == "sf":
        return run_sf(args, cfg, ag, torch, dev, step)

    # ---- (1) device-resident timing, untraced ----------------------------------------------------------
    for _ in range(args.warmup):
        out = step()
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    l0 = ag.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        out = step()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = ag.launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None
    iters_used = out["iters_used"].cpu().tolist()
    del out
    ms = multirank.max_over_ranks(ms, dev, dist)
    # units = samples x iterations EXECUTED: a curve that converged (changed = 0) after k < max_iter iterations counts k
    # (the short-curve path leaves the loop there; identical every step: the inputs are seeded)
    iters_executed = int(sum(iters_used))
    units_per_step = N * iters_executed
    units_all = units_per_step
    if dist is not None:
        tu = torch.tensor([float(units_per_step)], dtype=torch.float64, device=dev)
        dist.all_reduce(tu)
        units_all = float(tu.item())
    else:
        units_all = float(units_per_step)
    value = units_all * args.steps / (ms * 1e-3)

    # ---- (3) one traced step: CUDA events around every launch -> per-kernel table, stages, roofline ---------
    barrier()
    ag.trace_begin()
    t0e, t1e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0e.record()
    marks = []                       # (phase name, library launch count when the phase's C-ABI call starts)
    out = step(want_fallbacks=True, phase_hook=lambda name: marks.append((name, ag.launch_count())))
    t1e.record()
    torch.cuda.synchronize()
    trace = ag.trace_end()
    # launches of the E13 call only (the loop): setup FFTs / sorts of S1, S2 and P use the same kernel families and
    # must not be booked on the loop's stages
    lc0 = marks[0][1]
    bounds = {name: c - lc0 for name, c in marks}
    nxt = {marks[i][0]: marks[i + 1][1] - lc0 for i in range(len(marks) - 1)}
    loop_trace = trace[bounds["E13"]:nxt["E13"]] if "E13" in bounds else trace
    phase_ms = {name: sum(t for _, t in trace[bounds[name]:nxt[name]]) for name in nxt}
    ms_traced = t0e.elapsed_time(t1e)
    fallbacks = int(out["sort_fallbacks"].sum()) if out.get("sort_fallbacks") is not None else None
    del out
    fam = {}
    for name, t in trace:
        f = fam.setdefault(name, [0, 0.0])
        f[0] += 1
        f[1] += t
    peak, peak_src = measured_peaks()
    kernels = {k: {"launches": v[0], "ms_total": round(v[1], 4), "ms_avg": v[1] / v[0],
                   "algorithmic_bytes_per_sample": ALGO_BYTES_PER_SAMPLE.get(k)} for k, v in fam.items()}
    lfam = {}
    for name, t in loop_trace:
        f = lfam.setdefault(name, [0, 0.0])
        f[0] += 1
        f[1] += t
    loop = {k: v for k, v in lfam.items() if k in STAGE_OF}
    roofline = None
    stages = {}
    traffic_model = None
    if loop:
        top = max(loop, key=lambda k: loop[k][1])
        n_l, t_l = loop[top]
        bytes_per_launch = ALGO_BYTES_PER_SAMPLE[top] * B * N       # every loop kernel covers the whole batch
        achieved = bytes_per_launch / (t_l / n_l * 1e-3) / 1e9
        roofline = {"bound": "hbm", "kernel": top, "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": bytes_per_launch, "avg_launch_ms": t_l / n_l,
                    "share_of_step": t_l / ms_traced, "timing": "one traced step (CUDA events around every launch)"}
        prof = os.path.join(ROOT, "profiles", "traffic.json")     # dram bytes per launch from the committed ncu capture
        try:
            with open(prof) as f:
                tj = json.load(f)
            roofline["traffic"] = tj.get(top)
            roofline["traffic_source"] = "committed ncu capture (profiles/traffic.json), not measured in this run"
        except Exception:
            pass
        # stage view (the north_star target: each stage >= 60% of the HBM roofline on the 2-level byte model)
        st_ms, st_bytes = {}, {}
        for k, v in loop.items():
            st_ms[STAGE_OF[k]] = st_ms.get(STAGE_OF[k], 0.0) + v[1]
            st_bytes[STAGE_OF[k]] = st_bytes.get(STAGE_OF[k], 0.0) + ALGO_BYTES_PER_SAMPLE[k] * v[0] / iters
        stages = {s: {"ms_per_iteration": t / iters,
                      "model_bytes_per_sample": STAGE_MODEL_BYTES[s],
                      "moved_bytes_per_sample": st_bytes[s],        # what this build's kernels move (algorithmic, summed)
                      "moved_over_model": st_bytes[s] / STAGE_MODEL_BYTES[s],
                      "achieved_GBps": STAGE_MODEL_BYTES[s] * B * N / (t / iters * 1e-3) / 1e9,
                      "frac_of_peak": STAGE_MODEL_BYTES[s] * B * N / (t / iters * 1e-3) / 1e9 / peak,
                      "floor_bytes_per_sample": STAGE_FLOOR_BYTES[s],
                      "frac_of_peak_floor_model": STAGE_FLOOR_BYTES[s] * B * N / (t / iters * 1e-3) / 1e9 / peak}
                  for s, t in st_ms.items()}
        if "argsort" in st_ms and "scatter" in st_ms:
            # the write-back sort does part of L5 inside the sort's finish kernel (values go home along the partition
            # records), so the split between these two stages is a convention: their sum is the robust figure
            t2 = st_ms["argsort"] + st_ms["scatter"]
            m2 = STAGE_MODEL_BYTES["argsort"] + STAGE_MODEL_BYTES["scatter"]
            stages["argsort+scatter"] = {"ms_per_iteration": t2 / iters, "model_bytes_per_sample": m2,
                                         "moved_bytes_per_sample": st_bytes["argsort"] + st_bytes["scatter"],
                                         "moved_over_model": (st_bytes["argsort"] + st_bytes["scatter"]) / m2,
                                         "achieved_GBps": m2 * B * N / (t2 / iters * 1e-3) / 1e9,
                                         "frac_of_peak": m2 * B * N / (t2 / iters * 1e-3) / 1e9 / peak}
        traffic_model = {"iteration_model_bytes_per_sample": sum(STAGE_MODEL_BYTES.values()),
                         "iteration_moved_bytes_per_sample": sum(st_bytes.values())}

    if "e13_onchip_loop" in fam:
        # short curves: the whole loop runs on chip, HBM sees perm0 / x / perm once per call (12 B per sample) and per
        # executed iteration A_norm (2 B) and sorted (4 B) through L1/L2.  The kernel is bound by shared-memory
        # wavefronts and issue slots, not by HBM: `achieved` is its real algorithmic HBM traffic over its duration, and
        # the SURVEY 8(d) "HBM-equivalent" (the 86 B/sample/iteration two-level model over the same time) is given
        # beside it, labelled as such.
        n_l, t_l = fam["e13_onchip_loop"]
        real_bytes = 12.0 * B * N + 6.0 * units_per_step
        achieved = real_bytes / (t_l / n_l * 1e-3) / 1e9
        roofline = {"bound": "hbm", "kernel": "e13_onchip_loop", "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": real_bytes, "avg_launch_ms": t_l / n_l, "share_of_step": t_l / ms_traced,
                    "note": "on-chip loop: per-iteration HBM traffic ~0 by design; bound by shared-memory wavefronts / issue "
                            "slots (profiles/), so the HBM fraction is not a quality measure here",
                    "hbm_equivalent_GBps": sum(STAGE_MODEL_BYTES.values()) * units_per_step / (t_l / n_l * 1e-3) / 1e9,
                    "hbm_equivalent_frac_of_peak": sum(STAGE_MODEL_BYTES.values()) * units_per_step / (t_l / n_l * 1e-3) / 1e9 / peak,
                    "loop_samples_x_iterations_per_s": units_per_step / (t_l / n_l * 1e-3)}

    # ---- (2) end to end: host parameters in, light curves out to pinned host memory -------------------------
    e2e = None
    if not args.no_e2e:
        host = torch.empty((B, N), dtype=torch.float32 if cfg["dtype"] == "f32" else torch.float64).pin_memory()
        step(host_out=host)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            step(host_out=host)     # synchronises: the result is on the host when it returns
        barrier()
        dt = time.perf_counter() - t0
        dt = multirank.max_over_ranks(dt, dev, dist)
        h2d = 32 * len(cfg["psd"]) + 64 * len(cfg["erdf"]) + (8 * (cfg["nbins"] + 1) if cfg.get("nbins") else 0)
        d2h = host.numel() * host.element_size() + 4 * B
        e2e = {"value": units_all * args.steps / dt, "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h}
        del host

    # ---- the other configurations of BASELINE.json (parity-test cases, not bench lines): a short timing of each, so
    # that DESIGN.md section 11's table is driver-run.  Rank 0, N = 1, default workload only.
    other = None
    if rank == 0 and world == 1 and args.workload == "C4" and not args.no_other_configs and args.batch is None \
            and args.max_iter is None and args.sampler == "inverse_cdf" and args.delta <= 0.0:
        ag.free_workspace()
        torch.cuda.empty_cache()
        other = {}
        for name in ("C1", "C2", "C3", "C5"):
            try:
                other[name] = time_other_config(ag, torch, workloads, name, dev, peak)
            except Exception as exc:          # context only: never fails the bench line
                other[name] = {"error": repr(exc)}
            ag.free_workspace()
            torch.cuda.empty_cache()

    # ---- the oracle on this box's host cores (rank 0, N = 1 only) ---------------------------------------
    cpu = None
    context = None
    if rank == 0 and world == 1:
        if not args.no_context and cfg["dtype"] == "f32":
            try:
                context = fp32_context(ag, cfg, dev)
            except Exception as exc:      # context only: never fails the bench line
                context = {"error": repr(exc)}
        ag.free_workspace()
        if not args.no_cpu_baseline:
            # `value`: the sample the reference arm times (one CPU figure per record); then, as context, the same loop at
            # the workload's own N (C4: 2^26, one iteration, about 40 s) and one curve per host thread
            lr, sample = reference_sample(cfg)
            inputs = oracle_sample_inputs(cfg, lr)
            oracle_time(lr, 1, inputs)
            reps, t_ref = 0, 0.0
            while reps < 3 or (t_ref < 8.0 and reps < 64):
                t_ref += oracle_time(lr, 1, inputs)[1]
                reps += 1
            logn = N.bit_length() - 1
            v, dt = oracle_time(logn, 1, synthetic_loop_inputs(logn))
            la = min(22, logn)
            va, dta, cores = oracle_all_cores(cfg, la, 1)
            cpu = {"value": reps * (1 << lr) / t_ref, "unit": UNIT, "cores": 1, "kind": "oracle",
                   "sample": f"{sample}; {reps} repetitions, {t_ref:.1f} s (the sample `--impl reference` times)",
                   "host_cores_available": os.cpu_count(),
                   "full_size": {"value": v, "unit": UNIT, "cores": 1,
                                 "sample": f"1 curve at the workload's own N=2^{logn}, 1 E13 iteration (L1-L6), fp64, 1 thread, "
                                           f"{dt:.1f} s; inputs of that size from numpy (sorted log-normal draw, random "
                                           f"permutation, red-noise amplitudes)"},
                   "all_cores": {"value": va, "unit": UNIT, "cores": cores,
                                 "sample": f"{cores} curves at N=2^{la}, one per host thread, 1 E13 iteration each, {dta:.1f} s"}}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": cfg["dtype"], "data": "synthetic",
                "config": {"workload": workload_label(cfg), "curves_per_gpu": B, "max_iter": iters,
                           "iterations_executed_per_curve_mean": iters_executed / B,
                           "nominal_value_at_max_iter": world * B * N * iters * args.steps / (ms * 1e-3),
                           "iters_used": iters_used[:8], "l2": "inputs larger than L2 (every array >= 1 GiB)"
                           if B * N * 4 > 2 ** 28 else "arrays smaller than L2: not flushed between steps",
                           "step": "S1 + S2 + max_iter x (L1..L6) + P",
                           "timing": "value: untraced; kernels/stages/roofline: one extra traced step; stages and roofline count the launches of the E13 call only"},
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "stages": stages,
                "traffic_model": traffic_model, "sort_fallbacks": fallbacks, "ms_traced_step": ms_traced,
                "ms_by_call_traced": phase_ms,   # S1 / S2 / E13 / P: kernel time of each C-ABI call in the traced step
                "cpu_baseline": cpu, "fp32_free_running_context": context, "other_configs": other, "kernels": kernels}
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
